// plan_types.cuh -- parameter blocks passed by value to the kernels (and to the host stepping
// harness in tests/emu).  Pointers are device pointers in libfsei, host pointers in the harness.
#pragma once
#include "fft_core.cuh"

namespace fsei {

enum { BC_PERIODIC = 0, BC_NEUMANN = 1 };
enum { COMP_U = 0, COMP_V = 1, COMP_W = 2, DIR_X = 0, DIR_Y = 1, DIR_Z = 2 };   // velocity components, directions

// Transform along x: real lines of n = nx values handled as N = nx/2 complex values.
//   periodic: real-to-complex FFT, slot pos[k] holds X_k (k = 1..N-1), slot 0 holds (X_0, X_N) (both real)
//   Neumann : DCT-II (Makhoul: even/odd reorder + real FFT + quarter-wave twiddle),
//             slot pos[k] holds (X_k, X_{n-k}), slot 0 holds (X_0, X_{n/2})
struct XParams {
    int n;                // nx
    int N;                // nx / 2
    int bc;
    int pitch;            // complex elements per line in the shared tile (padded)
    FftPlan1D f;
    const cplx* tw;       // e^{-2 pi i m / N}, m in [0, N)
    const int* pos;       // pos[k], k in [0, N)
    const cplx* tw_r2c;   // e^{-2 pi i k / n}, k in [0, N/2]
    const cplx* tw_dct;   // e^{-i pi k / (2 n)}, k in [0, N]   (Neumann only)
    double scale;         // 1 / ((nx/2) * ny), applied by the inverse store
};

// Transform along y on complex columns of N = ny values.
//   periodic: complex FFT, row pos[k] holds frequency k
//   Neumann : DCT-II of Re and Im separately (real-linear), physical row perm(pos[k]) holds k
struct YParams {
    int N;                // ny
    int bc;
    FftPlan1D f;
    const cplx* tw;       // e^{-2 pi i m / N}
    const int* pos;
    const cplx* tw_dct;   // e^{-i pi k / (2 N)}, k in [0, N)   (Neumann only)
};

// z-solve.  Spectrum element (k, row, slot) at ((k*ny + row)*nxc + slot), complex.
struct ZParams {
    int nxc, ny, nz;
    int ncomp;            // 1: one factorisation per slot column; 2: Re and Im have their own
    const double* za;     // a_k  (a_0 = 0)
    const double* zcc;    // c_k  (c_{nz-1} = 0)
    const double* ipiv;   // [nz][ny][nxc][ncomp] reciprocal pivots of the Thomas factorisation
    const double* lamx;   // [nxc][2]  (lambda of Re part, lambda of Im part) per slot
    const double* lamy;   // [ny]      per physical row
    const int* posy;      // y pos table (paired kernel: rows of ky and ny-ky)
    const double* gauge;  // [nz] solution of the (0,0) column, written by the gauge kernel
    double* cpw;          // scratch for the paired kernel: c' of both factorisations
    const double* dzc;    // [nz]
    const double* dzm;    // [nz] (dzm[0] unused)
};

// Stencil metrics (doubles computed exactly as the definition states, R20).
struct SParams {
    int nx, ny, nz, bcx, bcy;
    double rdx, rdy;
    const double* rdzc;   // 1/(zc[k+1]-zc[k])
    const double* rdzm;   // 1/(zm[k]-zm[k-1]), rdzm[0] = 0
    // z-slab view (multi-GPU decomposition, slab.py): the fields hold planes [kofs, kofs + nz) of the global grid; the
    // metric tables stay global (indexed k + kofs); halo_lo / halo_hi: the plane below the first / above the last one
    // is present in memory (a neighbour's plane) instead of being a wall
    int kofs = 0, halo_lo = 0, halo_hi = 0;
};

FSEI_HD int padx(int n) { return n + (n >> 3); }
// Makhoul reorder: logical index n of the reordered sequence v -> index of the natural sequence
FSEI_HD int dct_perm(int n, int N) { return (n < (N >> 1)) ? 2 * n : 2 * (N - 1 - n) + 1; }

}  // namespace fsei
