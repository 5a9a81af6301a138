// plan_host.hpp -- host-side construction of every table the kernels read: pass radices,
// digit-reversal maps, twiddles, modified wavenumbers (R6), wall-normal metric
// coefficients (R2, R5).  Trigonometry and reciprocals are evaluated in long double and rounded
// once.  Plain C++ (no CUDA), shared by libfsei (which uploads the tables) and tests/emu.
#pragma once
#include <cmath>
#include <cstddef>
#include <string>
#include <vector>
#include "plan_types.cuh"

namespace fsei {

struct HostTables {
    int nx, ny, nz, bcx, bcy, nxc;
    double Lx, Ly;
    FftPlan1D fx, fy;
    std::vector<cplx> twx, twx_r2c, twx_dct, twy, twy_dct;
    std::vector<int> posx, posy;
    std::vector<double> za, zcc, dzc, dzm, lamx, lamy, rdzc, rdzm;
    double rdx, rdy, scale;
    int ncomp;          // 1 or 2 reciprocal-pivot components per slot (see ZParams)
    bool paired_all;    // x Neumann + y periodic: every slot goes through the paired kernel
    bool paired_slot0;  // x periodic + y periodic: slot 0 only
    bool fast;          // natural-order spectrum layout of the fast path (xfast.cuh / yfast.cuh): pos tables are the identity
};

static const long double FSEI_PI_L = 3.14159265358979323846264338327950288L;

inline bool is_2a3b(int n) { if (n < 1) return false; while (n % 2 == 0) n /= 2; while (n % 3 == 0) n /= 3; return n == 1; }
inline bool is_2a3b5c(int n) { if (n < 1) return false; while (n % 5 == 0) n /= 5; return is_2a3b(n); }

// radices: all factors 3 and 5 first (large strides), then the power of two split into ceil(a/4)
// passes of radix 16/8/4/2, largest first.
inline FftPlan1D make_fft_plan(int N)
{
    FftPlan1D f; f.N = N; f.npass = 0;
    for (int i = 0; i < 8; i++) f.radix[i] = 1;
    int n = N, a = 0;
    while (n % 3 == 0) { f.radix[f.npass++] = 3; n /= 3; }
    while (n % 5 == 0) { f.radix[f.npass++] = 5; n /= 5; }
    while (n % 2 == 0) { a++; n /= 2; }
    if (a > 0) {
        int np = (a + 3) / 4, base = a / np, extra = a % np;
        for (int i = 0; i < np; i++) f.radix[f.npass++] = 1 << (base + (i < extra ? 1 : 0));
    }
    return f;
}

inline std::vector<int> make_pos(const FftPlan1D& f)
{
    std::vector<int> pos(f.N);
    for (int k = 0; k < f.N; k++) {
        int kk = k, M = f.N, p = 0;
        for (int s = 0; s < f.npass; s++) { M /= f.radix[s]; p += (kk % f.radix[s]) * M; kk /= f.radix[s]; }
        pos[k] = p;
    }
    return pos;
}

inline cplx unit(long double ang) { return cmake((double)cosl(ang), (double)sinl(ang)); }

inline long double lam_periodic(int m, int n, long double h) { long double s = sinl(FSEI_PI_L * m / n); return -4.0L * s * s / (h * h); }
inline long double lam_neumann(int m, int n, long double h) { long double s = sinl(FSEI_PI_L * m / (2.0L * n)); return -4.0L * s * s / (h * h); }

// returns "" on success, else a message; code = FSEI_ERR_* value (2 size, 3 grid, 1 arg)
inline std::string build_tables(HostTables& T, int nx, int ny, int nz, double Lx, double Ly, const double* zc,
                                int bcx, int bcy, int& code, bool fast_layout = false)
{
    code = 0;
    if (zc == nullptr) { code = 1; return "zc is NULL"; }
    if ((bcx != BC_PERIODIC && bcx != BC_NEUMANN) || (bcy != BC_PERIODIC && bcy != BC_NEUMANN)) { code = 1; return "unknown boundary condition"; }
    if (nx < 4 || ny < 4 || nx > 8192 || ny > 8192 || nx % 4 != 0 || ny % 2 != 0 || !is_2a3b5c(nx) || !is_2a3b5c(ny)) {
        code = 2; return "nx must be a multiple of 4, ny even, both of the form 2^a 3^b 5^c in [4, 8192]";
    }
    if (nz < 2 || nz > 8192) { code = 2; return "nz must be in [2, 8192]"; }
    if (!(Lx > 0) || !(Ly > 0) || !std::isfinite(Lx) || !std::isfinite(Ly)) { code = 3; return "Lx, Ly must be positive and finite"; }
    for (int k = 0; k <= nz; k++) if (!std::isfinite(zc[k])) { code = 3; return "zc holds a non-finite value"; }
    for (int k = 0; k < nz; k++) if (!(zc[k + 1] > zc[k])) { code = 3; return "zc must be strictly increasing"; }

    T.nx = nx; T.ny = ny; T.nz = nz; T.bcx = bcx; T.bcy = bcy; T.Lx = Lx; T.Ly = Ly; T.nxc = nx / 2;
    const int N = nx / 2;
    T.fx = make_fft_plan(N); T.fy = make_fft_plan(ny);
    T.posx = make_pos(T.fx); T.posy = make_pos(T.fy);
    T.fast = fast_layout;
    if (fast_layout) {                      // Stockham passes leave natural order
        for (int k = 0; k < N; k++) T.posx[k] = k;
        for (int k = 0; k < ny; k++) T.posy[k] = k;
    }
    T.twx.resize(N); for (int m = 0; m < N; m++) T.twx[m] = unit(-2.0L * FSEI_PI_L * m / N);
    T.twx_r2c.resize(N / 2 + 1); for (int k = 0; k <= N / 2; k++) T.twx_r2c[k] = unit(-2.0L * FSEI_PI_L * k / nx);
    T.twx_dct.resize(N + 1); for (int k = 0; k <= N; k++) T.twx_dct[k] = unit(-FSEI_PI_L * k / (2.0L * nx));
    T.twy.resize(ny); for (int m = 0; m < ny; m++) T.twy[m] = unit(-2.0L * FSEI_PI_L * m / ny);
    T.twy_dct.resize(ny); for (int k = 0; k < ny; k++) T.twy_dct[k] = unit(-FSEI_PI_L * k / (2.0L * ny));
    T.scale = (double)(1.0L / ((long double)N * (long double)ny));

    // Wall-normal metrics.  They are fp64 data of the grid, evaluated in double exactly as the stencils a1/a7
    // use them (R5, R20); the tridiagonal coefficients are the products of those very reciprocals so
    // that the operator solved IS the D G the divergence and projection kernels apply (a mismatch of
    // ulp(zc)/dz ~ 1e-12 near the upper wall would cost ~30x in post-projection divergence).
    T.za.assign(nz, 0.0); T.zcc.assign(nz, 0.0); T.dzc.assign(nz, 0.0); T.dzm.assign(nz, 0.0);
    T.rdx = 1.0 / (Lx / (double)nx); T.rdy = 1.0 / (Ly / (double)ny);
    T.rdzc.assign(nz, 0.0); T.rdzm.assign(nz, 0.0);
    for (int k = 0; k < nz; k++) { T.dzc[k] = zc[k + 1] - zc[k]; T.rdzc[k] = 1.0 / T.dzc[k]; }
    for (int k = 1; k < nz; k++) { T.dzm[k] = 0.5 * (zc[k] + zc[k + 1]) - 0.5 * (zc[k - 1] + zc[k]); T.rdzm[k] = 1.0 / T.dzm[k]; }
    for (int k = 0; k < nz; k++) {
        T.za[k] = (k > 0) ? T.rdzm[k] * T.rdzc[k] : 0.0;
        T.zcc[k] = (k < nz - 1) ? T.rdzm[k + 1] * T.rdzc[k] : 0.0;
    }

    // modified wavenumbers per x-slot (Re part, Im part) and per physical y-row
    const long double hx = (long double)Lx / nx, hy = (long double)Ly / ny;
    T.lamx.assign(2 * (size_t)N, 0.0);
    if (bcx == BC_PERIODIC) {
        T.lamx[0] = (double)lam_periodic(0, nx, hx); T.lamx[1] = (double)lam_periodic(N, nx, hx);
        for (int k = 1; k < N; k++) { double l = (double)lam_periodic(k, nx, hx); T.lamx[2 * T.posx[k]] = l; T.lamx[2 * T.posx[k] + 1] = l; }
    } else {
        T.lamx[0] = (double)lam_neumann(0, nx, hx); T.lamx[1] = (double)lam_neumann(N, nx, hx);
        for (int k = 1; k < N; k++) { T.lamx[2 * T.posx[k]] = (double)lam_neumann(k, nx, hx); T.lamx[2 * T.posx[k] + 1] = (double)lam_neumann(nx - k, nx, hx); }
    }
    T.lamy.assign(ny, 0.0);
    for (int k = 0; k < ny; k++) {
        if (bcy == BC_PERIODIC) T.lamy[T.posy[k]] = (double)lam_periodic(k, ny, hy);
        else T.lamy[fast_layout ? k : dct_perm(T.posy[k], ny)] = (double)lam_neumann(k, ny, hy);
    }
    T.paired_all = (bcx == BC_NEUMANN && bcy == BC_PERIODIC);
    T.paired_slot0 = (bcx == BC_PERIODIC && bcy == BC_PERIODIC);
    T.ncomp = (bcy == BC_NEUMANN) ? 2 : 1;
    return "";
}

}  // namespace fsei
