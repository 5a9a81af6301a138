// yfast.cuh -- fast-path kernel of steps a3 / a5: the transform along y of the packed x-spectrum, in
// place, for ny = 2^a or 3 2^a (include/fsei.h; R15, sec. 6).
//
// A CTA of T*CY threads owns a tile of CY adjacent x-slots (CY*16 contiguous bytes per row) times all ny
// rows of one z-plane and loops over planes.  The tile of the next plane is fetched by the TMA engine
// (cp.async.bulk.tensor.2d boxes of <= 256 rows x CY*16 bytes through a CUtensorMap of the spectrum, into a
// dense shared-memory landing tile [n][CY], completion on an mbarrier) while the CTA transforms the current
// one.  Thread (c, tl) holds butterflies of column c in registers: the first pass reads the landing tile,
// the last writes global memory (row stride nxc); in between the column tile sits in a padded shared
// buffer [pad(n)][CY].
//
//   periodic y: complex FFT.  Columns whose Re and Im are two different real x-sequences A, B (slot 0 of
//               a periodic x-transform: (X_0, X_N); every slot of a Neumann x-transform) carry two
//               Hermitian y-spectra; the forward kernel splits them (rows 1..ny/2-1 <- A^(ky), rows
//               ny-ky <- B^(ky), rows 0 and ny/2 keep (A^, B^) which are real there) so that every
//               z-column has ONE wavenumber pair per component; the inverse kernel merges them back.
//   Neumann y : DCT-II of Re and Im (Makhoul reorder on the row index, complex FFT, Hermitian split +
//               quarter-wave twiddle); row k holds coefficient k of both parts.
#pragma once
#include "xfast.cuh"

namespace fsei {

struct YFast {
    int nxc, ny, nz;
    int untangle;               // periodic y: columns [0, untangle) are split / merged (0, 1 or nxc)
    const cplx* tw;             // e^{-2 pi i j / ny}
    const cplx* tw_dct;         // e^{-i pi k / (2 ny)}, k in [0, ny)   (Neumann only)
    // multi-GPU slab decomposition, peer-store exchange (slab.py): when npeer > 0 the FORWARD transform
    // does not write its result back to the local spectrum but straight into the pencils of the ranks that own the slots:
    // element (k, row, slot) -> peer_base[d][((kofs + k) ny + row) nsl_d + slot - peer_s0[d]], peer_s0[d] <= slot < peer_s0[d+1]
    // (peer_base[d] may be a peer-mapped pointer: the stores then travel over NVLink while the CTA transforms its next tile)
    int npeer = 0, kofs = 0;
    cplx* peer_base[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int peer_s0[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
};

template <class C, int CY, bool NEU> struct YSmemLayout {
    static constexpr int LAND = C::N * CY;                      // complex, dense TMA destination
    static constexpr int BUF = C::PITCH * CY;
    static constexpr int TWS = C::TW;
    static constexpr int DCT = NEU ? C::N / 2 + 1 : 0;
    static constexpr size_t BYTES = 128 + sizeof(cplx) * (LAND + BUF + TWS + DCT);
};
// rows per TMA box: the largest divisor of N that is <= 256
FSEI_HD constexpr int y_box_rows(int N) { int b = N < 256 ? N : 256; while (N % b) b--; return b; }

template <class C, int CY> struct YIn {
    const cplx* s; int c;
    FSEI_HD cplx operator()(int n) const { return s[C::pad(n) * CY + c]; }
};
template <class C, int CY> struct YOut {
    cplx* s; int c;
    FSEI_HD void operator()(int n, cplx v, int = 0) const { s[C::pad(n) * CY + c] = v; }
};

// same pass sequence as fft_line (xfast.cuh) on a column of the [n][CY] tile
// hook_last() runs right before the arithmetic of the last pass (its inputs are already in registers).
template <class C, int CY, bool INV, bool IN_BUF, bool OUT_BUF, class Load0, class Out, class Hook, class HookL>
FSEI_DEV void fft_column(int tl, int c, bool act, cplx* buf, const cplx* tws, Load0 load0, Out out, Hook hook, HookL hook_last)
{
    constexpr int N = C::N, T = C::T;
    static_assert(C::NP >= 2, "pipelined kernels need at least two passes");
    YIn<C, CY> bin{buf, c}; YOut<C, CY> bout{buf, c};
    {
        cplx v[PassShape<N, C::R0, 1, T>::PER][C::R0];
        if (act) load0(v);
        if (IN_BUF) { FSEI_SYNC(); hook(); }
        if (act) fft_pass_compute<N, C::R0, 1, T, INV>(tl, tws, v, bout);
    }
    FSEI_SYNC();
    if (!IN_BUF) hook();
    {
        cplx v[PassShape<N, C::R1, C::R0, T>::PER][C::R1];
        if (act) fft_pass_load<N, C::R1, C::R0, T>(tl, bin, v);
        if constexpr (C::NP == 2) {
            if (OUT_BUF) FSEI_SYNC();
            hook_last();
            if (act) fft_pass_compute<N, C::R1, C::R0, T, INV>(tl, tws, v, out);
            return;
        } else {
            FSEI_SYNC();
            if (act) fft_pass_compute<N, C::R1, C::R0, T, INV>(tl, tws, v, bout);
        }
    }
    FSEI_SYNC();
    if constexpr (C::NP >= 3) {
        cplx v[PassShape<N, C::R2, C::R0 * C::R1, T>::PER][C::R2];
        if (act) fft_pass_load<N, C::R2, C::R0 * C::R1, T>(tl, bin, v);
        if (OUT_BUF) FSEI_SYNC();
        hook_last();
        if (act) fft_pass_compute<N, C::R2, C::R0 * C::R1, T, INV>(tl, tws + C::TW1, v, out);
    }
}
template <class C, int CY, bool INV, bool IN_BUF, bool OUT_BUF, class Load0, class Out, class Hook>
FSEI_DEV void fft_column(int tl, int c, bool act, cplx* buf, const cplx* tws, Load0 load0, Out out, Hook hook)
{
    fft_column<C, CY, INV, IN_BUF, OUT_BUF>(tl, c, act, buf, tws, load0, out, hook, NoHook{});
}

// grid (ceil(nxc / CY), gy <= nz), block T*CY, dynamic shared memory YSmemLayout::BYTES.
// map: 2-D tensor map of the spectrum, inner dimension 2 nxc doubles, outer ny nz rows, box 2 CY x y_box_rows(ny)
template <class C, int CY, bool INV, bool NEU>
FSEI_GLOBAL(C::T * CY, 1) k_y_fast(YFast P, const FSEI_GRID_CONSTANT TmaMap2D map, cplx* spec)
{
    using L = YSmemLayout<C, CY, NEU>;
    constexpr int N = C::N, T = C::T, R0 = C::R0;
    constexpr int NB0 = N / R0, PER0 = PassShape<N, R0, 1, T>::PER;
    constexpr int BOX = y_box_rows(N);
    static_assert(NB0 % T == 0, "first pass must tile the column exactly");
    FSEI_DYN_SMEM(smraw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    cplx* land = reinterpret_cast<cplx*>(smraw + 128);           // [N][CY]
    cplx* buf = land + L::LAND;
    cplx* tws = buf + L::BUF;
    cplx* tdct = tws + L::TWS;
    const int tid = threadIdx.x, nt = T * CY;
    const int tl = tid / CY, c = tid - tl * CY;
    const int nxc = P.nxc;
    const int c0 = blockIdx.x * CY, col = c0 + c;
    const bool act = col < nxc;
    const bool pairing = NEU || (c0 < P.untangle);            // CTA-uniform
    const bool mine = NEU || (col < P.untangle);              // this column is split / merged
    const double SQ2 = 1.41421356237309504880168872420969808;
    const int kstep = gridDim.y;

    auto issue = [&](int k) {
        abar_expect(bar, (unsigned)(N * CY * sizeof(cplx)));
#pragma unroll
        for (int b = 0; b < N / BOX; b++) tma_load_2d(land + b * BOX * CY, &map, 2 * c0, k * N + b * BOX, bar);
    };
    if (tid == 0) abar_init(bar);
    fft_fill_twiddles<C>(tws, P.tw, tid, nt);
    if (NEU) for (int i = tid; i < L::DCT; i += nt) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();
    if (tid == 0 && (int)blockIdx.y < P.nz) issue(blockIdx.y);
    unsigned parity = 0;

    for (int k = blockIdx.y; k < P.nz; k += kstep) {
        abar_wait(bar, parity); parity ^= 1;
        cplx* g = spec + (size_t)k * N * nxc + col;            // row r of this column at g[r * gs]
        size_t gs = (size_t)nxc;
        if (!INV && P.npeer > 0 && act) {                      // peer-store exchange: this column's rows go to the owner of its slot
            int d = 0;
            while (d + 1 < P.npeer && col >= P.peer_s0[d + 1]) d++;
            gs = (size_t)(P.peer_s0[d + 1] - P.peer_s0[d]);
            g = P.peer_base[d] + (size_t)(P.kofs + k) * N * gs + (col - P.peer_s0[d]);
        }
        auto next = [&]() { if (tid == 0 && k + kstep < P.nz) issue(k + kstep); };
        if (!INV) {
            auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
                for (int i = 0; i < PER0; i++) {
#pragma unroll
                    for (int q = 0; q < R0; q++) {
                        const int n = tl + i * T + q * NB0;
                        v0[i][q] = land[(NEU ? dct_perm(n, N) : n) * CY + c];
                    }
                }
            };
            if (!pairing) {
                auto out = [&](int n, cplx z, int) { g[(size_t)n * gs] = z; };
                fft_column<C, CY, false, false, false>(tl, c, act, buf, tws, load0, out, next);
            } else {
                fft_column<C, CY, false, false, true>(tl, c, act, buf, tws, load0, YOut<C, CY>{buf, c}, next);
                FSEI_SYNC();
                if (act) {
                    for (int kk = tl; kk <= N / 2; kk += T) {
                        cplx p1 = buf[C::pad(kk) * CY + c];
                        if (kk == 0 || (!NEU && (2 * kk == N || !mine))) {
                            g[(size_t)kk * gs] = p1;
                            if (kk != 0 && 2 * kk != N) g[(size_t)(N - kk) * gs] = buf[C::pad(N - kk) * CY + c];
                            continue;
                        }
                        cplx p2 = buf[C::pad(N - kk) * CY + c];
                        cplx A = cmake(0.5 * (p1.re + p2.re), 0.5 * (p1.im - p2.im));   // (P1 + conj P2)/2
                        cplx D = cmake(p1.re - p2.re, p1.im + p2.im);
                        cplx B = cmake(0.5 * D.im, -0.5 * D.re);                        // (P1 - conj P2)/(2i)
                        if (NEU) {
                            cplx wk = tdct[kk];
                            cplx ta = cmul(A, wk), tb = cmul(B, wk);
                            g[(size_t)kk * gs] = cmake(ta.re, tb.re);
                            if (2 * kk != N) g[(size_t)(N - kk) * gs] = cmake(-ta.im, -tb.im);
                        } else {
                            g[(size_t)kk * gs] = A;
                            g[(size_t)(N - kk) * gs] = B;
                        }
                    }
                }
            }
        } else {
            auto out = [&](int n, cplx z, int) { g[(size_t)(NEU ? dct_perm(n, N) : n) * gs] = z; };
            if (!pairing) {
                auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
                    for (int i = 0; i < PER0; i++) {
#pragma unroll
                        for (int q = 0; q < R0; q++) v0[i][q] = land[(tl + i * T + q * NB0) * CY + c];
                    }
                };
                fft_column<C, CY, true, false, false>(tl, c, act, buf, tws, load0, out, next);
            } else {
                if (act) {
                    for (int kk = tl; kk <= N / 2; kk += T) {
                        cplx a = land[kk * CY + c];
                        if (kk == 0 || (!NEU && (2 * kk == N || !mine))) {
                            buf[C::pad(kk) * CY + c] = a;
                            if (kk != 0 && 2 * kk != N) buf[C::pad(N - kk) * CY + c] = land[(N - kk) * CY + c];
                            continue;
                        }
                        if (NEU && 2 * kk == N) { buf[C::pad(kk) * CY + c] = cmake(a.re * SQ2, a.im * SQ2); continue; }
                        cplx b = land[(N - kk) * CY + c];
                        if (NEU) {
                            cplx wk = tdct[kk];
                            cplx ta = cmulc(cmake(a.re, -b.re), wk);     // V^a_k
                            cplx tb = cmulc(cmake(a.im, -b.im), wk);     // V^b_k
                            a = ta; b = tb;
                        }
                        buf[C::pad(kk) * CY + c] = cmake(a.re - b.im, a.im + b.re);          // A + i B
                        buf[C::pad(N - kk) * CY + c] = cmake(a.re + b.im, -a.im + b.re);     // conj A + i conj B
                    }
                }
                FSEI_SYNC();
                next();                                         // landing tile consumed
                auto load0 = [&](cplx (*v0)[R0]) { fft_pass_load<N, R0, 1, T>(tl, YIn<C, CY>{buf, c}, v0); };
                fft_column<C, CY, true, true, false>(tl, c, act, buf, tws, load0, out, NoHook{});
            }
        }
        FSEI_SYNC();
    }
}

}  // namespace fsei
