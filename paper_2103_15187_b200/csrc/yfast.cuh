// yfast.cuh -- fast-path kernel of steps a3 / a5: the transform along y of the packed x-spectrum, in
// place, for ny = 2^a or 3 2^a (include/fsei.h; R15, sec. 6).
//
// A CTA of T*CY threads owns a tile of CY adjacent x-slots (CY*16 contiguous bytes per row) times all ny
// rows of one z-plane and loops over planes.  Thread (c, tl) holds butterflies of column c in registers;
// the first pass reads global memory directly (row stride nxc), the last writes it; in between the
// column tile sits in one shared buffer [pad(n)][CY].
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
};

template <class C, int CY, bool NEU> struct YSmemLayout {
    static constexpr int BUF = C::PITCH * CY;
    static constexpr int TWS = C::TW;
    static constexpr int DCT = NEU ? C::N / 2 + 1 : 0;
    static constexpr size_t BYTES = sizeof(cplx) * (BUF + TWS + DCT);
};

template <class C, int CY> struct YIn {
    const cplx* s; int c;
    FSEI_HD cplx operator()(int n) const { return s[C::pad(n) * CY + c]; }
};
template <class C, int CY> struct YOut {
    cplx* s; int c;
    FSEI_HD void operator()(int n, cplx v) const { s[C::pad(n) * CY + c] = v; }
};

// same pass sequence as fft_line (xfast.cuh) on a column of the [n][CY] tile
template <class C, int CY, bool INV, bool IN_BUF, bool OUT_BUF, class Load0, class Out>
FSEI_DEV void fft_column(int tl, int c, bool act, cplx* buf, const cplx* tws, Load0 load0, Out out)
{
    constexpr int N = C::N, T = C::T;
    YIn<C, CY> bin{buf, c}; YOut<C, CY> bout{buf, c};
    {
        cplx v[PassShape<N, C::R0, 1, T>::PER][C::R0];
        if (act) load0(v);
        if constexpr (C::NP == 1) {
            if (IN_BUF && OUT_BUF) FSEI_SYNC();
            if (act) fft_pass_compute<N, C::R0, 1, T, INV>(tl, tws, v, out);
            return;
        } else {
            if (IN_BUF) FSEI_SYNC();
            if (act) fft_pass_compute<N, C::R0, 1, T, INV>(tl, tws, v, bout);
        }
    }
    FSEI_SYNC();
    if constexpr (C::NP >= 2) {
        cplx v[PassShape<N, C::R1, C::R0, T>::PER][C::R1];
        if (act) fft_pass_load<N, C::R1, C::R0, T>(tl, bin, v);
        if constexpr (C::NP == 2) {
            if (OUT_BUF) FSEI_SYNC();
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
        if (act) fft_pass_compute<N, C::R2, C::R0 * C::R1, T, INV>(tl, tws + C::TW1, v, out);
    }
}

// grid (ceil(nxc / CY), gy <= nz), block T*CY, dynamic shared memory YSmemLayout::BYTES
template <class C, int CY, bool INV, bool NEU>
FSEI_GLOBAL(C::T * CY, (C::RMAX >= 16 || C::T * CY > 256 ? 1 : 2)) k_y_fast(YFast P, cplx* spec)
{
    using L = YSmemLayout<C, CY, NEU>;
    constexpr int N = C::N, T = C::T, R0 = C::R0;
    constexpr int NB0 = N / R0, PER0 = PassShape<N, R0, 1, T>::PER;
    static_assert(NB0 % T == 0, "first pass must tile the column exactly");
    FSEI_DYN_SMEM(smraw);
    cplx* buf = reinterpret_cast<cplx*>(smraw);
    cplx* tws = buf + L::BUF;
    cplx* tdct = tws + L::TWS;
    const int tid = threadIdx.x, nt = T * CY;
    const int tl = tid / CY, c = tid - tl * CY;
    fft_fill_twiddles<C>(tws, P.tw, tid, nt);
    if (NEU) for (int i = tid; i < L::DCT; i += nt) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();

    const int nxc = P.nxc;
    const int c0 = blockIdx.x * CY, col = c0 + c;
    const bool act = col < nxc;
    const bool pairing = NEU || (c0 < P.untangle);            // CTA-uniform
    const bool mine = NEU || (col < P.untangle);              // this column is split / merged
    const double SQ2 = 1.41421356237309504880168872420969808;

    for (int k = blockIdx.y; k < P.nz; k += gridDim.y) {
        cplx* g = spec + (size_t)k * N * nxc + col;            // row r of this column at g[r * nxc]
        auto row_of = [&](int n) -> size_t { return (size_t)(NEU ? dct_perm(n, N) : n) * nxc; };
        if (!INV) {
            auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
                for (int i = 0; i < PER0; i++) {
#pragma unroll
                    for (int q = 0; q < R0; q++) v0[i][q] = g[row_of(tl + i * T + q * NB0)];
                }
            };
            if (!pairing) {
                auto out = [&](int n, cplx z) { g[(size_t)n * nxc] = z; };
                fft_column<C, CY, false, false, false>(tl, c, act, buf, tws, load0, out);
            } else {
                fft_column<C, CY, false, false, true>(tl, c, act, buf, tws, load0, YOut<C, CY>{buf, c});
                FSEI_SYNC();
                if (act) {
                    for (int kk = tl; kk <= N / 2; kk += T) {
                        cplx p1 = buf[C::pad(kk) * CY + c];
                        if (kk == 0 || (!NEU && (2 * kk == N || !mine))) {
                            g[(size_t)kk * nxc] = p1;
                            if (kk != 0 && 2 * kk != N) g[(size_t)(N - kk) * nxc] = buf[C::pad(N - kk) * CY + c];
                            continue;
                        }
                        cplx p2 = buf[C::pad(N - kk) * CY + c];
                        cplx A = cmake(0.5 * (p1.re + p2.re), 0.5 * (p1.im - p2.im));   // (P1 + conj P2)/2
                        cplx D = cmake(p1.re - p2.re, p1.im + p2.im);
                        cplx B = cmake(0.5 * D.im, -0.5 * D.re);                        // (P1 - conj P2)/(2i)
                        if (NEU) {
                            cplx wk = tdct[kk];
                            cplx ta = cmul(A, wk), tb = cmul(B, wk);
                            g[(size_t)kk * nxc] = cmake(ta.re, tb.re);
                            if (2 * kk != N) g[(size_t)(N - kk) * nxc] = cmake(-ta.im, -tb.im);
                        } else {
                            g[(size_t)kk * nxc] = A;
                            g[(size_t)(N - kk) * nxc] = B;
                        }
                    }
                }
            }
        } else {
            auto out = [&](int n, cplx z) { g[row_of(n)] = z; };
            if (!pairing) {
                auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
                    for (int i = 0; i < PER0; i++) {
#pragma unroll
                        for (int q = 0; q < R0; q++) v0[i][q] = g[(size_t)(tl + i * T + q * NB0) * nxc];
                    }
                };
                fft_column<C, CY, true, false, false>(tl, c, act, buf, tws, load0, out);
            } else {
                if (act) {
                    for (int kk = tl; kk <= N / 2; kk += T) {
                        cplx a = g[(size_t)kk * nxc];
                        if (kk == 0 || (!NEU && (2 * kk == N || !mine))) {
                            buf[C::pad(kk) * CY + c] = a;
                            if (kk != 0 && 2 * kk != N) buf[C::pad(N - kk) * CY + c] = g[(size_t)(N - kk) * nxc];
                            continue;
                        }
                        if (NEU && 2 * kk == N) { buf[C::pad(kk) * CY + c] = cmake(a.re * SQ2, a.im * SQ2); continue; }
                        cplx b = g[(size_t)(N - kk) * nxc];
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
                auto load0 = [&](cplx (*v0)[R0]) { fft_pass_load<N, R0, 1, T>(tl, YIn<C, CY>{buf, c}, v0); };
                fft_column<C, CY, true, true, false>(tl, c, act, buf, tws, load0, out);
            }
        }
        FSEI_SYNC();
    }
}

}  // namespace fsei
