// fft_core.cuh -- register-level pieces of the transforms: complex type, small DFTs
// (radix 2, 3, 4, 5, 8, 16) and one in-place decimation-in-frequency / decimation-in-time pass
// over a shared-memory tile.  Everything is __host__ __device__ so that the per-thread phases
// of the kernels can also be stepped through on the host by tests/emu (thread by thread,
// phase by phase) -- that harness is a test of this code, not a fallback: libfsei.so holds
// device code only.
//
// Transform conventions (R15): forward e^{-i...} unnormalised; the inverse here is
// the exact algebraic inverse of the forward pass sequence WITHOUT the 1/N (the caller folds
// 1/(nx*ny) into the last store).
//
// In-place mixed-radix scheme.  N = R_0 R_1 ... R_{P-1}.  Forward pass s works on sub-length
// Ns (N, N/R_0, ...), M = Ns/R_s: for every block blk of Ns consecutive logical indices and
// every n2 in [0,M) the R_s elements blk*Ns + n1*M + n2 are replaced by their R_s-point DFT
// times w_Ns^{n2 k1}.  After all passes frequency k sits at the mixed-radix digit-reversed
// logical index pos(k) = sum_s digit_s(k) * (N / (R_0..R_s)).  The inverse runs the passes
// backwards with conjugate twiddles (digit-reversed in, natural out), so no reordering pass
// is ever needed; the z-solve reads its wavenumbers through the same pos() tables.
#pragma once

#if defined(__CUDACC__)
#define FSEI_HD __host__ __device__ __forceinline__
#else
#define FSEI_HD inline
#endif
#define FSEI_RESTRICT __restrict__

namespace fsei {

struct alignas(16) cplx { double re, im; };      // 16-byte aligned: one 128-bit load/store per element

FSEI_HD cplx cmake(double a, double b) { cplx c; c.re = a; c.im = b; return c; }
FSEI_HD cplx cadd(cplx a, cplx b) { return cmake(a.re + b.re, a.im + b.im); }
FSEI_HD cplx csub(cplx a, cplx b) { return cmake(a.re - b.re, a.im - b.im); }
FSEI_HD cplx cmul(cplx a, cplx b) { return cmake(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
FSEI_HD cplx cmulc(cplx a, cplx b) { /* a * conj(b) */ return cmake(a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im); }
FSEI_HD cplx cconj(cplx a) { return cmake(a.re, -a.im); }
FSEI_HD cplx cscale(cplx a, double s) { return cmake(a.re * s, a.im * s); }
// multiply by -i (forward quarter turn) or +i (inverse)
template <bool INV> FSEI_HD cplx crot(cplx a) { return INV ? cmake(-a.im, a.re) : cmake(a.im, -a.re); }
// multiply by w (forward) or conj(w) (inverse)
template <bool INV> FSEI_HD cplx ctw(cplx a, double wr, double wi) {
    return INV ? cmake(a.re * wr + a.im * wi, a.im * wr - a.re * wi) : cmake(a.re * wr - a.im * wi, a.re * wi + a.im * wr);
}

#define FSEI_SQRT1_2 0.70710678118654752440084436210484903928
#define FSEI_SQRT3_2 0.86602540378443864676372317075293618347
#define FSEI_COS_PI_8 0.92387953251128675612818318939678828682
#define FSEI_SIN_PI_8 0.38268343236508977172845998403039886676

// ---- small DFTs, in place on v[0..R), natural order in and out -------------------------------
template <int R, bool INV> struct SmallDft;

template <bool INV> struct SmallDft<2, INV> {
    static FSEI_HD void run(cplx* v) { cplx a = v[0], b = v[1]; v[0] = cadd(a, b); v[1] = csub(a, b); }
};
template <bool INV> struct SmallDft<3, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx s = cadd(v[1], v[2]), d = csub(v[1], v[2]);
        cplx m = cmake(v[0].re - 0.5 * s.re, v[0].im - 0.5 * s.im);
        cplx n = cscale(crot<INV>(d), FSEI_SQRT3_2);          // (-+ i sqrt3/2) d
        v[0] = cadd(v[0], s); v[1] = cadd(m, n); v[2] = csub(m, n);
    }
};
// 5: X_k = x0 + sum_{r=1..4} w5^{rk} x_r with the pairs (x1, x4), (x2, x3) folded (Winograd-style, 2 real tables)
#define FSEI_COS_2PI_5 0.30901699437494742410229341718281905886
#define FSEI_COS_4PI_5 -0.80901699437494742410229341718281905886
#define FSEI_SIN_2PI_5 0.95105651629515357211643933337938214340
#define FSEI_SIN_4PI_5 0.58778525229247312916870595463907276860
template <bool INV> struct SmallDft<5, INV> {
    static FSEI_HD void run(cplx* v) {
        const cplx a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]), b1 = csub(v[1], v[4]), b2 = csub(v[2], v[3]);
        const cplx m1 = cmake(v[0].re + FSEI_COS_2PI_5 * a1.re + FSEI_COS_4PI_5 * a2.re, v[0].im + FSEI_COS_2PI_5 * a1.im + FSEI_COS_4PI_5 * a2.im);
        const cplx m2 = cmake(v[0].re + FSEI_COS_4PI_5 * a1.re + FSEI_COS_2PI_5 * a2.re, v[0].im + FSEI_COS_4PI_5 * a1.im + FSEI_COS_2PI_5 * a2.im);
        // (-+ i) (s1 b1 + s2 b2) and (-+ i) (s2 b1 - s1 b2)
        const cplx n1 = crot<INV>(cmake(FSEI_SIN_2PI_5 * b1.re + FSEI_SIN_4PI_5 * b2.re, FSEI_SIN_2PI_5 * b1.im + FSEI_SIN_4PI_5 * b2.im));
        const cplx n2 = crot<INV>(cmake(FSEI_SIN_4PI_5 * b1.re - FSEI_SIN_2PI_5 * b2.re, FSEI_SIN_4PI_5 * b1.im - FSEI_SIN_2PI_5 * b2.im));
        v[0] = cadd(v[0], cadd(a1, a2));
        v[1] = cadd(m1, n1); v[4] = csub(m1, n1);
        v[2] = cadd(m2, n2); v[3] = csub(m2, n2);
    }
};
template <bool INV> struct SmallDft<4, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]), t2 = cadd(v[1], v[3]), t3 = crot<INV>(csub(v[1], v[3]));
        v[0] = cadd(t0, t2); v[1] = cadd(t1, t3); v[2] = csub(t0, t2); v[3] = csub(t1, t3);
    }
};
template <bool INV> struct SmallDft<8, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
        SmallDft<4, INV>::run(e); SmallDft<4, INV>::run(o);
        o[1] = ctw<INV>(o[1], FSEI_SQRT1_2, -FSEI_SQRT1_2);
        o[2] = crot<INV>(o[2]);
        o[3] = ctw<INV>(o[3], -FSEI_SQRT1_2, -FSEI_SQRT1_2);
#pragma unroll
        for (int k = 0; k < 4; k++) { v[k] = cadd(e[k], o[k]); v[k + 4] = csub(e[k], o[k]); }
    }
};
template <bool INV> struct SmallDft<16, INV> {
    static FSEI_HD void run(cplx* v) {
        // n = 4 n1 + n2, k = k1 + 4 k2
        cplx y[4][4];                                  // y[n2][k1]
#pragma unroll
        for (int n2 = 0; n2 < 4; n2++) {
            cplx t[4] = {v[n2], v[4 + n2], v[8 + n2], v[12 + n2]};
            SmallDft<4, INV>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < 4; k1++) y[n2][k1] = t[k1];
        }
        // twiddles w16^{n2 k1}
        const double c1 = FSEI_COS_PI_8, s1 = FSEI_SIN_PI_8, h = FSEI_SQRT1_2;
        y[1][1] = ctw<INV>(y[1][1], c1, -s1); y[1][2] = ctw<INV>(y[1][2], h, -h);   y[1][3] = ctw<INV>(y[1][3], s1, -c1);
        y[2][1] = ctw<INV>(y[2][1], h, -h);   y[2][2] = crot<INV>(y[2][2]);          y[2][3] = ctw<INV>(y[2][3], -h, -h);
        y[3][1] = ctw<INV>(y[3][1], s1, -c1); y[3][2] = ctw<INV>(y[3][2], -h, -h);   y[3][3] = ctw<INV>(y[3][3], -c1, s1);
#pragma unroll
        for (int k1 = 0; k1 < 4; k1++) {
            cplx t[4] = {y[0][k1], y[1][k1], y[2][k1], y[3][k1]};
            SmallDft<4, INV>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < 4; k2++) v[k1 + 4 * k2] = t[k2];
        }
    }
};

// ---- one butterfly of one pass on a tile ------------------------------------------------------
// A(n) maps a logical index of the line to its element in `sm`.  tw[m] = e^{-2 pi i m / N}.
// tmul = N / Ns.  Forward (INV=false): DFT then twiddle; inverse: conj twiddle then conj DFT.
template <int R, bool INV, class Addr>
FSEI_HD void fft_butterfly(cplx* sm, const Addr& A, int blk, int n2, int Ns, int M, int tmul, const cplx* tw)
{
    cplx v[R];
    const int base = blk * Ns + n2;
#pragma unroll
    for (int q = 0; q < R; q++) v[q] = sm[A(base + q * M)];
    if (INV && M > 1) {
#pragma unroll
        for (int q = 1; q < R; q++) { cplx w = tw[tmul * n2 * q]; v[q] = cmulc(v[q], w); }
    }
    SmallDft<R, INV>::run(v);
    if (!INV && M > 1) {
#pragma unroll
        for (int q = 1; q < R; q++) { cplx w = tw[tmul * n2 * q]; v[q] = cmul(v[q], w); }
    }
#pragma unroll
    for (int q = 0; q < R; q++) sm[A(base + q * M)] = v[q];
}

// Pass description shared by host (plan) and device.
struct FftPlan1D {
    int N;            // complex length
    int npass;
    int radix[8];
};

}  // namespace fsei
