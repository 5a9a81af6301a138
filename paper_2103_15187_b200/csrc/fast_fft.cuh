// fast_fft.cuh -- register-resident Stockham passes shared by the fast x and y transforms.
//
// Fast path (lengths 2^a and 3*2^a, a line of N complex values): N = R0 R1 R2 with radices from
// {2,4,5,6,8,10,12,16}.  Pass s with Ns = R0..R_{s-1}: butterfly b in [0, N/R) reads elements b + q N/R
// (q < R), multiplies element q by w_{Ns R}^{q (b mod Ns)}, takes the R-point DFT in registers and
// writes output q to (b / Ns) Ns R + (b mod Ns) + q Ns  (Stockham autosort: natural order in, natural
// order out, every pass reads with unit stride across threads).  The first pass reads global memory
// (or a staging tile), the last writes global memory (or a tile for the pair post-processing); in
// between the data sits in ONE shared buffer (read -> barrier -> write -> barrier).  Twiddles come
// from per-pass shared-memory tables laid out [q-1][m] (unit stride across threads).
// Conventions as in fft_core.cuh (R15): forward e^{-i..} unnormalised, the inverse is the
// conjugate pass sequence without 1/N.
#pragma once
#include "fft_core.cuh"
#include "kernel_env.cuh"

namespace fsei {

// 6 = 3 x 2:  n = 2 n1 + n2,  k = k1 + 3 k2
template <bool INV> struct SmallDft<6, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx e[3] = {v[0], v[2], v[4]}, o[3] = {v[1], v[3], v[5]};
        SmallDft<3, INV>::run(e); SmallDft<3, INV>::run(o);
        o[1] = ctw<INV>(o[1], 0.5, -FSEI_SQRT3_2);
        o[2] = ctw<INV>(o[2], -0.5, -FSEI_SQRT3_2);
#pragma unroll
        for (int k = 0; k < 3; k++) { v[k] = cadd(e[k], o[k]); v[k + 3] = csub(e[k], o[k]); }
    }
};

// 10 = 5 x 2:  n = 2 n1 + n2,  k = k1 + 5 k2
#define FSEI_COS_PI_5 0.80901699437494742410229341718281905886
#define FSEI_SIN_PI_5 0.58778525229247312916870595463907276860
template <bool INV> struct SmallDft<10, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx e[5] = {v[0], v[2], v[4], v[6], v[8]}, o[5] = {v[1], v[3], v[5], v[7], v[9]};
        SmallDft<5, INV>::run(e); SmallDft<5, INV>::run(o);
        o[1] = ctw<INV>(o[1], FSEI_COS_PI_5, -FSEI_SIN_PI_5);
        o[2] = ctw<INV>(o[2], FSEI_COS_2PI_5, -FSEI_SIN_2PI_5);
        o[3] = ctw<INV>(o[3], -FSEI_COS_2PI_5, -FSEI_SIN_2PI_5);
        o[4] = ctw<INV>(o[4], -FSEI_COS_PI_5, -FSEI_SIN_PI_5);
#pragma unroll
        for (int k = 0; k < 5; k++) { v[k] = cadd(e[k], o[k]); v[k + 5] = csub(e[k], o[k]); }
    }
};

// 12 = 3 x 4:  n = 4 n1 + n2,  k = k1 + 3 k2
template <bool INV> struct SmallDft<12, INV> {
    static FSEI_HD void run(cplx* v) {
        cplx y[4][3];                                  // y[n2][k1]
#pragma unroll
        for (int n2 = 0; n2 < 4; n2++) {
            cplx t[3] = {v[n2], v[4 + n2], v[8 + n2]};
            SmallDft<3, INV>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < 3; k1++) y[n2][k1] = t[k1];
        }
        // twiddles w12^{n2 k1}
        y[1][1] = ctw<INV>(y[1][1], FSEI_SQRT3_2, -0.5);  y[1][2] = ctw<INV>(y[1][2], 0.5, -FSEI_SQRT3_2);
        y[2][1] = ctw<INV>(y[2][1], 0.5, -FSEI_SQRT3_2);  y[2][2] = ctw<INV>(y[2][2], -0.5, -FSEI_SQRT3_2);
        y[3][1] = crot<INV>(y[3][1]);                     y[3][2] = cmake(-y[3][2].re, -y[3][2].im);
#pragma unroll
        for (int k1 = 0; k1 < 3; k1++) {
            cplx t[4] = {y[0][k1], y[1][k1], y[2][k1], y[3][k1]};
            SmallDft<4, INV>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < 4; k2++) v[k1 + 3 * k2] = t[k2];
        }
    }
};

constexpr int ilog2c(int n) { return n <= 1 ? 0 : 1 + ilog2c(n >> 1); }

template <int N_, int R0_, int R1_, int R2_> struct FftCfg {
    static constexpr int N = N_, R0 = R0_, R1 = R1_, R2 = R2_;
    static_assert(R0_ * R1_ * R2_ == N_, "radices must multiply to N");
    static constexpr int NP = 1 + (R1_ > 1) + (R2_ > 1);
    static constexpr int RMAX = (R0_ > R1_ ? (R0_ > R2_ ? R0_ : R2_) : (R1_ > R2_ ? R1_ : R2_));
    static constexpr int T = N_ / RMAX;                 // threads per line
    static constexpr int TW1 = (R1_ > 1) ? (R1_ - 1) * R0_ : 0;          // twiddle table sizes (complex)
    static constexpr int TW2 = (R2_ > 1) ? (R2_ - 1) * R0_ * R1_ : 0;
    static constexpr int TW = TW1 + TW2;
    // shared-memory index padding: one extra element every R0 (R0 a power of two): makes the stride-R0
    // writes of the first pass conflict-free for 16-byte elements and keeps aligned groups of 8 whole
    static constexpr int PSH = ilog2c(R0_);
    static_assert((1 << PSH) == R0_ || NP == 1, "first radix must be a power of two");
    static FSEI_HD int pad(int n) { return n + (n >> PSH); }
    static constexpr int PITCH = N_ + (N_ >> PSH) + 1;  // complex elements per padded line
};

// per-pass twiddle tables in shared memory: tws[(q-1) NS + m] = e^{-2 pi i q m / (NS R)}, from the plan's
// table tw[j] = e^{-2 pi i j / N}.  Called by all threads of the CTA (no barrier inside).
template <class C> FSEI_DEV void fft_fill_twiddles(cplx* tws, const cplx* tw, int tid, int nt)
{
    if (C::NP >= 2) {
        constexpr int NS = C::R0, R = C::R1;
        for (int i = tid; i < (R - 1) * NS; i += nt) { int q = i / NS + 1, m = i % NS; tws[i] = tw[q * m * (C::N / (NS * R))]; }
    }
    if (C::NP >= 3) {
        constexpr int NS = C::R0 * C::R1, R = C::R2;
        for (int i = tid; i < (R - 1) * NS; i += nt) { int q = i / NS + 1, m = i % NS; tws[C::TW1 + i] = tw[q * m * (C::N / (NS * R))]; }
    }
}

// Pass s of one line for one thread: tl = thread index within the line (T threads per line).
// in(n) -> cplx, out(n, cplx, slot) with slot = i R + q the (compile-time) register index of the value; `active` false = the thread's line does not exist (ragged tile).
template <int N, int R, int NS, int T> struct PassShape {
    static constexpr int NB = N / R;                  // butterflies per line
    static constexpr int PER = (NB + T - 1) / T;      // butterflies per thread
    static constexpr bool FULL = (NB % T == 0);
};

template <int N, int R, int NS, int T, class In>
FSEI_DEV void fft_pass_load(int tl, In in, cplx (*v)[R])
{
    using S = PassShape<N, R, NS, T>;
#pragma unroll
    for (int i = 0; i < S::PER; i++) {
        const int b = tl + i * T;
        if (S::FULL || b < S::NB) {
#pragma unroll
            for (int q = 0; q < R; q++) v[i][q] = in(b + q * S::NB);
        }
    }
}

template <int N, int R, int NS, int T, bool INV, class Out>
FSEI_DEV void fft_pass_compute(int tl, const cplx* tw, cplx (*v)[R], Out out)
{
    using S = PassShape<N, R, NS, T>;
    // twiddle loads of every butterfly first (shared-memory loads cannot be hoisted over the stores below)
    if (NS > 1) {
#pragma unroll
        for (int i = 0; i < S::PER; i++) {
            const int b = tl + i * T;
            if (S::FULL || b < S::NB) {
                const int m = b % NS;
#pragma unroll
                for (int q = 1; q < R; q++) {
                    const cplx w = tw[(q - 1) * NS + m];
                    v[i][q] = INV ? cmulc(v[i][q], w) : cmul(v[i][q], w);
                }
            }
        }
    }
#pragma unroll
    for (int i = 0; i < S::PER; i++) {
        const int b = tl + i * T;
        if (S::FULL || b < S::NB) {
            const int m = b % NS;
            SmallDft<R, INV>::run(v[i]);
            const int j0 = (b / NS) * NS * R + m;
#pragma unroll
            for (int q = 0; q < R; q++) out(j0 + q * NS, v[i][q], i * R + q);      // slot = register index of the value
        }
    }
}

}  // namespace fsei
