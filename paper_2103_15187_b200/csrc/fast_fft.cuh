// fast_fft.cuh -- register-resident Stockham passes shared by the fast x and y transforms.
//
// Fast path (x and y periodic, power-of-two lengths): a line of N complex values is transformed
// by NP <= 3 radix passes (radices R0 R1 R2 from {2,4,8,16}).  Pass s with Ns = R0..R_{s-1}:
// butterfly b in [0, N/R) reads elements b + q N/R (q < R), multiplies element q by
// w_{Ns R}^{q (b mod Ns)}, takes the R-point DFT in registers and writes output q to
// (b / Ns) Ns R + (b mod Ns) + q Ns  (Stockham autosort: natural order in, natural order out,
// every pass reads with unit stride across threads).  The first pass reads global memory, the last
// writes it; in between the data sits in shared memory, alternating between two buffers so that one
// barrier per pass is enough.  Twiddles come from per-pass shared-memory tables laid out [q-1][m]
// (conflict-free for consecutive m).  Conventions as in fft_core.cuh (R15).
#pragma once
#include "fft_core.cuh"

namespace fsei {

template <int N_, int R0_, int R1_, int R2_> struct FftCfg {
    static constexpr int N = N_, R0 = R0_, R1 = R1_, R2 = R2_;
    static_assert(R0_ * R1_ * R2_ == N_, "radices must multiply to N");
    static constexpr int NP = 1 + (R1_ > 1) + (R2_ > 1);
    static constexpr int RMAX = (R0_ > R1_ ? (R0_ > R2_ ? R0_ : R2_) : (R1_ > R2_ ? R1_ : R2_));
    static constexpr int T = N_ / RMAX;                 // threads per line
    static constexpr int E = RMAX;                      // elements per thread
    static constexpr int TW1 = (R1_ > 1) ? (R1_ - 1) * R0_ : 0;          // table sizes (complex)
    static constexpr int TW2 = (R2_ > 1) ? (R2_ - 1) * R0_ * R1_ : 0;
    static constexpr int TW = TW1 + TW2;
};

// shared-memory index padding for 16-byte elements: one extra slot every 8
__host__ __device__ __forceinline__ constexpr int padi(int n) { return n + (n >> 3); }

// One pass for one thread.  in(n) -> cplx, out(n, cplx).  tl = thread index within the line.
template <int N, int R, int NS, int T, bool INV, class In, class Out>
__device__ __forceinline__ void fft_pass(int tl, const cplx* __restrict__ tw, In in, Out out)
{
    constexpr int NB = N / R;                 // butterflies per line
    constexpr int PER = (NB + T - 1) / T;     // butterflies per thread
    cplx v[PER][R];
#pragma unroll
    for (int i = 0; i < PER; i++) {
        const int b = tl + i * T;
        if (NB % T == 0 || b < NB) {
#pragma unroll
            for (int q = 0; q < R; q++) v[i][q] = in(b + q * NB);
        }
    }
#pragma unroll
    for (int i = 0; i < PER; i++) {
        const int b = tl + i * T;
        if (NB % T == 0 || b < NB) {
            if (NS > 1) {
                const int m = b % NS;
#pragma unroll
                for (int q = 1; q < R; q++) {
                    const cplx w = tw[(q - 1) * NS + m];
                    v[i][q] = INV ? cmulc(v[i][q], w) : cmul(v[i][q], w);
                }
            }
            SmallDft<R, INV>::run(v[i]);
            const int j0 = (b / NS) * NS * R + (b % NS);
#pragma unroll
            for (int q = 0; q < R; q++) out(j0 + q * NS, v[i][q]);
        }
    }
}

struct SmIn {
    const cplx* s;
    __device__ __forceinline__ cplx operator()(int n) const { return s[padi(n)]; }
};
struct SmOut {
    cplx* s;
    __device__ __forceinline__ void operator()(int n, cplx v) const { s[padi(n)] = v; }
};

// Whole line: first pass from `in`, last pass to `out`, shared buffers bufA/bufB (each padi(N)+1 complex
// for this line).  tws: shared twiddle tables [TW1 | TW2].  Must be called by all threads of the CTA
// (contains __syncthreads()).
template <class C, bool INV, class In, class Out>
__device__ __forceinline__ void fft_line(int tl, cplx* bufA, cplx* bufB, const cplx* tws, In in, Out out)
{
    if (C::NP == 1) {
        fft_pass<C::N, C::R0, 1, C::T, INV>(tl, nullptr, in, out);
    } else if (C::NP == 2) {
        fft_pass<C::N, C::R0, 1, C::T, INV>(tl, nullptr, in, SmOut{bufA});
        __syncthreads();
        fft_pass<C::N, C::R1, C::R0, C::T, INV>(tl, tws, SmIn{bufA}, out);
    } else {
        fft_pass<C::N, C::R0, 1, C::T, INV>(tl, nullptr, in, SmOut{bufA});
        __syncthreads();
        fft_pass<C::N, C::R1, C::R0, C::T, INV>(tl, tws, SmIn{bufA}, SmOut{bufB});
        __syncthreads();
        fft_pass<C::N, C::R2, C::R0 * C::R1, C::T, INV>(tl, tws + C::TW1, SmIn{bufB}, out);
    }
}

}  // namespace fsei
