/*
 * gen.c -- seeded synthetic INPUT generators.
 *
 * Serves both the CUDA path's tests/bench and the oracle's tests.  Holds none of
 * the method's arithmetic: only a counter-based random stream and a separable
 * sum of products used to lay down smooth fields.  Values are produced once on
 * the host; both sides then see identical bits.
 *
 * Stream: splitmix64 started at state s0 = seed*2^32 + stream; element `idx`
 * uses outputs number 2*idx and 2*idx+1 of that sequence (order-independent, so
 * the loop parallelises).  Normal deviates by Box-Muller from two 53-bit uniforms.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#define GAMMA 0x9E3779B97F4A7C15ULL

static inline uint64_t sm64_out(uint64_t s0, uint64_t n)   /* n-th output (n = 0,1,..) of splitmix64(s0) */
{
    uint64_t z = s0 + (n + 1) * GAMMA;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t fsei_gen_raw(uint64_t seed, uint64_t stream, uint64_t n)
{
    return sm64_out((seed << 32) + stream, n);
}

/* out[i] = (accumulate ? out[i] : 0) + sigma * N(0,1)_i */
void fsei_gen_normal(uint64_t seed, uint64_t stream, size_t n, double sigma, int accumulate, double *out)
{
    const uint64_t s0 = (seed << 32) + stream;
    const double two_pi = 6.283185307179586476925286766559;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; i++) {
        uint64_t a = sm64_out(s0, 2 * (uint64_t)i), b = sm64_out(s0, 2 * (uint64_t)i + 1);
        double u1 = ((double)(a >> 11) + 1.0) * 0x1.0p-53;      /* (0,1] */
        double u2 = (double)(b >> 11) * 0x1.0p-53;              /* [0,1) */
        double g = sqrt(-2.0 * log(u1)) * cos(two_pi * u2);
        out[i] = (accumulate ? out[i] : 0.0) + sigma * g;
    }
}

/* out[k][j][i] = sum_m amp[m] * fx[m][i] * fy[m][j] * fz[m][k]   (m ascending) */
void fsei_gen_separable(int nx, int ny, int nz, int M, const double *amp,
                        const double *fx, const double *fy, const double *fz, double *out)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++) {
            double *row = out + ((size_t)k * ny + j) * nx;
            for (int i = 0; i < nx; i++) row[i] = 0.0;
            for (int m = 0; m < M; m++) {
                double c = amp[m] * fy[(size_t)m * ny + j] * fz[(size_t)m * nz + k];
                const double *f = fx + (size_t)m * nx;
                for (int i = 0; i < nx; i++) row[i] += c * f[i];
            }
        }
}
