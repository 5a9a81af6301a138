// fast_visc.cu -- instantiations, host-side line tables and launchers of the fast viscous family (visc_fast.cuh).
#include <cuda_runtime.h>
#include <cmath>
#include "visc_fast.cuh"
#include "fast_launch.hpp"
#include "tma_host.hpp"

namespace fsei {

#ifndef FSEI_VA_TMA
#define FSEI_VA_TMA 1               // chunk lengths 8, 16, 24, 32 take the tensor-map variant of pass A
#endif
#define FSEI_VA_TMA_ON (FSEI_VA_TMA != 0)

// chunk lengths with an instantiation: pass A needs M % 4 == 0 (conflict-free 128-bit slots; 2 for small test grids)
#define FSEI_VA_LIST(X) X(2) X(4) X(8) X(12) X(16) X(24) X(32) X(10) X(20) X(18) X(30)
#define FSEI_VB_LIST(X) X(2) X(3) X(4) X(6) X(8) X(12) X(16) X(24) X(32) X(5) X(10) X(20) X(18) X(30)

// z-slabs: pass A only in its tensor-map variant (chunk lengths 8, 16, 24, 32)
bool visc_fast_slab_supported(int nx, int ny)
{
    const int M = nx / 32;
    return visc_fast_supported(nx, ny) && M % 8 == 0 && M <= 32 && FSEI_VA_TMA_ON;
}

bool visc_fast_supported(int nx, int ny)
{
    if (nx % 32 || ny % 32 || nx % 8) return false;
    bool a = false, b = false;
#define X(M) if (nx / 32 == M) a = true;
    FSEI_VA_LIST(X)
#undef X
#define X(M) if (ny / 32 == M) b = true;
    FSEI_VB_LIST(X)
#undef X
    return a && b;
}

static size_t vb_smem(int M) { return 128 + (size_t)2 * 32 * M * 64 + (size_t)M * 256 * 8; }
static size_t va_smem(int M) { return (size_t)FSEI_VA_WPB * (FSEI_VA_STAGES * 32 * (8 * M + 16) + 64); }
static size_t va_tma_smem(int M) { return 1024 + (size_t)FSEI_VA_TMA_WPB * (FSEI_VA_STAGES * 256 * M + 64); }
#ifndef FSEI_VA_TMA
#define FSEI_VA_TMA 1               // chunk lengths 8, 16, 24, 32 take the tensor-map variant of pass A
#endif

cudaError_t visc_fast_init()
{
    cudaError_t e = cudaSuccess;
#define X(M) if (e == cudaSuccess) e = kernel_smem(k_visc_xz<M>, (int)va_smem(M));
    FSEI_VA_LIST(X)
#undef X
    if (e == cudaSuccess) e = kernel_smem(k_visc_xz_tma<8>, (int)va_tma_smem(8));
    if (e == cudaSuccess) e = kernel_smem(k_visc_xz_tma<16>, (int)va_tma_smem(16));
    if (e == cudaSuccess) e = kernel_smem(k_visc_xz_tma<24>, (int)va_tma_smem(24));
    if (e == cudaSuccess) e = kernel_smem(k_visc_xz_tma<32>, (int)va_tma_smem(32));
#define X(M) if (e == cudaSuccess) e = kernel_smem(k_visc_zy<M>, (int)vb_smem(M));
    FSEI_VB_LIST(X)
#undef X
    return e;
}

// Tables of one uniform periodic line of n = 32 M unknowns, (1 + 2r) on the diagonal and -r beside it, in long double
void visc_fast_line(int n, double h_recip, double beta, VFastLine* out)
{
    const int M = n / 32, Mi = M - 1;
    const long double r = (long double)beta * (long double)h_recip * (long double)h_recip, b = 1.0L + 2.0L * r;
    long double ip[32], cp[32], ls[32], rs[32];
    // interior factorisation: piv_0 = b, piv_i = b - (-r) c'_{i-1}, c'_i = -r / piv_i
    for (int i = 0; i < Mi; i++) {
        const long double piv = i == 0 ? b : b + r * cp[i - 1];
        ip[i] = 1.0L / piv; cp[i] = -r * ip[i];
    }
    // spikes: T ls = r e_0, T rs = r e_{Mi-1}
    for (int which = 0; which < 2; which++) {
        long double y[32];
        for (int i = 0; i < Mi; i++) {
            const long double d = ((which == 0 && i == 0) || (which == 1 && i == Mi - 1)) ? r : 0.0L;
            y[i] = (i == 0 ? d : d + r * y[i - 1]) * ip[i];
        }
        for (int i = Mi - 2; i >= 0; i--) y[i] -= cp[i] * y[i + 1];
        for (int i = 0; i < Mi; i++) (which == 0 ? ls : rs)[i] = y[i];
    }
    // separator system: circulant tridiagonal, diag sd, off-diagonals so (both sides); dense solve S z = e_0
    long double sd = b, so = -r;
    if (Mi > 0) { sd = b - r * (rs[Mi - 1] + ls[0]); so = -r * ls[Mi - 1]; }
    long double S[32][33];
    for (int p = 0; p < 32; p++) {
        for (int q = 0; q < 33; q++) S[p][q] = 0.0L;
        S[p][p] += sd; S[p][(p + 1) & 31] += so; S[p][(p + 31) & 31] += so;
    }
    S[0][32] = 1.0L;
    for (int c = 0; c < 32; c++) {
        int piv = c;
        for (int p = c + 1; p < 32; p++) if (fabsl(S[p][c]) > fabsl(S[piv][c])) piv = p;
        if (piv != c) for (int q = 0; q < 33; q++) { const long double t = S[c][q]; S[c][q] = S[piv][q]; S[piv][q] = t; }
        for (int p = c + 1; p < 32; p++) {
            const long double m = S[p][c] / S[c][c];
            if (m != 0.0L) for (int q = c; q < 33; q++) S[p][q] -= m * S[c][q];
        }
    }
    long double z[32];
    for (int c = 31; c >= 0; c--) {
        long double s = S[c][32];
        for (int q = c + 1; q < 32; q++) s -= S[c][q] * z[q];
        z[c] = s / S[c][c];
    }
    out->r = (double)r;
    for (int i = 0; i < 31; i++) {
        out->ip[i] = i < Mi ? (double)ip[i] : 0.0; out->cp[i] = i < Mi ? (double)cp[i] : 0.0;
        out->ls[i] = i < Mi ? (double)ls[i] : 0.0; out->rs[i] = i < Mi ? (double)rs[i] : 0.0;
    }
    for (int s = 0; s < 32; s++) out->sinv[s] = (double)z[s];      // S^-1[p][q] = z[(p - q) mod 32]; z[s] = z[32 - s]
}

// number of terms of sinv on either side of s = 0 that can reach the last bit of sum_s sinv[s] g_{p-s}:
// |sinv[s]| decays geometrically away from s = 0; terms below 2^-70 of the largest are dropped (exact to rounding:
// with |g| bounded by 32 max|g| cancellation such a term is < 2^-65 ulp-relative of the separator value)
int visc_fast_nsig(const VFastLine& L)
{
    double mx = 0.0;
    for (int s = 0; s < 32; s++) mx = std::fmax(mx, std::fabs(L.sinv[s]));
    int n = 0;
    for (int s = 1; s <= 16; s++) if (std::fabs(L.sinv[s]) > mx * 0x1p-70) n = s;
    return n;
}

cudaError_t launch_visc_xz(const VFastArgs& A, cudaStream_t st)
{
    const dim3 grid((A.ny + FSEI_VA_WPB - 1) / FSEI_VA_WPB, 3);
    const int M = A.nx / 32;
    if (A.slab && !(FSEI_VA_TMA && M % 8 == 0 && M <= 32 && (size_t)32 * A.ny * A.nz < (1ull << 31))) return cudaErrorInvalidValue;
    if (FSEI_VA_TMA && M % 8 == 0 && M <= 32 && ((size_t)32 * A.ny * A.nz < (1ull << 31) || A.slab)) {
        EncodeTiledFn fn = tma_encode_fn();
        if (!fn) return cudaErrorNotSupported;
        VFastMapsA Mp;
        for (int c = 0; c < 3; c++) {                               // the field as [32 ny nz chunks][M doubles]
            cuuint64_t dims[2] = {(cuuint64_t)M, (cuuint64_t)32 * A.ny * A.nz};
            cuuint64_t strides[1] = {(cuuint64_t)M * sizeof(double)};
            const bool wide = M % 16 == 0;                        // 128-byte boxes and swizzle, else 64-byte
            cuuint32_t box[2] = {wide ? 16u : 8u, 32u}, estr[2] = {1, 1};
            if (fn(&Mp.r[c].m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, A.r[c], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   wide ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                return cudaErrorInvalidValue;
        }
        const dim3 gt((A.ny + FSEI_VA_TMA_WPB - 1) / FSEI_VA_TMA_WPB, 3);
        switch (M) {
            case 8: k_visc_xz_tma<8><<<gt, 32 * FSEI_VA_TMA_WPB, va_tma_smem(8), st>>>(A, Mp); break;
            case 16: k_visc_xz_tma<16><<<gt, 32 * FSEI_VA_TMA_WPB, va_tma_smem(16), st>>>(A, Mp); break;
            case 24: k_visc_xz_tma<24><<<gt, 32 * FSEI_VA_TMA_WPB, va_tma_smem(24), st>>>(A, Mp); break;
            default: k_visc_xz_tma<32><<<gt, 32 * FSEI_VA_TMA_WPB, va_tma_smem(32), st>>>(A, Mp); break;
        }
        return cudaGetLastError();
    }
    switch (A.nx / 32) {
#define X(M) case M: k_visc_xz<M><<<grid, 32 * FSEI_VA_WPB, va_smem(M), st>>>(A); break;
        FSEI_VA_LIST(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// 2-D fp64 view of a field: inner dimension nx doubles, outer ny nz rows; box = 8 doubles x box_rows rows
static cudaError_t field_map(const VFastArgs& A, int box_rows, double* f, TmaMap2D* out)
{
    EncodeTiledFn fn = tma_encode_fn();
    if (!fn) return cudaErrorNotSupported;
    cuuint64_t dims[2] = {(cuuint64_t)A.nx, (cuuint64_t)A.ny * A.nz};
    cuuint64_t strides[1] = {(cuuint64_t)A.nx * sizeof(double)};
    cuuint32_t box[2] = {8u, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(&out->m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, f, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t launch_visc_zy(const VFastArgs& A, cudaStream_t st)
{
    const dim3 grid(A.split ? 3 * (A.nx / 8) : A.nx / 8);
    VFastMaps Mp;
    Mp.box_rows = 256;
    while (A.ny % Mp.box_rows) Mp.box_rows--;                   // largest divisor of ny that fits a TMA box
    for (int c = 0; c < 3; c++) {
        cudaError_t e = field_map(A, Mp.box_rows, A.r[c], &Mp.d[c]);
        if (e == cudaSuccess) e = field_map(A, Mp.box_rows, A.slab ? A.r[c] : A.q[c], &Mp.q[c]);
        if (e != cudaSuccess) return e;
    }
    switch (A.ny / 32) {
#define X(M) case M: k_visc_zy<M><<<grid, 256, vb_smem(M), st>>>(A, Mp); break;
        FSEI_VB_LIST(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace fsei
