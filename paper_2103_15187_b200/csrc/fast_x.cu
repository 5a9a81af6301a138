// fast_x.cu -- instantiations and launchers of the fast x-direction kernels (xfast.cuh).
#include "fast_launch.hpp"
#include "fast_configs.hpp"
#include "tma_host.hpp"

namespace fsei {


bool xfast_supported(int N)
{
    switch (N) {
#define X(n, a, b, c) case n:
        FSEI_X_CONFIGS(X)
#undef X
        return true;
        default: return false;
    }
}

int xfast_lines_per_block(int N, bool neu)
{
    switch (N) {
#define X(n, a, b, c) case n: return neu ? XShape<FftCfg<n, a, b, c>, true>::LPB : XShape<FftCfg<n, a, b, c>, false>::LPB;
        FSEI_X_CONFIGS(X)
#undef X
        default: return 1;
    }
}

template <class C, bool NEU> static cudaError_t init_one()
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    const int bf = (int)XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, b1 = (int)XSmemLayout<C, LPB, NEU, LPB>::BYTES;
    cudaError_t e;
    if ((e = kernel_smem(k_xf_fast<C, LPB, NEU, true>, bf))) return e;
    if ((e = kernel_smem(k_xf_fast<C, LPB, NEU, false>, b1))) return e;
    return kernel_smem(k_xi_fast<C, LPB, NEU>, b1);
}

template <class C, bool NEU> static cudaError_t init_one_blocked()
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    const int bf = (int)XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, b1 = (int)XSmemLayout<C, LPB, NEU, LPB>::BYTES;
    cudaError_t e;
    if ((e = kernel_smem(k_xf_fast<C, LPB, NEU, true, FSEI_CB>, bf))) return e;
    if ((e = kernel_smem(k_xf_fast<C, LPB, NEU, false, FSEI_CB>, b1))) return e;
    return kernel_smem(k_xi_fast<C, LPB, NEU, FSEI_CB>, b1);
}

bool xblocked_supported(int N)
{
    switch (N) {
#define X(n, a, b, c) case n:
        FSEI_XB_CONFIGS(X)
#undef X
        return true;
        default: return false;
    }
}

cudaError_t xblocked_init()
{
    cudaError_t e;
#define X(n, a, b, c) \
    if ((e = init_one_blocked<FftCfg<n, a, b, c>, false>())) return e; \
    if ((e = init_one_blocked<FftCfg<n, a, b, c>, true>())) return e;
    FSEI_XB_CONFIGS(X)
#undef X
    return cudaSuccess;
}

// 3-D fp64 view of the blocked spectrum [N / CB][nz][ny][CB] complex: (2 ny CB doubles, nz, N / CB);
// box = (2 LPB CB doubles, 1 plane, xi_box_tiles(N / CB) tiles)
template <class C, bool NEU> static cudaError_t xi_map_one(const XFast& P, const cplx* spec, TmaMap3D* out)
{
    constexpr int LPB = XShape<C, NEU>::LPB, CB = FSEI_CB, NXT = C::N / CB;
    EncodeTiledFn fn = tma_encode_fn();
    if (!fn) return cudaErrorNotSupported;
    cuuint64_t dims[3] = {(cuuint64_t)2 * P.ny * CB, (cuuint64_t)P.nz, (cuuint64_t)NXT};
    cuuint64_t strides[2] = {(cuuint64_t)P.ny * CB * sizeof(cplx), (cuuint64_t)P.nz * P.ny * CB * sizeof(cplx)};
    cuuint32_t box[3] = {(cuuint32_t)(2 * LPB * CB), 1u, (cuuint32_t)xi_box_tiles(NXT)};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(&out->m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<cplx*>(spec), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t make_xi_blocked_map(const XFast& P, bool neu, const cplx* spec, TmaMap3D* out)
{
    switch (P.N) {
#define X(n, a, b, c) case n: return neu ? xi_map_one<FftCfg<n, a, b, c>, true>(P, spec, out) : xi_map_one<FftCfg<n, a, b, c>, false>(P, spec, out);
        FSEI_XB_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t xfast_init()
{
    cudaError_t e;
#define X(n, a, b, c) \
    if ((e = init_one<FftCfg<n, a, b, c>, false>())) return e; \
    if ((e = init_one<FftCfg<n, a, b, c>, true>())) return e;
    FSEI_X_CONFIGS(X)
#undef X
    return cudaSuccess;
}

template <class C, bool NEU, int CB = 0> static cudaError_t xf_one(const XFast& P, const SParams& S, bool fused, const double* u, const double* v,
                                                       const double* w, double inv_adt, cplx* spec, cudaStream_t st)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    if (fused) k_xf_fast<C, LPB, NEU, true, CB><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, st>>>(P, S, u, v, w, inv_adt, spec);
    else k_xf_fast<C, LPB, NEU, false, CB><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, st>>>(P, S, u, v, w, inv_adt, spec);
    return cudaGetLastError();
}

cudaError_t launch_xf_fast(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v,
                           const double* w, double inv_adt, cplx* spec, cudaStream_t st, bool blocked)
{
    if (blocked) switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xf_one<FftCfg<n, a, b, c>, true, FSEI_CB>(P, S, fused, u, v, w, inv_adt, spec, st) \
                           : xf_one<FftCfg<n, a, b, c>, false, FSEI_CB>(P, S, fused, u, v, w, inv_adt, spec, st);
        FSEI_XB_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xf_one<FftCfg<n, a, b, c>, true>(P, S, fused, u, v, w, inv_adt, spec, st) \
                           : xf_one<FftCfg<n, a, b, c>, false>(P, S, fused, u, v, w, inv_adt, spec, st);
        FSEI_X_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

template <class C, bool NEU, int CB = 0> static cudaError_t xi_one(const XFast& P, const cplx* spec, double* phi, cudaStream_t st, const TmaMap3D* map)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    static const TmaMap3D none{};
    k_xi_fast<C, LPB, NEU, CB><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, st>>>(P, map ? *map : none, spec, phi);
    return cudaGetLastError();
}

cudaError_t launch_xi_fast(const XFast& P, bool neu, const cplx* spec, double* phi, cudaStream_t st, const TmaMap3D* map)
{
    if (map) switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xi_one<FftCfg<n, a, b, c>, true, FSEI_CB>(P, spec, phi, st, map) : xi_one<FftCfg<n, a, b, c>, false, FSEI_CB>(P, spec, phi, st, map);
        FSEI_XB_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
    switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xi_one<FftCfg<n, a, b, c>, true>(P, spec, phi, st, nullptr) : xi_one<FftCfg<n, a, b, c>, false>(P, spec, phi, st, nullptr);
        FSEI_X_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace fsei
