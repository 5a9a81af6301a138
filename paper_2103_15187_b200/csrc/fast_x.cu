// fast_x.cu -- instantiations and launchers of the fast x-direction kernels (xfast.cuh).
#include "fast_launch.hpp"
#include "fast_configs.hpp"

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

template <class C, bool NEU> static cudaError_t init_one()
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    const int bf = (int)XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, b1 = (int)XSmemLayout<C, LPB, NEU, LPB>::BYTES;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_xf_fast<C, LPB, NEU, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bf))) return e;
    if ((e = cudaFuncSetAttribute(k_xf_fast<C, LPB, NEU, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1))) return e;
    return cudaFuncSetAttribute(k_xi_fast<C, LPB, NEU>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1);
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

template <class C, bool NEU> static cudaError_t xf_one(const XFast& P, const SParams& S, bool fused, const double* u, const double* v,
                                                       const double* w, double inv_adt, cplx* spec, cudaStream_t st)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    if (fused) k_xf_fast<C, LPB, NEU, true><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, st>>>(P, S, u, v, w, inv_adt, spec);
    else k_xf_fast<C, LPB, NEU, false><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, st>>>(P, S, u, v, w, inv_adt, spec);
    return cudaGetLastError();
}

cudaError_t launch_xf_fast(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v,
                           const double* w, double inv_adt, cplx* spec, cudaStream_t st)
{
    switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xf_one<FftCfg<n, a, b, c>, true>(P, S, fused, u, v, w, inv_adt, spec, st) \
                           : xf_one<FftCfg<n, a, b, c>, false>(P, S, fused, u, v, w, inv_adt, spec, st);
        FSEI_X_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

template <class C, bool NEU> static cudaError_t xi_one(const XFast& P, const cplx* spec, double* phi, cudaStream_t st)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    k_xi_fast<C, LPB, NEU><<<grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, st>>>(P, spec, phi);
    return cudaGetLastError();
}

cudaError_t launch_xi_fast(const XFast& P, bool neu, const cplx* spec, double* phi, cudaStream_t st)
{
    switch (P.N) {
#define X(n, a, b, c) \
        case n: return neu ? xi_one<FftCfg<n, a, b, c>, true>(P, spec, phi, st) : xi_one<FftCfg<n, a, b, c>, false>(P, spec, phi, st);
        FSEI_X_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace fsei
