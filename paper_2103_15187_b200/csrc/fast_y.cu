// fast_y.cu -- instantiations and launchers of the fast y-direction kernel (yfast.cuh).
#include "fast_launch.hpp"
#include "fast_configs.hpp"

namespace fsei {

bool yfast_supported(int N)
{
    switch (N) {
#define X(n, a, b, c, cy) case n:
        FSEI_Y_CONFIGS(X)
#undef X
        return true;
        default: return false;
    }
}

template <class C, int CY> static cudaError_t init_one()
{
    cudaError_t e;
    const int b0 = (int)YSmemLayout<C, CY, false>::BYTES, b1 = (int)YSmemLayout<C, CY, true>::BYTES;
    if ((e = cudaFuncSetAttribute(k_y_fast<C, CY, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, b0))) return e;
    if ((e = cudaFuncSetAttribute(k_y_fast<C, CY, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, b0))) return e;
    if ((e = cudaFuncSetAttribute(k_y_fast<C, CY, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1))) return e;
    return cudaFuncSetAttribute(k_y_fast<C, CY, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, b1);
}

cudaError_t yfast_init()
{
    cudaError_t e;
#define X(n, a, b, c, cy) if ((e = init_one<FftCfg<n, a, b, c>, cy>())) return e;
    FSEI_Y_CONFIGS(X)
#undef X
    return cudaSuccess;
}

template <class C, int CY> static cudaError_t y_one(const YFast& P, bool inv, bool neu, cplx* spec, cudaStream_t st)
{
    const int gx = (P.nxc + CY - 1) / CY;
    int gy = 148 * 16 / gx; if (gy < 1) gy = 1; if (gy > P.nz) gy = P.nz;
    dim3 grid(gx, gy);
    const int nt = C::T * CY;
    const size_t b0 = YSmemLayout<C, CY, false>::BYTES, b1 = YSmemLayout<C, CY, true>::BYTES;
    if (!inv && !neu) k_y_fast<C, CY, false, false><<<grid, nt, b0, st>>>(P, spec);
    else if (inv && !neu) k_y_fast<C, CY, true, false><<<grid, nt, b0, st>>>(P, spec);
    else if (!inv && neu) k_y_fast<C, CY, false, true><<<grid, nt, b1, st>>>(P, spec);
    else k_y_fast<C, CY, true, true><<<grid, nt, b1, st>>>(P, spec);
    return cudaGetLastError();
}

cudaError_t launch_y_fast(const YFast& P, bool inv, bool neu, cplx* spec, cudaStream_t st)
{
    switch (P.ny) {
#define X(n, a, b, c, cy) case n: return y_one<FftCfg<n, a, b, c>, cy>(P, inv, neu, spec, st);
        FSEI_Y_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace fsei
