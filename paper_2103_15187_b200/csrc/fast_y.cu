// fast_y.cu -- instantiations and launchers of the fast y-direction kernel (yfast.cuh).
#include "fast_launch.hpp"
#include "fast_configs.hpp"
#include "tma_host.hpp"

namespace fsei {

// 2-D fp64 view of the spectrum: inner dimension 2 nxc doubles (one row of one plane), outer ny nz rows;
// box = 2 CY doubles x box_rows rows
static cudaError_t make_map(const YFast& P, int CY, int box_rows, cplx* spec, TmaMap2D* out)
{
    EncodeTiledFn fn = tma_encode_fn();
    if (!fn) return cudaErrorNotSupported;
    cuuint64_t dims[2] = {(cuuint64_t)2 * P.nxc, (cuuint64_t)P.ny * P.nz};
    cuuint64_t strides[1] = {(cuuint64_t)P.nxc * sizeof(cplx)};
    cuuint32_t box[2] = {(cuuint32_t)(2 * CY), (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(&out->m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, spec, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

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
    if ((e = kernel_smem(k_y_fast<C, CY, false, false>, b0))) return e;
    if ((e = kernel_smem(k_y_fast<C, CY, true, false>, b0))) return e;
    if ((e = kernel_smem(k_y_fast<C, CY, false, true>, b1))) return e;
    return kernel_smem(k_y_fast<C, CY, true, true>, b1);
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
    TmaMap2D map;
    cudaError_t e = make_map(P, CY, y_box_rows(C::N), spec, &map);
    if (e != cudaSuccess) return e;
    if (!inv && !neu) k_y_fast<C, CY, false, false><<<grid, nt, b0, st>>>(P, map, spec);
    else if (inv && !neu) k_y_fast<C, CY, true, false><<<grid, nt, b0, st>>>(P, map, spec);
    else if (!inv && neu) k_y_fast<C, CY, false, true><<<grid, nt, b1, st>>>(P, map, spec);
    else k_y_fast<C, CY, true, true><<<grid, nt, b1, st>>>(P, map, spec);
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
