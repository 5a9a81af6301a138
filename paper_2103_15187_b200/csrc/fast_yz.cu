// fast_yz.cu -- instantiations and launchers of the z-marching y kernels of the fused path (yzfused.cuh).
#include "fast_launch.hpp"
#include "fast_configs.hpp"

namespace fsei {

bool yzfused_supported(int N)
{
    switch (N) {
#define X(n, a, b, c) case n:
        FSEI_YZ_CONFIGS(X)
#undef X
        return true;
        default: return false;
    }
}

int yzfused_block_threads(int N)
{
    switch (N) {
#define X(n, a, b, c) case n: return FftCfg<n, a, b, c>::T * FSEI_CB;
        FSEI_YZ_CONFIGS(X)
#undef X
        default: return 0;
    }
}

// boundary-condition variants: (periodic y, 1 pivot component) = (P,P); (periodic y, 2) = (N,P); (Neumann y, 2)
template <class C, bool NEU, int NCOMP> static cudaError_t init_variant()
{
    using L = YZSmem<C, FSEI_CB, NEU, NCOMP>;
    cudaError_t e;
    if ((e = kernel_smem(k_yz_forward<C, FSEI_CB, NEU, NCOMP>, (int)L::FWD))) return e;
    return kernel_smem(k_yz_backward<C, FSEI_CB, NEU, NCOMP>, (int)L::BWD);
}

cudaError_t yzfused_init()
{
    cudaError_t e;
#define X(n, a, b, c) \
    if ((e = init_variant<FftCfg<n, a, b, c>, false, 1>())) return e; \
    if ((e = init_variant<FftCfg<n, a, b, c>, false, 2>())) return e; \
    if ((e = init_variant<FftCfg<n, a, b, c>, true, 2>())) return e;
    FSEI_YZ_CONFIGS(X)
#undef X
    return cudaSuccess;
}

template <class C, bool NEU, int NCOMP> static cudaError_t run_variant(const YZFused& P, bool backward, cplx* spec, cudaStream_t st)
{
    using L = YZSmem<C, FSEI_CB, NEU, NCOMP>;
    const dim3 grid(P.nxc / FSEI_CB, P.ktw < P.nz ? 2 : 1);
    const int nt = C::T * FSEI_CB;
    if (!backward) k_yz_forward<C, FSEI_CB, NEU, NCOMP><<<grid, nt, L::FWD, st>>>(P, spec);
    else k_yz_backward<C, FSEI_CB, NEU, NCOMP><<<grid, nt, L::BWD, st>>>(P, spec);
    return cudaGetLastError();
}

template <class C> static cudaError_t run_cfg(const YZFused& P, bool backward, bool neu, int ncomp, cplx* spec, cudaStream_t st)
{
    if (neu) return ncomp == 2 ? run_variant<C, true, 2>(P, backward, spec, st) : cudaErrorInvalidValue;
    return ncomp == 1 ? run_variant<C, false, 1>(P, backward, spec, st) : run_variant<C, false, 2>(P, backward, spec, st);
}

static cudaError_t run(const YZFused& P, bool backward, bool neu, int ncomp, cplx* spec, cudaStream_t st)
{
    if (P.nxc % FSEI_CB) return cudaErrorInvalidValue;
    switch (P.ny) {
#define X(n, a, b, c) case n: return run_cfg<FftCfg<n, a, b, c>>(P, backward, neu, ncomp, spec, st);
        FSEI_YZ_CONFIGS(X)
#undef X
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_yz_forward(const YZFused& P, bool neu, int ncomp, cplx* spec, cudaStream_t st) { return run(P, false, neu, ncomp, spec, st); }
cudaError_t launch_yz_backward(const YZFused& P, bool neu, int ncomp, cplx* spec, cudaStream_t st) { return run(P, true, neu, ncomp, spec, st); }

}  // namespace fsei
