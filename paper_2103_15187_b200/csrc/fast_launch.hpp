// fast_launch.hpp -- host-side entry points of the fast-path transform kernels (fast_x.cu, fast_y.cu):
// which line lengths have a register-resident Stockham instantiation, and the launchers.
#pragma once
#include <cuda_runtime.h>
#include "xfast.cuh"
#include "yfast.cuh"
#include "yzfused.cuh"

namespace fsei {

// raise a kernel's dynamic shared-memory limit and ask for the largest shared-memory carve-out, so that as many
// CTAs as fit in 227 KB are resident (the default carve-out heuristic stops at one CTA for these kernels)
template <class K> inline cudaError_t kernel_smem(K kernel, int bytes)
{
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}

bool xfast_supported(int N);     // N = nx / 2
bool yfast_supported(int N);     // N = ny
int xfast_lines_per_block(int N, bool neu);   // LPB of the x kernels for this line length
// raise the dynamic shared-memory limit of every instantiation (once per process)
cudaError_t xfast_init();
cudaError_t yfast_init();

// fused path (blocked spectrum layout, FSEI_CB slots per tile)
bool xblocked_supported(int N);  // N = nx / 2
bool yzfused_supported(int N);   // N = ny
int yzfused_block_threads(int N);  // threads per CTA of the z-marching y kernels
cudaError_t xblocked_init();
cudaError_t yzfused_init();
// tensor map of the blocked spectrum for the x-inverse loads (plan time; spec = the plan's workspace)
cudaError_t make_xi_blocked_map(const XFast& P, bool neu, const cplx* spec, TmaMap3D* out);
cudaError_t launch_yz_forward(const YZFused& P, bool neu, int ncomp, cplx* spec, cudaStream_t st);
cudaError_t launch_yz_backward(const YZFused& P, bool neu, int ncomp, cplx* spec, cudaStream_t st);

// a1+a2 (fused: rhs = D(u,v,w) * inv_adt) or a2 alone (u = rhs, v = w = nullptr)
// blocked: spec is in the blocked layout (xi: read through `map`)
cudaError_t launch_xf_fast(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v,
                           const double* w, double inv_adt, cplx* spec, cudaStream_t st, bool blocked = false);
cudaError_t launch_xi_fast(const XFast& P, bool neu, const cplx* spec, double* phi, cudaStream_t st,
                           const TmaMap3D* map = nullptr);
// fast family of the implicit viscous step (visc_fast.cuh): periodic x and y, nx/32 and ny/32 instantiated
struct VFastLine; struct VFastArgs;
bool visc_fast_supported(int nx, int ny);
bool visc_fast_slab_supported(int nx, int ny);
cudaError_t visc_fast_init();
void visc_fast_line(int n, double h_recip, double beta, VFastLine* out);
int visc_fast_nsig(const VFastLine& L);
cudaError_t launch_visc_xz(const VFastArgs& A, cudaStream_t st);
cudaError_t launch_visc_zy(const VFastArgs& A, cudaStream_t st);

// a3 / a5, in place
cudaError_t launch_y_fast(const YFast& P, bool inv, bool neu, cplx* spec, cudaStream_t st);

}  // namespace fsei
