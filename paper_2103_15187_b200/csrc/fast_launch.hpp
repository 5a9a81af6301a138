// fast_launch.hpp -- host-side entry points of the fast-path transform kernels (fast_x.cu, fast_y.cu):
// which line lengths have a register-resident Stockham instantiation, and the launchers.
#pragma once
#include <cuda_runtime.h>
#include "xfast.cuh"
#include "yfast.cuh"

namespace fsei {

bool xfast_supported(int N);     // N = nx / 2
bool yfast_supported(int N);     // N = ny
// raise the dynamic shared-memory limit of every instantiation (once per process)
cudaError_t xfast_init();
cudaError_t yfast_init();

// a1+a2 (fused: rhs = D(u,v,w) * inv_adt) or a2 alone (u = rhs, v = w = nullptr)
cudaError_t launch_xf_fast(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v,
                           const double* w, double inv_adt, cplx* spec, cudaStream_t st);
cudaError_t launch_xi_fast(const XFast& P, bool neu, const cplx* spec, double* phi, cudaStream_t st);
// a3 / a5, in place
cudaError_t launch_y_fast(const YFast& P, bool inv, bool neu, cplx* spec, cudaStream_t st);

}  // namespace fsei
