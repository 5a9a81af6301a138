// kernel_env.cuh -- the few macros the fast-path kernels are written against, so that the same kernel
// source compiles (a) with nvcc for sm_100a into libfsei.so and (b) with g++ inside the host stepping
// harness of tests/emu, where a CTA is a team of host threads and the barrier is a host barrier.
// (b) is test infrastructure for the index arithmetic, not a fallback: libfsei.so holds device code only.
#pragma once

#if defined(__CUDACC__)
#define FSEI_GLOBAL(maxthreads, minblocks) __global__ void __launch_bounds__(maxthreads, minblocks)
#define FSEI_DEV __device__ __forceinline__
#define FSEI_SYNC() __syncthreads()
#define FSEI_DYN_SMEM(name) extern __shared__ __align__(16) unsigned char name[]
#else
#include "cuda_shim.hpp"            // tests/emu/cuda_shim.hpp (on the include path of the harness only)
#define FSEI_GLOBAL(maxthreads, minblocks) inline void
#define FSEI_DEV inline
#define FSEI_SYNC() ::cuda_shim::sync_block()
#define FSEI_DYN_SMEM(name) unsigned char* name = ::cuda_shim::dyn_smem()
#endif
