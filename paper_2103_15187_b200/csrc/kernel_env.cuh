// kernel_env.cuh -- the few macros and primitives the fast-path kernels are written against, so that the
// same kernel source compiles (a) with nvcc for sm_100a into libfsei.so and (b) with g++ inside the host
// harness of tests/emu, where a CTA is a team of host threads and the barrier is a host barrier.
// (b) is test infrastructure for the index arithmetic, not a fallback: libfsei.so holds device code only.
//
// Asynchronous tile loads (sm_100a): the TMA engine copies global memory into a shared-memory "landing"
// tile while the CTA computes on the previous tile; completion is tracked by an mbarrier transaction
// count.  bulk_g2s = cp.async.bulk (1-D, contiguous bytes), tma_load_2d = cp.async.bulk.tensor.2d through a
// CUtensorMap (row-strided boxes).  In the host harness both are plain copies done by the issuing thread
// and the wait is the block barrier.
#pragma once
#include <cstddef>
#include <cstdint>

#if defined(__CUDACC__)
#include <cuda.h>
#define FSEI_GLOBAL(maxthreads, minblocks) __global__ void __launch_bounds__(maxthreads, minblocks)
#define FSEI_DEV __device__ __forceinline__
#define FSEI_SYNC() __syncthreads()
// barrier among the `n` threads (a multiple of 32) that use named barrier `id` (1..15): the warps of one line only
#define FSEI_GROUP_SYNC(id, n) asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory")
#define FSEI_DYN_SMEM(name) extern __shared__ __align__(128) unsigned char name[]
#define FSEI_GRID_CONSTANT __grid_constant__

namespace fsei {

struct alignas(64) TmaMap2D { CUtensorMap m; };
struct alignas(64) TmaMap3D { CUtensorMap m; };

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// one thread; follow with FSEI_SYNC() before first use
__device__ __forceinline__ void abar_init(uint64_t* bar)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(1) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// one thread: this phase completes when `bytes` have landed
__device__ __forceinline__ void abar_expect(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// box (x0 .. , y0 ..) of the 2-D tensor, x = fastest coordinate (in elements of the map's data type)
__device__ __forceinline__ void tma_load_2d(void* dst, const TmaMap2D* map, int x0, int y0, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(x0), "r"(y0), "r"(smem_u32(bar)) : "memory");
}
// box (x0 .., y0 .., z0 ..) of a 3-D tensor, x = fastest coordinate
__device__ __forceinline__ void tma_load_3d(void* dst, const TmaMap3D* map, int x0, int y0, int z0, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(x0), "r"(y0), "r"(z0), "r"(smem_u32(bar)) : "memory");
}
// L2 prefetch of contiguous bytes / of a box: deepens the load pipeline at the DRAM level without shared memory
// (the later bulk load of the same bytes then completes at L2 latency)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_prefetch_3d(const TmaMap3D* map, int x0, int y0, int z0)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global [%0, {%1, %2, %3}];" ::"l"(map), "r"(x0), "r"(y0), "r"(z0) : "memory");
}
// read-only 8-byte load that does not allocate in L1
__device__ __forceinline__ double ld_stream(const double* p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
// value of `v` held by the lane `d` below / above (own value returned when that lane is outside the warp;
// callers mask by lane index).  All 32 lanes of the warp must call.
__device__ __forceinline__ double lane_up(double v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ double lane_down(double v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }
// every thread that reads the landing tile
__device__ __forceinline__ void abar_wait(uint64_t* bar, unsigned parity)
{
    unsigned ok = 0;
    const unsigned a = smem_u32(bar);
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}

}  // namespace fsei

#else
#include <cstring>
#include "cuda_shim.hpp"            // tests/emu/cuda_shim.hpp (on the include path of the harness only)
#define FSEI_GLOBAL(maxthreads, minblocks) inline void
#define FSEI_DEV inline
#define FSEI_SYNC() ::cuda_shim::sync_block()
#define FSEI_GROUP_SYNC(id, n) ::cuda_shim::sync_block()      // conservative stand-in (control flow is block-uniform)
#define FSEI_DYN_SMEM(name) unsigned char* name = ::cuda_shim::dyn_smem()
#define FSEI_GRID_CONSTANT

namespace fsei {

// host stand-in of a tiled tensor map: boxes of box_rows rows x box_bytes bytes out of a row-strided array
struct TmaMap2D { const unsigned char* base; size_t pitch_bytes; unsigned elem_bytes, box_elems, box_rows; };

// 3-D: dims (nx elements, ny, nz) with byte pitches of y and z; boxes of (bx, by, bz); out-of-range elements read 0
struct TmaMap3D { const unsigned char* base; size_t pitch_y, pitch_z; unsigned elem_bytes, nx, ny, nz, bx, by, bz; };

inline void abar_init(uint64_t*) {}
inline void abar_expect(uint64_t*, unsigned) {}
inline void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t*) { std::memcpy(dst, src, bytes); }
inline void tma_load_2d(void* dst, const TmaMap2D* m, int x0, int y0, uint64_t*)
{
    const size_t bb = (size_t)m->box_elems * m->elem_bytes;
    for (unsigned r = 0; r < m->box_rows; r++)
        std::memcpy(static_cast<unsigned char*>(dst) + r * bb, m->base + (size_t)(y0 + (int)r) * m->pitch_bytes + (size_t)x0 * m->elem_bytes, bb);
}
inline void tma_load_3d(void* dst, const TmaMap3D* m, int x0, int y0, int z0, uint64_t*)
{
    unsigned char* d = static_cast<unsigned char*>(dst);
    for (unsigned z = 0; z < m->bz; z++)
        for (unsigned y = 0; y < m->by; y++)
            for (unsigned x = 0; x < m->bx; x++, d += m->elem_bytes) {
                const unsigned X = x0 + x, Y = y0 + y, Z = z0 + z;
                if (X < m->nx && Y < m->ny && Z < m->nz)
                    std::memcpy(d, m->base + (size_t)Z * m->pitch_z + (size_t)Y * m->pitch_y + (size_t)X * m->elem_bytes, m->elem_bytes);
                else std::memset(d, 0, m->elem_bytes);
            }
}
inline double lane_up(double v, int d) { return ::cuda_shim::shfl(v, -d); }      // every thread of the block must call
inline double lane_down(double v, int d) { return ::cuda_shim::shfl(v, d); }
inline void bulk_prefetch_l2(const void*, unsigned) {}
inline void tma_prefetch_3d(const TmaMap3D*, int, int, int) {}
inline double ld_stream(const double* p) { return *p; }
inline void abar_wait(uint64_t*, unsigned) { ::cuda_shim::sync_block(); }      // the issuing thread copied before it got here

}  // namespace fsei
#endif
