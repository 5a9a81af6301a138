// cuda_shim.hpp -- just enough of the CUDA execution model to run the fast-path kernels of libfsei on the
// host for tests: a CTA is a team of host threads, __syncthreads() a std::barrier, dynamic shared memory a
// heap block, blocks run one after the other.  Test infrastructure only (tests/emu); never shipped.
#pragma once
#include <barrier>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

struct uint3_shim { unsigned x = 0, y = 0, z = 0; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};

namespace cuda_shim {
inline thread_local uint3_shim t_threadIdx, t_blockIdx;
inline dim3 g_blockDim, g_gridDim;
inline std::barrier<>* g_bar = nullptr;
inline unsigned char* g_smem = nullptr;

inline void sync_block() { g_bar->arrive_and_wait(); }
inline double g_shfl[1024];
// warp shuffle by lane offset for a block in uniform control flow: every thread of the block calls (two barriers)
inline double shfl(double v, int delta)
{
    const unsigned tid = t_threadIdx.x;                   // 1-D blocks only
    g_shfl[tid] = v;
    g_bar->arrive_and_wait();
    const int lane = (int)(tid & 31u), src = lane + delta;
    const double r = (src >= 0 && src < 32 && (tid - lane + src) < g_blockDim.x) ? g_shfl[tid - lane + src] : v;
    g_bar->arrive_and_wait();
    return r;
}
inline unsigned char* dyn_smem() { return g_smem; }

// run body() as every thread of every block of the grid (blocks sequential, threads concurrent)
template <class F> void launch(dim3 grid, dim3 block, size_t smem_bytes, F body)
{
    const unsigned nt = block.x * block.y * block.z;
    std::barrier<> bar((std::ptrdiff_t)nt);
    unsigned char* smem = static_cast<unsigned char*>(std::aligned_alloc(128, ((smem_bytes + 127) / 128 + 1) * 128));
    g_bar = &bar; g_smem = smem; g_blockDim = block; g_gridDim = grid;
    auto worker = [&](unsigned tid) {
        t_threadIdx.x = tid % block.x; t_threadIdx.y = (tid / block.x) % block.y; t_threadIdx.z = tid / (block.x * block.y);
        for (unsigned bz = 0; bz < grid.z; bz++)
            for (unsigned by = 0; by < grid.y; by++)
                for (unsigned bx = 0; bx < grid.x; bx++) {
                    t_blockIdx.x = bx; t_blockIdx.y = by; t_blockIdx.z = bz;
                    body();
                    bar.arrive_and_wait();          // block boundary: shared memory is reused by the next block
                }
    };
    std::vector<std::thread> th;
    th.reserve(nt);
    for (unsigned t = 0; t < nt; t++) th.emplace_back(worker, t);
    for (auto& t : th) t.join();
    std::free(smem);
    g_bar = nullptr; g_smem = nullptr;
}
}  // namespace cuda_shim

#define threadIdx (::cuda_shim::t_threadIdx)
#define blockIdx (::cuda_shim::t_blockIdx)
#define blockDim (::cuda_shim::g_blockDim)
#define gridDim (::cuda_shim::g_gridDim)
