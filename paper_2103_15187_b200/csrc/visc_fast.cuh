// visc_fast.cuh -- fast family of the implicit viscous step (Eq. 3) for the paper's own
// case: periodic, uniform x and y ("Thomas' algorithm with a Sherman-Morrison perturbation in the two periodic
// dimensions"), stretched wall-normal z.
//
//   q += [(1 - beta dxx)(1 - beta dyy)(1 - beta dzz)]^-1 rhs      (the three factors commute: each acts on its own index)
//
// TWO launches move each component 40 B/cell (the generic family: six passes, 104 B/cell):
//   pass A  k_visc_xz : one WARP owns one x-line and marches k = 0 .. nz-1.  Per plane the line arrives by 32 bulk
//           copies (cp.async.bulk, one 8M-byte chunk per lane into a padded slot: conflict-free 128-bit reads), is solved
//           in REGISTERS (lane = chunk of M = nx/32 unknowns) and goes straight through the forward elimination of the
//           z system, whose previous row d'(k-1) is carried in registers; d' leaves by bulk stores.  rhs -> d' in place.
//   pass B  k_visc_zy : one CTA owns 8 adjacent columns x all ny rows and marches k = nz-1 .. 0: back substitution of
//           the z system with x(k+1) carried in registers, then the periodic y-solve of the tile (thread = one column x
//           one chunk of M = ny/32 rows, lanes along x: 64-byte row segments), then q += result.
//
// A periodic line of n = 32 M unknowns is solved by a PARTITION method instead of a serial sweep: each of the 32 chunks
// eliminates its M-1 interior unknowns against its two separators with a local Thomas solve (the matrix has constant
// coefficients, so factorisation and spikes are the same for every chunk: warp-uniform constants in the kernel
// parameter bank), the 32 separators obey a circulant tridiagonal system whose inverse is ONE row of 32 numbers (built on
// the host per beta, in long double), applied by 32 shuffles (x) or 32 shared-memory reads (y), and the interiors are
// corrected with the two spikes.  Exact up to rounding (no truncation of the decay), ~7 FMA per unknown.
#pragma once
#include "kernel_env.cuh"
#include "plan_types.cuh"

namespace fsei {

// uniform periodic line: a = c = -r, b = 1 + 2r (r = beta / h^2); M = n / 32 unknowns per chunk, the last one the separator
struct VFastLine {
    double r;
    double ip[31], cp[31];      // interior Thomas factorisation: reciprocal pivots, c'_i      (entries < M-1)
    double ls[31], rs[31];      // spikes: interior response to a unit left / right separator  (entries < M-1)
    double sinv[32];            // first row of the inverse of the 32 x 32 circulant separator system
};

struct VFastArgs {
    VFastLine L;                // x line (pass A) or y line (pass B)
    const double* zam[3];       // z tables of u, v, w (device): sub-diagonal, reciprocal pivot, c'
    const double* zip[3];
    const double* zcp[3];
    double* r[3];               // right-hand sides: rhs -> d' (pass A, in place); d' read by pass B
    double* q[3];               // velocity components (pass B)
    int nx, ny, nz;
    int nsig;                   // terms of sinv kept on either side of s = 0 (16 = all)
    int slab;                   // 1 = a z-slab (fsei_slab_viscous_xy): pass A solves x only, pass B solves y only and stores in place of d'
    int split;                  // pass B: 1 = one CTA per (tile, component) instead of one per tile (host: grids with few tiles)
};

#if defined(__CUDACC__)
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// interior solve of one chunk, in place: x[0 .. M-2] -> y = T^-1 x   (T: constant-coefficient tridiagonal of size M-1)
template <int M> __device__ __forceinline__ void chunk_interior(const VFastLine& L, double (&x)[M])
{
    x[0] *= L.ip[0];
#pragma unroll
    for (int i = 1; i < M - 1; i++) x[i] = fma(L.r, x[i - 1], x[i]) * L.ip[i];
#pragma unroll
    for (int i = M - 3; i >= 0; i--) x[i] = fma(-L.cp[i], x[i + 1], x[i]);
}
// interiors corrected with the separators to their left (xl) and right (xs); the separator itself stored last
template <int M> __device__ __forceinline__ void chunk_correct(const VFastLine& L, double (&x)[M], double xl, double xs)
{
#pragma unroll
    for (int i = 0; i < M - 1; i++) x[i] = fma(L.rs[i], xs, fma(L.ls[i], xl, x[i]));
    x[M - 1] = xs;
}

// ---------------------------------------------------------------------------------------------------------------
// pass A: grid (ny / WPB, 3), block 32 * WPB.  Dynamic shared memory: WPB * (S * 32 * (8 M + 16) + 8 S) bytes.
// ---------------------------------------------------------------------------------------------------------------
#define FSEI_VA_STAGES 3
#define FSEI_VA_WPB 2

template <int M>
FSEI_GLOBAL(32 * FSEI_VA_WPB, 1) k_visc_xz(const FSEI_GRID_CONSTANT VFastArgs A)
{
    constexpr int S = FSEI_VA_STAGES, PITCH = 8 * M + 16, STAGE = 32 * PITCH;
    FSEI_DYN_SMEM(smraw);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, comp = blockIdx.y;
    const int j = blockIdx.x * FSEI_VA_WPB + wid;
    if (j >= A.ny) return;
    unsigned char* buf = smraw + (size_t)wid * (S * STAGE + 64);
    uint64_t* bar = reinterpret_cast<uint64_t*>(buf + S * STAGE);
    const size_t plane = (size_t)A.nx * A.ny;
    double* f = A.r[comp] + (size_t)j * A.nx + (size_t)lane * M;          // this lane's chunk of line j at plane 0
    const double* __restrict__ zam = A.zam[comp];
    const double* __restrict__ zip = A.zip[comp];
    const VFastLine& L = A.L;
    const int nz = A.nz, nsig = A.nsig;
    if (lane == 0) for (int s = 0; s < S; s++) abar_init(bar + s);
    __syncwarp();
    for (int s = 0; s < S - 1 && s < nz; s++) {                  // prologue: planes 0 .. S-2 in flight
        if (lane == 0) abar_expect(bar + s, 32 * 8 * M);
        __syncwarp();
        bulk_g2s(buf + s * STAGE + lane * PITCH, f + (size_t)s * plane, 8 * M, bar + s);
    }
    double dprev[M];
#pragma unroll
    for (int i = 0; i < M; i++) dprev[i] = 0.0;
    const bool wfix = comp == COMP_W;                                       // w: plane 0 is the wall (row fixed)
    int st = 0; unsigned par = 0;
    double* fk = f;                                                         // plane k
    double* fn = f + (size_t)(S - 1) * plane;                               // plane k + S - 1
    for (int k = 0; k < nz; k++, fk += plane, fn += plane) {
        abar_wait(bar + st, par);
        double x[M];
        const double2* src = reinterpret_cast<const double2*>(buf + st * STAGE + lane * PITCH);
#pragma unroll
        for (int i = 0; i < M / 2; i++) { const double2 t = src[i]; x[2 * i] = t.x; x[2 * i + 1] = t.y; }
        // ---- periodic x-solve of the line
        const double sep = x[M - 1];
        chunk_interior<M>(L, x);
        const double y0n = __shfl_sync(0xffffffffu, x[0], (lane + 1) & 31);
        const double g = fma(L.r, x[M - 2] + y0n, sep);
        // separators: xs_p = sum_s sinv[s] g_{p-s}; sinv[s] = sinv[32-s] decays away from s = 0 and only the nsig terms on
        // either side that can reach the last bit of the sum are kept (nsig = 16: all of them)
        double xs = L.sinv[0] * g;
        for (int s = 1; s <= nsig; s++) {
            const double gm = __shfl_sync(0xffffffffu, g, (lane - s) & 31), gp = __shfl_sync(0xffffffffu, g, (lane + s) & 31);
            xs = fma(L.sinv[s], s == 16 ? gm : gm + gp, xs);
        }
        const double xl = __shfl_sync(0xffffffffu, xs, (lane - 1) & 31);
        chunk_correct<M>(L, x, xl, xs);
        // ---- forward elimination of the z system: d'_k = (x_k - a_k d'_{k-1}) / piv_k
        const double am = zam[k], ipk = zip[k];
        const bool zero = wfix && k == 0;
#pragma unroll
        for (int i = 0; i < M; i++) dprev[i] = zero ? 0.0 : fma(-am, dprev[i], x[i]) * ipk;
        // ---- out: through the same slot
        double2* dst = reinterpret_cast<double2*>(buf + st * STAGE + lane * PITCH);
#pragma unroll
        for (int i = 0; i < M / 2; i++) dst[i] = make_double2(dprev[2 * i], dprev[2 * i + 1]);
        fence_async_smem();
        bulk_s2g(fk, dst, 8 * M);
        bulk_commit();
        // ---- next load into the slot of plane k-1 once its store has been read out
        const int sn = st == 0 ? S - 1 : st - 1;
        if (k + S - 1 < nz) {
            bulk_wait_read<1>();
            if (lane == 0) abar_expect(bar + sn, 32 * 8 * M);
            __syncwarp();
            bulk_g2s(buf + sn * STAGE + lane * PITCH, fn, 8 * M, bar + sn);
        }
        if (++st == S) { st = 0; par ^= 1u; }
    }
    bulk_wait_all<0>();
}

// ---------------------------------------------------------------------------------------------------------------
// pass A through tensor maps (chunk lengths 8, 16, 24, 32, i.e. nx = 256, 512, 768, 1024): a line is the 2-D array [32 chunks][M doubles];
// boxes of (16 doubles = 128 bytes) x 32 chunks land with the 128-byte swizzle, which puts the 16-byte piece i of chunk l at
// piece i ^ (l & 7) of its row, so that the 32 lanes -- each reading ITS chunk with 128-bit loads -- fall on all banks.  Two
// TMA instructions per line and direction instead of 32 bulk copies issued lane by lane (a warp-serial loop that took half
// of k_visc_xz's stall samples).  Same arithmetic as k_visc_xz.  Dynamic shared memory: 1024 + WPB * (S * 256 M + 64) bytes.
// ---------------------------------------------------------------------------------------------------------------
#ifndef FSEI_VA_TMA_WPB
#define FSEI_VA_TMA_WPB 1            // warps per CTA of the tensor-map variant
#endif
struct VFastMapsA { TmaMap2D r[3]; };      // per component: fp64 [32 ny nz rows][M], box 16 x 32, CU_TENSOR_MAP_SWIZZLE_128B

__device__ __forceinline__ void tma_store_2d(const TmaMap2D* map, int x0, int y0, const void* src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(x0), "r"(y0), "r"(smem_u32(src)) : "memory");
}

template <int M>
FSEI_GLOBAL(32 * FSEI_VA_TMA_WPB, 1) k_visc_xz_tma(const FSEI_GRID_CONSTANT VFastArgs A, const FSEI_GRID_CONSTANT VFastMapsA Mp)
{
    static_assert(M % 8 == 0, "whole 64- or 128-byte boxes");
    // box width: 16 doubles with the 128-byte swizzle where M allows it, else 8 doubles with the 64-byte swizzle (there the 16-byte
    // piece i of chunk l sits at piece i ^ ((l >> 1) & 3))
    constexpr int S = FSEI_VA_STAGES, BW = (M % 16 == 0) ? 16 : 8, CH = BW / 2, ROWB = 8 * BW, BOXB = 32 * ROWB, NBOX = M / BW, STAGE = NBOX * BOXB;
    FSEI_DYN_SMEM(smraw);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, comp = blockIdx.y;
    const int j = blockIdx.x * FSEI_VA_TMA_WPB + wid;
    if (j >= A.ny) return;
    unsigned char* base = smraw + ((1024u - (smem_u32(smraw) & 1023u)) & 1023u);       // the swizzle pattern repeats every 1024 bytes
    unsigned char* buf = base + (size_t)wid * (S * STAGE);
    uint64_t* bar = reinterpret_cast<uint64_t*>(base + (size_t)FSEI_VA_TMA_WPB * S * STAGE) + wid * 8;
    const double* __restrict__ zam = A.zam[comp];
    const double* __restrict__ zip = A.zip[comp];
    const VFastLine& L = A.L;
    const int nz = A.nz, nsig = A.nsig, ny = A.ny;
    const TmaMap2D* map = &Mp.r[comp];
    auto load_line = [&](int s, int k) {             // plane k of line j -> stage s (lane 0)
        abar_expect(bar + s, 32 * 8 * M);
#pragma unroll
        for (int h = 0; h < NBOX; h++) tma_load_2d(buf + s * STAGE + h * BOXB, map, BW * h, (k * ny + j) * 32, bar + s);
    };
    if (lane == 0) for (int s = 0; s < S; s++) abar_init(bar + s);
    __syncwarp();
    if (lane == 0) for (int s = 0; s < S - 1 && s < nz; s++) load_line(s, s);          // prologue: planes 0 .. S-2 in flight
    double dprev[M];
#pragma unroll
    for (int i = 0; i < M; i++) dprev[i] = 0.0;
    const bool wfix = comp == COMP_W;                                       // w: plane 0 is the wall (row fixed)
    int st = 0; unsigned par = 0;
    const int sw = BW == 16 ? (lane & 7) : ((lane >> 1) & 3);
    for (int k = 0; k < nz; k++) {
        abar_wait(bar + st, par);
        double x[M];
        unsigned char* row = buf + st * STAGE + lane * ROWB;
#pragma unroll
        for (int h = 0; h < NBOX; h++)
#pragma unroll
            for (int i = 0; i < CH; i++) {
                const double2 t = *reinterpret_cast<const double2*>(row + h * BOXB + ((i ^ sw) << 4));
                x[BW * h + 2 * i] = t.x; x[BW * h + 2 * i + 1] = t.y;
            }
        // ---- periodic x-solve of the line
        const double sep = x[M - 1];
        chunk_interior<M>(L, x);
        const double y0n = __shfl_sync(0xffffffffu, x[0], (lane + 1) & 31);
        const double g = fma(L.r, x[M - 2] + y0n, sep);
        double xs = L.sinv[0] * g;
        for (int s = 1; s <= nsig; s++) {
            const double gm = __shfl_sync(0xffffffffu, g, (lane - s) & 31), gp = __shfl_sync(0xffffffffu, g, (lane + s) & 31);
            xs = fma(L.sinv[s], s == 16 ? gm : gm + gp, xs);
        }
        const double xl = __shfl_sync(0xffffffffu, xs, (lane - 1) & 31);
        chunk_correct<M>(L, x, xl, xs);
        if (A.slab) {                                // a z-slab: the z system is solved on pencils, after a transpose
#pragma unroll
            for (int i = 0; i < M; i++) dprev[i] = x[i];
        } else {
            // ---- forward elimination of the z system: d'_k = (x_k - a_k d'_{k-1}) / piv_k
            const double am = zam[k], ipk = zip[k];
            const bool zero = wfix && k == 0;
#pragma unroll
            for (int i = 0; i < M; i++) dprev[i] = zero ? 0.0 : fma(-am, dprev[i], x[i]) * ipk;
        }
        // ---- out: through the same slot
#pragma unroll
        for (int h = 0; h < NBOX; h++)
#pragma unroll
            for (int i = 0; i < CH; i++)
                *reinterpret_cast<double2*>(row + h * BOXB + ((i ^ sw) << 4)) = make_double2(dprev[BW * h + 2 * i], dprev[BW * h + 2 * i + 1]);
        fence_async_smem();
        __syncwarp();
        if (lane == 0) {
#pragma unroll
            for (int h = 0; h < NBOX; h++) tma_store_2d(map, BW * h, (k * ny + j) * 32, buf + st * STAGE + h * BOXB);
            bulk_commit();
            // ---- next load into the slot of plane k-1 once its store has been read out
            if (k + S - 1 < nz) { bulk_wait_read<1>(); load_line(st == 0 ? S - 1 : st - 1, k + S - 1); }
        }
        if (++st == S) { st = 0; par ^= 1u; }
    }
    if (lane == 0) bulk_wait_all<0>();
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------------------------
// pass B: grid nx / 8, block 256 (the CTA walks its tile through u, v, w): thread = (column i = tid & 7, chunk c = tid >> 3).
// The (ny x 8) tile of d' of plane k-1 lands by 2-D TMA boxes in one of two shared-memory tiles while plane k is being
// solved in the other; the result goes back into its tile and leaves as a TMA REDUCE-ADD onto q (the addition q + dq is
// done by the L2: the SM never loads q), so the LSU only sees shared memory.  x(k+1) of the z back substitution is
// carried in a third shared-memory tile [M][256].  Dynamic shared memory: 128 + 2 * ny * 64 + M * 256 * 8 bytes.
// ---------------------------------------------------------------------------------------------------------------
struct VFastMaps { TmaMap2D d[3], q[3]; int box_rows; };      // 2-D fp64 views [nz * ny rows][nx], box 8 x box_rows

__device__ __forceinline__ void tma_reduce_add_2d(const TmaMap2D* map, int x0, int y0, const void* src)
{
    asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(x0), "r"(y0), "r"(smem_u32(src)) : "memory");
}

template <int M>
FSEI_GLOBAL(256, 1) k_visc_zy(const FSEI_GRID_CONSTANT VFastArgs A, const FSEI_GRID_CONSTANT VFastMaps Mp)
{
    __shared__ double sm_y0[2][32][8], sm_g[2][32][8], sm_x[2][32][8];
    FSEI_DYN_SMEM(smraw);
    constexpr int NY = 32 * M;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    double* tile0 = reinterpret_cast<double*>(smraw + 128);     // [2][NY][8]
    double* carry = tile0 + 2 * NY * 8 + threadIdx.x;           // [M][256]
    const int tid = threadIdx.x, i = tid & 7, c = tid >> 3;
    // one CTA per tile of 8 columns walking u, v, w in turn -- all CTAs then sit on the same plane of the same field, which is what
    // keeps the 64-byte rows of neighbouring tiles in open DRAM pages -- or, where that leaves SMs idle (up to 1.5 marches per SM), one CTA
    // per (tile, component).  (Dealing the marches out in equal item ranges with carry hand-offs was tried: the CTAs drift apart
    // in k and large grids lose half their bandwidth.)
    const int col0 = (A.split ? blockIdx.x / 3 : blockIdx.x) * 8, comp0 = A.split ? blockIdx.x % 3 : 0;
    const int nb = NY / Mp.box_rows, nz = A.nz, nit = (A.split ? 1 : 3) * nz;
    const VFastLine& L = A.L;
    // items it = comp * nz + (nz - 1 - k): the tile walks down each component in turn; item it uses tile it & 1
    auto issue = [&](int it) {
        const int ci = it / nz, k = nz - 1 - (it - ci * nz), cc = comp0 + ci;
        double* t = tile0 + (it & 1) * NY * 8;
        abar_expect(bar + (it & 1), (unsigned)(NY * 64));
        for (int b = 0; b < nb; b++) tma_load_2d(t + b * Mp.box_rows * 8, &Mp.d[cc], col0, k * NY + b * Mp.box_rows, bar + (it & 1));
    };
    if (tid == 0) { abar_init(bar); abar_init(bar + 1); }
    __syncthreads();
    if (tid == 0) issue(0);
    for (int it = 0; it < nit; it++) {
        const int ci = it / nz, k = nz - 1 - (it - ci * nz), comp = comp0 + ci, pb = it & 1;
        double* tl = tile0 + pb * NY * 8 + (c * M) * 8 + i;
        if (tid == 0 && it + 1 < nit) { bulk_wait_read<0>(); issue(it + 1); }   // the other tile: its reduce-store has been read out
        abar_wait(bar + pb, (it >> 1) & 1);
        // The four chunks a warp touches start 64 M bytes apart: for even M all on the same half of the banks (two wavefronts
        // more than the two a warp's 32 doubles need).  Odd chunks therefore walk their rows in swapped pairs (row m+1 when the
        // even chunks are at row m), which puts them on the other half; the values end up in the same registers either way.
        constexpr bool SWZ = (M % 2 == 0) && M < 32;      // measured: M = 8 .. 24 gain 3-5 %, M = 32 (already DRAM-paced, 153 registers) loses 3 %
        const bool odd = SWZ && (c & 1);
        double* tA = tl + (odd ? 8 : 0);
        double* tB = tl + (odd ? 0 : 8);
        double x[M];
        if (SWZ) {
#pragma unroll
            for (int m = 0; m < M; m += 2) {
                const double a = tA[m * 8], b = tB[m * 8];
                x[m] = odd ? b : a; x[m + 1] = odd ? a : b;
            }
        } else {
#pragma unroll
            for (int m = 0; m < M; m++) x[m] = tl[m * 8];
        }
        // ---- back substitution of the z system: x_k = d'_k - c'_k x_{k+1}   (top plane: nothing above)
        const double cpk = A.slab ? 0.0 : A.zcp[comp][k];
        if (A.slab) {                                // a z-slab: no z coupling here
        } else if (k == nz - 1) {
#pragma unroll
            for (int m = 0; m < M; m++) carry[m * 256] = x[m];
        } else {
#pragma unroll
            for (int m = 0; m < M; m++) { x[m] = fma(-cpk, carry[m * 256], x[m]); carry[m * 256] = x[m]; }
        }
        // ---- periodic y-solve of the tile
        const double sep = x[M - 1];
        chunk_interior<M>(L, x);
        sm_y0[pb][c][i] = x[0];
        __syncthreads();
        const double g = fma(L.r, x[M - 2] + sm_y0[pb][(c + 1) & 31][i], sep);
        sm_g[pb][c][i] = g;
        __syncthreads();
        double xs = L.sinv[0] * g;
        for (int s = 1; s <= A.nsig; s++) {
            const double gm = sm_g[pb][(c - s) & 31][i], gp = sm_g[pb][(c + s) & 31][i];
            xs = fma(L.sinv[s], s == 16 ? gm : gm + gp, xs);
        }
        sm_x[pb][c][i] = xs;
        __syncthreads();
        const double xl = sm_x[pb][(c - 1) & 31][i];
        chunk_correct<M>(L, x, xl, xs);
        // ---- q += dq: the increments go back into the tile and leave as a reduce-add
        if (SWZ) {
#pragma unroll
            for (int m = 0; m < M; m += 2) {
                tA[m * 8] = odd ? x[m + 1] : x[m];
                tB[m * 8] = odd ? x[m] : x[m + 1];
            }
        } else {
#pragma unroll
            for (int m = 0; m < M; m++) tl[m * 8] = x[m];
        }
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            const double* t = tile0 + pb * NY * 8;
            if (A.slab) for (int b = 0; b < nb; b++) tma_store_2d(&Mp.d[comp], col0, k * NY + b * Mp.box_rows, t + b * Mp.box_rows * 8);
            else for (int b = 0; b < nb; b++) tma_reduce_add_2d(&Mp.q[comp], col0, k * NY + b * Mp.box_rows, t + b * Mp.box_rows * 8);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait_all<0>();
}
#endif  // __CUDACC__

}  // namespace fsei
