// fsei.cu -- libfsei: kernels and the C ABI of include/fsei.h (sm_100a, fp64).
//
// One projection = a1 divergence -> a2 x-forward -> a3 y-forward -> a4 z-tridiagonal (+ gauge
// column) -> a5 y-inverse -> a6 x-inverse -> a7 projection, all in place in the caller's phi
// buffer (packed half spectrum: nx/2 complex per row = the bytes of the real row).
// DESIGN.md sec. 6 describes each kernel, its launch shape and its algorithmic bytes.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/fsei.h"
#include "plan_host.hpp"
#include "stencil.cuh"
#include "xfft.cuh"
#include "yfft.cuh"
#include "zsolve.cuh"
#include "fast_launch.hpp"
#include "fast_configs.hpp"
#include "zfast.cuh"
#include "stencil_fast.cuh"
#include "fluid.cuh"
#include "ibm.cuh"
#include "visc_fast.cuh"
#include "tma_host.hpp"
#include <cmath>
#include <cstdlib>
#include <mutex>

using namespace fsei;

// ------------------------------------------------------------------------------------------
// error state
// ------------------------------------------------------------------------------------------
static thread_local std::string g_err;
static thread_local int g_err_code = FSEI_OK;
static int fail(int code, const std::string& msg) { g_err = msg; g_err_code = code; return code; }
static int cuda_fail(cudaError_t e, const char* what)
{
    return fail(FSEI_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
static bool misaligned(const void* p) { return (reinterpret_cast<size_t>(p) & 15u) != 0; }
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)
static int noalloc_resolve(double** out, int* dev_out);      // fsei_viscous_step_noalloc: device address of its static scratch array

// ------------------------------------------------------------------------------------------
// plan
// ------------------------------------------------------------------------------------------
#define FSEI_VSLOTS 4
enum { K_DIV = 0, K_XF, K_YF, K_GAUGE, K_ZD, K_ZP, K_YI, K_XI, K_PROJ, K_DIVXF, K_YZF, K_YZB, K_EXPL, K_VFACT, K_VX, K_VY, K_VZ, K_MLS, K_VXZ, K_VZY, K_MLSAPPLY, FSEI_NKERNELS };

struct fsei_plan {
    HostTables T;
    XParams X; YParams Y; ZParams Z; SParams S;
    bool fast = false;                 // register-resident Stockham path (xfast / yfast / zfast), natural-order spectrum
    XFast XF; YFast YF; ZFast ZF;
    int kchunk_inv = 16;               // planes per CTA of the x-inverse kernel (XF.kchunk: of the x-forward kernel)
    bool fused = false;                // fast path on the blocked spectrum layout with the z sweeps fused into the y kernels
    YZFused YZ; TmaMap3D xi_map; cplx* work = nullptr;   // work: plan-owned spectrum field (blocked layout)
    std::vector<void*> owned;          // device allocations freed with the plan
    size_t bytes = 0;
    int LX = 1, CY = 1;                // tile shapes
    size_t smem_x = 0, smem_y = 0;
    int last_launches = 0;
    const double* zc_dev = nullptr;      // z-face coordinates (IB-MLS node positions)
    SParams Sg;                        // slab plans: the stencil parameters of the GLOBAL grid (z tables of the viscous step)
    bool slab = false; int k0 = 0, k1 = 0, s0 = 0, s1 = 0;   // z-slab / x-slot-pencil share of a multi-GPU decomposition (fsei_slab_plan_create)
    // implicit viscous step: factorisation tables of the last FSEI_VSLOTS values of beta (a three-stage Runge-Kutta scheme
    // cycles through three), device tables in vtab[slot], host-built line tables of the fast family beside them
    int nsm = 148;                     // SMs of the plan's device
    bool visc_fast = false; VFastLine vline_x[FSEI_VSLOTS], vline_y[FSEI_VSLOTS]; int vnsig_x[FSEI_VSLOTS], vnsig_y[FSEI_VSLOTS];
    double* vtab = nullptr; int vnmax = 0; double visc_beta[FSEI_VSLOTS] = {NAN, NAN, NAN, NAN}; int visc_next = 0;
    double* hostpath[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // device u,v,w,p,phi of the host-buffer entry
    double* noalloc_tab = nullptr; int noalloc_dev = -1; int noalloc_err = 0;   // fsei_viscous_step_noalloc: static scratch of the plan's device
    cudaStream_t host_up = nullptr, host_dn = nullptr;                     // its copy streams (p up / results down, in z chunks)
    std::vector<cudaEvent_t> host_ev;
    // per-kernel CUDA-event timing (fsei_plan_profile): event pairs recorded around every launch
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;      // 2 events per recorded launch
    std::vector<int> ev_kid;               // kernel id of each recorded launch
    size_t ev_used = 0;
    double prof_ms[FSEI_NKERNELS] = {0};
    long prof_n[FSEI_NKERNELS] = {0};
};

static const char* const k_names[FSEI_NKERNELS] = {"divergence", "x_forward", "y_forward", "z_gauge", "z_direct", "z_paired",
                                                   "y_inverse", "x_inverse", "project", "div_x_forward", "yz_forward", "yz_backward",
                                                   "explicit_terms", "visc_factor", "visc_x", "visc_y", "visc_z", "ib_mls", "visc_xz", "visc_zy", "ib_apply"};

// record an event pair around one launch when profiling is on
struct LaunchTimer {
    fsei_plan* P; cudaStream_t st; bool on;
    LaunchTimer(fsei_plan* P_, int kid, cudaStream_t st_) : P(P_), st(st_), on(P_->profiling) {
        if (!on) return;
        if (P->ev_used + 2 > P->ev_pool.size()) { on = false; return; }      // pool exhausted (2048 launches since the last read): stop recording
        P->ev_kid.push_back(kid);
        cudaEventRecord(P->ev_pool[P->ev_used], st);
    }
    ~LaunchTimer() { if (on) { cudaEventRecord(P->ev_pool[P->ev_used + 1], st); P->ev_used += 2; } }
};

template <class T> static int upload(fsei_plan* P, const std::vector<T>& h, const T** d)
{
    void* p = nullptr;
    size_t n = h.size() * sizeof(T);
    if (n == 0) { *d = nullptr; return FSEI_OK; }
    cudaError_t e = cudaMalloc(&p, n);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(FSEI_ERR_ALLOC, std::string("cudaMalloc of a plan table failed: ") + cudaGetErrorString(e)); }
    P->owned.push_back(p); P->bytes += n;
    CU(cudaMemcpy(p, h.data(), n, cudaMemcpyHostToDevice));
    *d = static_cast<const T*>(p);
    return FSEI_OK;
}
static int dalloc(fsei_plan* P, size_t n, void** d)
{
    cudaError_t e = cudaMalloc(d, n);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(FSEI_ERR_ALLOC, std::string("cudaMalloc of plan workspace failed: ") + cudaGetErrorString(e)); }
    P->owned.push_back(*d); P->bytes += n;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// kernels
// ------------------------------------------------------------------------------------------
#define NT 256

// generic family: CTAs per SM the FORWARD transform kernels are compiled for (they would take 148 registers = one CTA per SM; the
// inverse ones fit two as they are and lose when squeezed) -- with the shared-memory carve-out of the forward kernels set to its
// maximum in plan_build, or the driver's default admits ONE 28-64 KB tile per SM (the inverse kernels get two by default and
// want their L1: with the maximum carve-out y_inverse goes from 4.9 to 7.5 ms at configs[3])
#ifndef FSEI_GEN_MINB
#define FSEI_GEN_MINB 2
#endif
template <bool INV> __device__ __forceinline__ void x_all_passes(const XParams& X, cplx* sm, int lines)
{
    int Ns[8]; int n = X.N;
#pragma unroll
    for (int s = 0; s < 8; s++) { Ns[s] = n; if (s < X.f.npass) n /= X.f.radix[s]; }
    for (int i = 0; i < X.f.npass; i++) {
        int s = INV ? X.f.npass - 1 - i : i;
        x_pass_dispatch<INV>(X, sm, lines, X.f.radix[s], Ns[s], threadIdx.x, NT);
        __syncthreads();
    }
}

__global__ void __launch_bounds__(NT, FSEI_GEN_MINB) k_x_forward(XParams X, const double* src, cplx* dst, long nlines, int LX)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    cplx* sm = reinterpret_cast<cplx*>(smraw);
    long l0 = (long)blockIdx.x * LX;
    int lines = (int)((nlines - l0 < LX) ? nlines - l0 : LX);
    x_load_real(X, sm, src + (size_t)l0 * X.n, lines, threadIdx.x, NT);
    __syncthreads();
    x_all_passes<false>(X, sm, lines);
    x_post_forward(X, sm, lines, threadIdx.x, NT);
    __syncthreads();
    x_store_spec(X, sm, dst + (size_t)l0 * X.N, lines, threadIdx.x, NT);
}

__global__ void __launch_bounds__(NT) k_x_inverse(XParams X, const cplx* src, double* dst, long nlines, int LX)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    cplx* sm = reinterpret_cast<cplx*>(smraw);
    long l0 = (long)blockIdx.x * LX;
    int lines = (int)((nlines - l0 < LX) ? nlines - l0 : LX);
    x_load_spec(X, sm, src + (size_t)l0 * X.N, lines, threadIdx.x, NT);
    __syncthreads();
    x_pre_inverse(X, sm, lines, threadIdx.x, NT);
    __syncthreads();
    x_all_passes<true>(X, sm, lines);
    x_store_real(X, sm, dst + (size_t)l0 * X.n, lines, threadIdx.x, NT);
}

template <bool INV, bool NEU> __device__ __forceinline__ void y_all_passes(const YParams& Y, cplx* sm, int C)
{
    int Ns[8]; int n = Y.N;
#pragma unroll
    for (int s = 0; s < 8; s++) { Ns[s] = n; if (s < Y.f.npass) n /= Y.f.radix[s]; }
    for (int i = 0; i < Y.f.npass; i++) {
        int s = INV ? Y.f.npass - 1 - i : i;
        y_pass_dispatch<INV, NEU>(Y, sm, C, Y.f.radix[s], Ns[s], threadIdx.x, NT);
        __syncthreads();
    }
}

// grid (nxc / C, nz): one tile = C adjacent slots of every row of one z-plane
template <bool INV, bool NEU>
__global__ void __launch_bounds__(NT, (INV ? 0 : FSEI_GEN_MINB)) k_y_transform(YParams Y, cplx* spec, int nxc, int C)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    cplx* sm = reinterpret_cast<cplx*>(smraw);
    cplx* g = spec + (size_t)blockIdx.y * Y.N * nxc + (size_t)blockIdx.x * C;
    y_load(sm, g, nxc, Y.N, C, threadIdx.x, NT);
    __syncthreads();
    if (INV && NEU) { y_pre_inverse_dct(Y, sm, C, threadIdx.x, NT); __syncthreads(); }
    y_all_passes<INV, NEU>(Y, sm, C);
    if (!INV && NEU) { y_post_forward_dct(Y, sm, C, threadIdx.x, NT); __syncthreads(); }
    y_store(sm, g, nxc, Y.N, C, threadIdx.x, NT);
}

__global__ void __launch_bounds__(NT) k_z_factor(ZParams Z, double* ipiv, int paired_slot0)
{
    size_t t = (size_t)blockIdx.x * NT + threadIdx.x;
    size_t n = (size_t)Z.ny * Z.nxc * Z.ncomp;
    if (t >= n) return;
    int comp = (int)(t % Z.ncomp); size_t r = t / Z.ncomp; int slot = (int)(r % Z.nxc), row = (int)(r / Z.nxc);
    bool zero = (row == 0 && slot == 0 && comp == 0) || (paired_slot0 && slot == 0);
    z_factor_column(Z, ipiv, row, slot, comp, zero);
}

// slots [slot0, nxc) of every row, slot fastest across the warp (coalesced 16-byte accesses)
template <int NCOMP>
__global__ void __launch_bounds__(128) k_z_direct(ZParams Z, cplx* spec, int slot0)
{
    const int ns = Z.nxc - slot0;
    size_t t = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (t >= (size_t)ns * Z.ny) return;
    int slot = slot0 + (int)(t % ns), row = (int)(t / ns);
    z_direct_column<NCOMP>(Z, spec, row, slot, row == 0 && slot == 0);
}

// pairs (slot, q): slot fastest
__global__ void __launch_bounds__(128) k_z_paired(ZParams Z, cplx* spec, int nslots)
{
    size_t npairs = (size_t)(Z.ny / 2 + 1) * nslots;
    size_t t = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (t >= npairs) return;
    int slot = (int)(t % nslots), q = (int)(t / nslots);
    z_paired_column(Z, spec, slot, q, t, npairs);
}

// the (0,0) column: gather it, solve it (thread 0, in shared memory), leave it in Z.gauge
__global__ void __launch_bounds__(NT) k_z_gauge(ZParams Z, const cplx* spec, double* gauge)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    double* d = reinterpret_cast<double*>(smraw);
    double* x = d + Z.nz;
    for (int k = threadIdx.x; k < Z.nz; k += NT) d[k] = spec[zidx(Z, k, 0, 0)].re;
    __syncthreads();
    if (threadIdx.x == 0) z_gauge_serial(Z, d, x);
    __syncthreads();
    for (int k = threadIdx.x; k < Z.nz; k += NT) gauge[k] = x[k];
}

// ------------------------------------------------------------------------------------------
// plan creation
// ------------------------------------------------------------------------------------------
static int plan_build(fsei_plan* P, int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy, unsigned flags)
{
    int code = 0;
    // fast path: line lengths with a register-resident Stockham instantiation, special columns fit in shared memory
    // fused path: the fast path on the blocked layout, where one CTA per x-slot tile marches along z -- for grids
    // with enough tiles to fill the GPU.  flags (fsei_plan_create_ex) may override the choice, per plan.
    if (flags & ~(unsigned)(FSEI_PLAN_PATH_MASK | FSEI_PLAN_TWIST_OFF | FSEI_PLAN_TWIST_ON | FSEI_PLAN_HOST_FIELDS | FSEI_PLAN_VISC_GENERIC)) return fail(FSEI_ERR_ARG, "fsei_plan_create_ex: unknown flag");
    if ((flags & FSEI_PLAN_TWIST_OFF) && (flags & FSEI_PLAN_TWIST_ON)) return fail(FSEI_ERR_ARG, "fsei_plan_create_ex: TWIST_OFF and TWIST_ON are exclusive");
    const unsigned pf = flags & FSEI_PLAN_PATH_MASK;
    const std::string want = pf == FSEI_PLAN_PATH_GENERIC ? "generic" : (pf == FSEI_PLAN_PATH_FAST ? "fast" : (pf == FSEI_PLAN_PATH_FUSED ? "fused" : ""));
    const bool fast = want != "generic" && nx >= 4 && ny >= 2 && xfast_supported(nx / 2) && yfast_supported(ny) &&
                      (size_t)nz * 4 * sizeof(cplx) <= 200 * 1024;
    const bool fused_ok = fast && xblocked_supported(nx / 2) && yzfused_supported(ny) && (nx / 2) % FSEI_CB == 0;
    const bool fused = fused_ok && want != "fast" && (want == "fused" || (nx / 2) / FSEI_CB >= 128);
    std::string msg = build_tables(P->T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code, fast);
    if (code) return fail(code, msg);
    P->fast = fast; P->fused = fused;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(FSEI_ERR_CUDA, "no CUDA device: libfsei has no CPU fallback"); }

    HostTables& T = P->T;
    int rc;
    XParams& X = P->X; YParams& Y = P->Y; ZParams& Z = P->Z; SParams& S = P->S;
    X.n = nx; X.N = nx / 2; X.bc = bcx; X.pitch = padx(nx / 2) + 1; X.f = T.fx; X.scale = T.scale;
    if ((rc = upload(P, T.twx, &X.tw))) return rc;
    if ((rc = upload(P, T.posx, &X.pos))) return rc;
    if ((rc = upload(P, T.twx_r2c, &X.tw_r2c))) return rc;
    if ((rc = upload(P, T.twx_dct, &X.tw_dct))) return rc;
    Y.N = ny; Y.bc = bcy; Y.f = T.fy;
    if ((rc = upload(P, T.twy, &Y.tw))) return rc;
    if ((rc = upload(P, T.posy, &Y.pos))) return rc;
    if ((rc = upload(P, T.twy_dct, &Y.tw_dct))) return rc;
    Z.nxc = T.nxc; Z.ny = ny; Z.nz = nz; Z.ncomp = T.ncomp; Z.posy = Y.pos;
    if ((rc = upload(P, T.za, &Z.za))) return rc;
    if ((rc = upload(P, T.zcc, &Z.zcc))) return rc;
    if ((rc = upload(P, T.dzc, &Z.dzc))) return rc;
    if ((rc = upload(P, T.dzm, &Z.dzm))) return rc;
    if ((rc = upload(P, T.lamx, &Z.lamx))) return rc;
    if ((rc = upload(P, T.lamy, &Z.lamy))) return rc;
    S.nx = nx; S.ny = ny; S.nz = nz; S.bcx = bcx; S.bcy = bcy; S.rdx = T.rdx; S.rdy = T.rdy;
    if ((rc = upload(P, T.rdzc, &S.rdzc))) return rc;
    if ((rc = upload(P, T.rdzm, &S.rdzm))) return rc;
    { std::vector<double> zcv(zc, zc + nz + 1); if ((rc = upload(P, zcv, &P->zc_dev))) return rc; }
    {
        P->vnmax = nx > ny ? (nx > nz ? nx : nz) : (ny > nz ? ny : nz);
        void* q = nullptr;
        if ((rc = dalloc(P, sizeof(double) * FSEI_VSLOTS * 9 * vtab_set_doubles(P->vnmax), &q))) return rc;
        P->vtab = static_cast<double*>(q);
        CU(kernel_smem(k_explicit_terms, FSEI_EXPL_SMEM_MAX));
        P->visc_fast = !(flags & FSEI_PLAN_VISC_GENERIC) && bcx == BC_PERIODIC && bcy == BC_PERIODIC && visc_fast_supported(nx, ny);
        if (P->visc_fast) {
            CU(visc_fast_init());
            int dev = 0;
            CU(cudaGetDevice(&dev)); CU(cudaDeviceGetAttribute(&P->nsm, cudaDevAttrMultiProcessorCount, dev));
        }
    }

    if (fast) {
        XFast& XF = P->XF; YFast& YF = P->YF; ZFast& ZF = P->ZF;
        XF.nx = nx; XF.ny = ny; XF.nz = nz; XF.N = nx / 2; XF.tw = X.tw; XF.tw_r2c = X.tw_r2c; XF.tw_dct = X.tw_dct; XF.scale = T.scale;
        {
            // planes per CTA of the x kernels: 16 on large grids (amortises the table fill and gives the fused divergence
            // its w(k+1) reuse), fewer on small ones so that the grid still covers the SMs a few times
            int dev = 0, nsm = 148;
            cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
            const int lpb = xfast_lines_per_block(nx / 2, bcx == BC_NEUMANN);
            const long jblocks = (ny + lpb - 1) / lpb;
            long kc = (jblocks * nz) / (4L * nsm);
            // measured at configs[3]: the fused forward kernel likes long marches (w reuse, fewer table fills), the inverse
            // kernel shorter ones
            XF.kchunk = (int)(kc < 1 ? 1 : (kc > 64 ? 64 : kc));
            P->kchunk_inv = (int)(kc < 1 ? 1 : (kc > 32 ? 32 : kc));
        }
        YF.nxc = T.nxc; YF.ny = ny; YF.nz = nz; YF.tw = Y.tw; YF.tw_dct = Y.tw_dct;
        YF.untangle = (bcy == BC_PERIODIC) ? (bcx == BC_PERIODIC ? 1 : T.nxc) : 0;
        ZF.nxc = T.nxc; ZF.ny = ny; ZF.nz = nz; ZF.bcx = bcx; ZF.bcy = bcy;
        ZF.ncomp = (bcx == BC_PERIODIC && bcy == BC_PERIODIC) ? 1 : 2;
        ZF.za = Z.za; ZF.zcc = Z.zcc; ZF.lamx = Z.lamx; ZF.lamy = Z.lamy; ZF.dzc = Z.dzc; ZF.dzm = Z.dzm;
        void* q = nullptr;
        if ((rc = dalloc(P, sizeof(cplx) * 2 * nz, &q))) return rc;
        ZF.special = static_cast<cplx*>(q);
        if ((rc = dalloc(P, sizeof(double) * 8 * nz, &q))) return rc;
        ZF.cpw = static_cast<double*>(q);
        ZF.cb = fused ? FSEI_CB : 0; ZF.special_in = nullptr;
        // Twisted factorisation (two CTAs per tile sweeping towards each other) where one CTA per tile would leave SMs
        // idle: fewer tiles than SMs.  FSEI_PLAN_TWIST_OFF / _ON override.
        int nsm = 148;
        { int dev = 0; CU(cudaGetDevice(&dev)); CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev)); }
        // ... or three-warp CTAs (ny = 3 2^a) that cannot fill their SM even two at a time (configs[4]: 23.5 -> 22.1 ms)
        bool twist = fused && nz >= 4 && (T.nxc / FSEI_CB <= nsm || (yzfused_block_threads(ny) < 128 && T.nxc / FSEI_CB <= 2 * nsm));
        if (flags & (FSEI_PLAN_TWIST_OFF | FSEI_PLAN_TWIST_ON)) twist = fused && nz >= 4 && (flags & FSEI_PLAN_TWIST_ON);
        ZF.ktw = twist ? nz / 2 : nz;
        if (fused) {
            if ((rc = dalloc(P, sizeof(cplx) * 2 * nz, &q))) return rc;
            CU(cudaMemset(q, 0, sizeof(cplx) * 2 * nz));
            ZF.special_in = static_cast<const cplx*>(q);
        }
        size_t nip = (size_t)nz * ny * T.nxc * ZF.ncomp;
        if ((rc = dalloc(P, sizeof(double) * nip, &q))) return rc;
        ZF.ipiv = static_cast<const double*>(q);
        size_t cols = (size_t)ny * T.nxc * ZF.ncomp;
        k_zf_factor<<<(unsigned)((cols + 255) / 256), 256>>>(ZF, static_cast<double*>(q));
        CU(cudaGetLastError());
        k_z_special_factor<<<1, 32>>>(ZF);
        CU(cudaGetLastError());
        CU(cudaDeviceSynchronize());
        CU(xfast_init());
        CU(yfast_init());
        if (fused) {
            YZFused& YZ = P->YZ;
            YZ.nxc = T.nxc; YZ.ny = ny; YZ.nz = nz; YZ.untangle = YF.untangle;
            YZ.pp = (bcx == BC_PERIODIC && bcy == BC_PERIODIC) ? 1 : 0;
            YZ.tw = Y.tw; YZ.tw_dct = Y.tw_dct; YZ.za = Z.za; YZ.zcc = Z.zcc; YZ.ip = ZF.ipiv;
            YZ.special_in = const_cast<cplx*>(ZF.special_in); YZ.special = ZF.special;
            {
                // CTAs are dealt to the SMs breadth first: with nsm < total < 2 nsm CTAs the linear ids total - nsm .. nsm - 1
                // get an SM to themselves; the tile that carries the split / merge work of a (P,P) grid (tile 0: the
                // straggler) is given such an id in each half of the grid
                const int ntiles = T.nxc / FSEI_CB, halves = twist ? 2 : 1, total = ntiles * halves;
                for (int h = 0; h < 2; h++) {
                    int bx0 = 0;
                    if (total > nsm && total < 2 * nsm) {
                        const int lo = total - nsm, hi = nsm - 1;             // lonely linear ids, inclusive
                        int cand = hi - ntiles * h;                           // blockIdx.x of linear id hi in half h
                        if (cand >= ntiles) cand = ntiles - 1;
                        if (cand >= 0 && cand + ntiles * h >= lo) bx0 = cand;
                    }
                    YZ.tile_shift[h] = (ntiles - bx0) % ntiles;
                }
            }
            YZ.ktw = ZF.ktw; YZ.mid = nullptr;
            if (twist) {
                if ((rc = dalloc(P, sizeof(cplx) * (size_t)T.nxc * ny * 2, &q))) return rc;
                YZ.mid = static_cast<cplx*>(q);
            }
            if ((rc = dalloc(P, sizeof(double) * (size_t)nx * ny * nz, &q))) return rc;
            P->work = static_cast<cplx*>(q);
            CU(xblocked_init());
            CU(yzfused_init());
            CU(make_xi_blocked_map(XF, bcx == BC_NEUMANN, P->work, &P->xi_map));
        }
        CU(cudaFuncSetAttribute(k_z_special, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)z_special_smem(nz, z_special_staged(nz))));
        return FSEI_OK;
    }

    void* g = nullptr;
    if ((rc = dalloc(P, sizeof(double) * nz, &g))) return rc;
    Z.gauge = static_cast<const double*>(g);
    const size_t npairs = (size_t)(ny / 2 + 1) * (T.paired_all ? T.nxc : 1);
    if (T.paired_all || T.paired_slot0) {
        void* c = nullptr;
        if ((rc = dalloc(P, sizeof(double) * 2 * npairs * nz, &c))) return rc;
        Z.cpw = static_cast<double*>(c);
    } else Z.cpw = nullptr;
    Z.ipiv = nullptr;
    if (!T.paired_all) {
        void* ip = nullptr;
        size_t n = (size_t)nz * ny * T.nxc * T.ncomp;
        if ((rc = dalloc(P, sizeof(double) * n, &ip))) return rc;
        Z.ipiv = static_cast<const double*>(ip);
        size_t cols = (size_t)ny * T.nxc * T.ncomp;
        k_z_factor<<<(unsigned)((cols + NT - 1) / NT), NT>>>(Z, static_cast<double*>(ip), T.paired_slot0 ? 1 : 0);
        CU(cudaGetLastError());
        CU(cudaDeviceSynchronize());
    }

    // tile shapes
    size_t line_bytes = (size_t)X.pitch * sizeof(cplx);
    int LX = (int)(32768 / line_bytes); if (LX < 1) LX = 1; if (LX > 32) LX = 32;
    P->LX = LX; P->smem_x = LX * line_bytes;
    int CY = 1;
    for (int c = 8; c >= 1; c /= 2)
        if (T.nxc % c == 0 && (size_t)ny * c * sizeof(cplx) <= 65536) { CY = c; break; }
    if ((size_t)ny * CY * sizeof(cplx) > 200 * 1024) return fail(FSEI_ERR_SIZE, "ny too large for the shared-memory y tile");
    P->CY = CY; P->smem_y = (size_t)ny * CY * sizeof(cplx);
    CU(cudaFuncSetAttribute(k_z_gauge, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * sizeof(double) * nz)));
    CU(cudaFuncSetAttribute(k_x_forward, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_x));
    CU(cudaFuncSetAttribute(k_x_forward, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    CU(cudaFuncSetAttribute(k_x_inverse, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_x));
    CU(cudaFuncSetAttribute(k_y_transform<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_y));
    CU(cudaFuncSetAttribute(k_y_transform<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    CU(cudaFuncSetAttribute(k_y_transform<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_y));
    CU(cudaFuncSetAttribute(k_y_transform<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_y));
    CU(cudaFuncSetAttribute(k_y_transform<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    CU(cudaFuncSetAttribute(k_y_transform<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->smem_y));
    return FSEI_OK;
}

static int host_fields(fsei_plan* P)
{
    const size_t bytes = sizeof(double) * (size_t)P->T.nx * P->T.ny * P->T.nz;
    for (int f = 0; f < 5; f++)
        if (!P->hostpath[f]) {
            cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&P->hostpath[f]), bytes);
            if (e != cudaSuccess) { cudaGetLastError(); P->hostpath[f] = nullptr; return fail(FSEI_ERR_ALLOC, "cudaMalloc of a device field failed"); }
            P->bytes += bytes;
        }
    return FSEI_OK;
}

extern "C" fsei_plan* fsei_plan_create_ex(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bc_x, int bc_y,
                                          unsigned flags)
{
    fsei_plan* P = new (std::nothrow) fsei_plan();
    if (!P) { fail(FSEI_ERR_ALLOC, "out of host memory"); return nullptr; }
    int rc = plan_build(P, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, flags);
    if (rc == FSEI_OK && (flags & FSEI_PLAN_HOST_FIELDS)) rc = host_fields(P);
    if (rc == FSEI_OK) {                                       // set-up of fsei_viscous_step_noalloc; a failure surfaces in that call only
        P->noalloc_err = noalloc_resolve(&P->noalloc_tab, &P->noalloc_dev);
        if (P->noalloc_err) P->noalloc_tab = nullptr;
    }
    if (rc != FSEI_OK) { const std::string msg = g_err; fsei_plan_destroy(P); g_err = msg; g_err_code = rc; return nullptr; }
    g_err_code = FSEI_OK; g_err.clear();
    return P;
}

extern "C" fsei_plan* fsei_plan_create(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bc_x, int bc_y)
{
    return fsei_plan_create_ex(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, 0u);
}

// 0: generic, 1: fast, 2: fused (+4 when the twisted factorisation is on)
extern "C" int fsei_plan_kernel_family(const fsei_plan* P)
{
    if (!P) return -FSEI_ERR_ARG;
    return (P->fused ? 2 : (P->fast ? 1 : 0)) + ((P->fused && P->ZF.ktw != P->T.nz) ? 4 : 0);
}

extern "C" void fsei_plan_destroy(fsei_plan* P)
{
    if (!P) return;
    for (void* p : P->owned) cudaFree(p);
    for (double* p : P->hostpath) if (p) cudaFree(p);
    for (cudaEvent_t e : P->ev_pool) cudaEventDestroy(e);
    for (cudaEvent_t e : P->host_ev) cudaEventDestroy(e);
    if (P->host_up) cudaStreamDestroy(P->host_up);
    if (P->host_dn) cudaStreamDestroy(P->host_dn);
    delete P;
}

extern "C" const char* fsei_last_error(void) { return g_err.c_str(); }
extern "C" int fsei_last_error_code(void) { return g_err_code; }
extern "C" size_t fsei_plan_workspace_bytes(const fsei_plan* P) { return P ? P->bytes : 0; }
extern "C" int fsei_plan_last_launch_count(const fsei_plan* P) { return P ? P->last_launches : 0; }

// ------------------------------------------------------------------------------------------
// the calls
// ------------------------------------------------------------------------------------------
extern "C" int fsei_divergence(fsei_plan* P, const double* u, const double* v, const double* w, double alpha_dt,
                               double* rhs, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_divergence: this is a slab plan (use the fsei_slab_* calls)");
    if (!P || !u || !v || !w || !rhs) return fail(FSEI_ERR_ARG, "fsei_divergence: NULL argument");
    if (alpha_dt == 0.0 || alpha_dt != alpha_dt) return fail(FSEI_ERR_ARG, "fsei_divergence: alpha_dt must be non-zero");
    if (rhs == u || rhs == v || rhs == w) return fail(FSEI_ERR_ARG, "fsei_divergence: rhs must not alias u, v, w");
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(rhs)) return fail(FSEI_ERR_ARG, "fsei_divergence: field pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    size_t n = (size_t)P->T.nx * P->T.ny * P->T.nz;
    { LaunchTimer t(P, K_DIV, st); k_divergence_fast<<<(unsigned)((n / 2 + 255) / 256), 256, 0, st>>>(P->S, u, v, w, 1.0 / alpha_dt, rhs); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

// a3 .. a6 of the fast path on a spectrum already in x-forward form: y forward, z solve, y inverse, x inverse
static int fast_spectral_solve(fsei_plan* P, cplx* spec, cudaStream_t st)
{
    const HostTables& T = P->T;
    const bool ny_neu = T.bcy == BC_NEUMANN;
    { LaunchTimer t(P, K_YF, st); CU(launch_y_fast(P->YF, false, ny_neu, spec, st)); }
    { LaunchTimer t(P, K_GAUGE, st); k_z_special<<<1, 128, z_special_smem(T.nz, z_special_staged(T.nz)), st>>>(P->ZF, spec, z_special_staged(T.nz)); }
    CU(cudaGetLastError());
    {
        LaunchTimer t(P, K_ZD, st);
        size_t nthr = (size_t)T.nxc * T.ny;
        if (T.nz <= 32) k_zf_pcr<<<(unsigned)((nthr * 32 + 127) / 128), 128, 0, st>>>(P->ZF, spec);     // one warp per column
        else if (P->ZF.ncomp == 1) k_zf_sweep<1><<<(unsigned)((nthr + 127) / 128), 128, 0, st>>>(P->ZF, spec);
        else k_zf_sweep<2><<<(unsigned)((nthr + 127) / 128), 128, 0, st>>>(P->ZF, spec);
    }
    CU(cudaGetLastError());
    { LaunchTimer t(P, K_YI, st); CU(launch_y_fast(P->YF, true, ny_neu, spec, st)); }
    { LaunchTimer t(P, K_XI, st); XFast xi = P->XF; xi.kchunk = P->kchunk_inv; CU(launch_xi_fast(xi, T.bcx == BC_NEUMANN, spec, reinterpret_cast<double*>(spec), st)); }
    return FSEI_OK;
}

// a3 .. a6 of the fused path on the blocked spectrum in the plan's workspace; phi receives the result
static int fused_spectral_solve(fsei_plan* P, double* phi, cudaStream_t st)
{
    const HostTables& T = P->T;
    const bool ny_neu = T.bcy == BC_NEUMANN;
    { LaunchTimer t(P, K_YZF, st); CU(launch_yz_forward(P->YZ, ny_neu, P->ZF.ncomp, P->work, st)); }
    { LaunchTimer t(P, K_GAUGE, st); k_z_special<<<1, 128, z_special_smem(T.nz, z_special_staged(T.nz)), st>>>(P->ZF, P->work, z_special_staged(T.nz)); }
    CU(cudaGetLastError());
    { LaunchTimer t(P, K_YZB, st); CU(launch_yz_backward(P->YZ, ny_neu, P->ZF.ncomp, P->work, st)); }
    { LaunchTimer t(P, K_XI, st); XFast xi = P->XF; xi.kchunk = P->kchunk_inv; CU(launch_xi_fast(xi, T.bcx == BC_NEUMANN, P->work, phi, st, &P->xi_map)); }
    return FSEI_OK;
}

extern "C" int fsei_poisson_solve(fsei_plan* P, const double* rhs, double* phi, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_poisson_solve: this is a slab plan (use the fsei_slab_* calls)");
    if (!P || !rhs || !phi) return fail(FSEI_ERR_ARG, "fsei_poisson_solve: NULL argument");
    if (misaligned(rhs) || misaligned(phi)) return fail(FSEI_ERR_ARG, "fsei_poisson_solve: field pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostTables& T = P->T;
    const long nlines = (long)T.ny * T.nz;
    cplx* spec = reinterpret_cast<cplx*>(phi);
    int launches = 0;
    if (P->fused) {
        { LaunchTimer t(P, K_XF, st); CU(launch_xf_fast(P->XF, P->S, T.bcx == BC_NEUMANN, false, rhs, nullptr, nullptr, 0.0, P->work, st, true)); }
        int rc = fused_spectral_solve(P, phi, st);
        if (rc) return rc;
        P->last_launches = 5;
        return FSEI_OK;
    }
    if (P->fast) {
        { LaunchTimer t(P, K_XF, st); CU(launch_xf_fast(P->XF, P->S, T.bcx == BC_NEUMANN, false, rhs, nullptr, nullptr, 0.0, spec, st)); }
        int rc = fast_spectral_solve(P, spec, st);
        if (rc) return rc;
        P->last_launches = 6;
        return FSEI_OK;
    }
    unsigned gx = (unsigned)((nlines + P->LX - 1) / P->LX);
    { LaunchTimer t(P, K_XF, st); k_x_forward<<<gx, NT, P->smem_x, st>>>(P->X, rhs, spec, nlines, P->LX); launches++; }
    CU(cudaGetLastError());
    dim3 gy(T.nxc / P->CY, T.nz);
    {
        LaunchTimer t(P, K_YF, st);
        if (T.bcy == BC_NEUMANN) k_y_transform<false, true><<<gy, NT, P->smem_y, st>>>(P->Y, spec, T.nxc, P->CY);
        else k_y_transform<false, false><<<gy, NT, P->smem_y, st>>>(P->Y, spec, T.nxc, P->CY);
        launches++;
    }
    CU(cudaGetLastError());
    { LaunchTimer t(P, K_GAUGE, st); k_z_gauge<<<1, NT, 2 * sizeof(double) * T.nz, st>>>(P->Z, spec, const_cast<double*>(P->Z.gauge)); launches++; }
    CU(cudaGetLastError());
    if (T.paired_all) {
        size_t np = (size_t)(T.ny / 2 + 1) * T.nxc;
        LaunchTimer t(P, K_ZP, st);
        k_z_paired<<<(unsigned)((np + 127) / 128), 128, 0, st>>>(P->Z, spec, T.nxc); launches++;
    } else {
        int s0 = T.paired_slot0 ? 1 : 0;
        size_t nthr = (size_t)(T.nxc - s0) * T.ny;
        {
            LaunchTimer t(P, K_ZD, st);
            if (T.ncomp == 1) k_z_direct<1><<<(unsigned)((nthr + 127) / 128), 128, 0, st>>>(P->Z, spec, s0);
            else k_z_direct<2><<<(unsigned)((nthr + 127) / 128), 128, 0, st>>>(P->Z, spec, s0);
            launches++;
        }
        CU(cudaGetLastError());
        if (T.paired_slot0) {
            size_t np = (size_t)(T.ny / 2 + 1);
            LaunchTimer t(P, K_ZP, st);
            k_z_paired<<<(unsigned)((np + 127) / 128), 128, 0, st>>>(P->Z, spec, 1); launches++;
        }
    }
    CU(cudaGetLastError());
    {
        LaunchTimer t(P, K_YI, st);
        if (T.bcy == BC_NEUMANN) k_y_transform<true, true><<<gy, NT, P->smem_y, st>>>(P->Y, spec, T.nxc, P->CY);
        else k_y_transform<true, false><<<gy, NT, P->smem_y, st>>>(P->Y, spec, T.nxc, P->CY);
        launches++;
    }
    CU(cudaGetLastError());
    { LaunchTimer t(P, K_XI, st); k_x_inverse<<<gx, NT, P->smem_x, st>>>(P->X, spec, phi, nlines, P->LX); launches++; }
    CU(cudaGetLastError());
    P->last_launches = launches;
    return FSEI_OK;
}

extern "C" int fsei_project(fsei_plan* P, double* u, double* v, double* w, double* p, const double* phi,
                            double alpha_dt, double beta, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_project: this is a slab plan (use the fsei_slab_* calls)");
    if (!P || !u || !v || !w || !p || !phi) return fail(FSEI_ERR_ARG, "fsei_project: NULL argument");
    if (alpha_dt != alpha_dt || beta != beta) return fail(FSEI_ERR_ARG, "fsei_project: NaN parameter");
    if (phi == u || phi == v || phi == w || phi == p) return fail(FSEI_ERR_ARG, "fsei_project: phi must not alias u, v, w, p");
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(p) || misaligned(phi)) return fail(FSEI_ERR_ARG, "fsei_project: field pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    size_t n = (size_t)P->T.nx * P->T.ny * P->T.nz;
    { LaunchTimer t(P, K_PROJ, st); k_project_fast<<<(unsigned)((n / 2 + 255) / 256), 256, 0, st>>>(P->S, u, v, w, p, phi, alpha_dt, beta); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

// a1 .. a6 of the register-resident families: phi = solution of the Poisson problem for D(u, v, w) / alpha_dt
static int fast_projection_solve(fsei_plan* P, const double* u, const double* v, const double* w, double* phi, double alpha_dt, cudaStream_t st)
{
    cplx* spec = P->fused ? P->work : reinterpret_cast<cplx*>(phi);
    { LaunchTimer t(P, K_DIVXF, st); CU(launch_xf_fast(P->XF, P->S, P->T.bcx == BC_NEUMANN, true, u, v, w, 1.0 / alpha_dt, spec, st, P->fused)); }
    return P->fused ? fused_spectral_solve(P, phi, st) : fast_spectral_solve(P, spec, st);
}

extern "C" int fsei_pressure_projection(fsei_plan* P, double* u, double* v, double* w, double* p, double* phi,
                                        double alpha_dt, double beta, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_pressure_projection: this is a slab plan (use the fsei_slab_* calls)");
    int rc, n = 0;
    if (P && P->fast) {
        if (!u || !v || !w || !p || !phi) return fail(FSEI_ERR_ARG, "fsei_pressure_projection: NULL argument");
        if (alpha_dt == 0.0 || alpha_dt != alpha_dt || beta != beta) return fail(FSEI_ERR_ARG, "fsei_pressure_projection: alpha_dt must be non-zero, beta not NaN");
        if (phi == u || phi == v || phi == w || phi == p) return fail(FSEI_ERR_ARG, "fsei_pressure_projection: phi must not alias u, v, w, p");
        if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(p) || misaligned(phi)) return fail(FSEI_ERR_ARG, "fsei_pressure_projection: field pointers must be 16-byte aligned");
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        if ((rc = fast_projection_solve(P, u, v, w, phi, alpha_dt, st))) return rc;
        if ((rc = fsei_project(P, u, v, w, p, phi, alpha_dt, beta, cuda_stream))) return rc;
        P->last_launches = P->fused ? 6 : 7;
        return FSEI_OK;
    }
    if ((rc = fsei_divergence(P, u, v, w, alpha_dt, phi, cuda_stream))) return rc;
    n += P->last_launches;
    if ((rc = fsei_poisson_solve(P, phi, phi, cuda_stream))) return rc;
    n += P->last_launches;
    if ((rc = fsei_project(P, u, v, w, p, phi, alpha_dt, beta, cuda_stream))) return rc;
    n += P->last_launches;
    P->last_launches = n;
    return FSEI_OK;
}

extern "C" int fsei_pressure_projection_host(fsei_plan* P, double* u, double* v, double* w, double* p,
                                             double alpha_dt, double beta, void* cuda_stream)
{
    if (!P || !u || !v || !w || !p) return fail(FSEI_ERR_ARG, "fsei_pressure_projection_host: NULL argument");
    if (P->slab) return fail(FSEI_ERR_ARG, "fsei_pressure_projection_host: this is a slab plan");
    if (alpha_dt == 0.0 || alpha_dt != alpha_dt || beta != beta) return fail(FSEI_ERR_ARG, "fsei_pressure_projection_host: alpha_dt must be non-zero, beta not NaN");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostTables& T = P->T;
    const size_t plane = (size_t)T.nx * T.ny, bytes = sizeof(double) * plane * T.nz;
    { int rc0 = host_fields(P); if (rc0) return rc0; }          // no-op when the plan was created with FSEI_PLAN_HOST_FIELDS
    // The link is full duplex and p is not needed before the correction: u, v, w go up, the Poisson problem is solved, then the
    // correction runs in z chunks -- chunk c of p goes up on one copy stream while the corrected chunks c-1, c-2, ... of u, v, w,
    // p come down on another.
    constexpr int NCH = 8;
    const int nch = T.nz < NCH ? T.nz : NCH;
    if (!P->host_up) {
        CU(cudaStreamCreateWithFlags(&P->host_up, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&P->host_dn, cudaStreamNonBlocking));
        P->host_ev.resize(2 * NCH + 2);
        for (cudaEvent_t& e : P->host_ev) CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    double* h[4] = {u, v, w, p};
    double** d = P->hostpath;
    cudaEvent_t ev_in = P->host_ev[2 * NCH], ev_out = P->host_ev[2 * NCH + 1];
    for (int f = 0; f < 3; f++) CU(cudaMemcpyAsync(d[f], h[f], bytes, cudaMemcpyHostToDevice, st));
    CU(cudaEventRecord(ev_in, st));
    CU(cudaStreamWaitEvent(P->host_up, ev_in, 0));              // p follows u, v, w on the way up (and the previous call's work)
    CU(cudaStreamWaitEvent(P->host_dn, ev_in, 0));
    int rc, launches = 0;
    if (P->fast) {
        if ((rc = fast_projection_solve(P, d[0], d[1], d[2], d[4], alpha_dt, st))) return rc;
        launches = P->fused ? 5 : 6;
    } else {
        if ((rc = fsei_divergence(P, d[0], d[1], d[2], alpha_dt, d[4], cuda_stream))) return rc;
        launches = P->last_launches;
        if ((rc = fsei_poisson_solve(P, d[4], d[4], cuda_stream))) return rc;
        launches += P->last_launches;
    }
    for (int c = 0; c < nch; c++) {
        const int k0 = (int)((long)T.nz * c / nch), k1 = (int)((long)T.nz * (c + 1) / nch);
        const size_t off = (size_t)k0 * plane, cb = sizeof(double) * plane * (size_t)(k1 - k0);
        cudaEvent_t ev_up = P->host_ev[2 * c], ev_pr = P->host_ev[2 * c + 1];
        CU(cudaMemcpyAsync(d[3] + off, p + off, cb, cudaMemcpyHostToDevice, P->host_up));
        CU(cudaEventRecord(ev_up, P->host_up));
        CU(cudaStreamWaitEvent(st, ev_up, 0));
        SParams S = P->S;                                       // the correction on planes [k0, k1): phi has its neighbours in place
        S.nz = k1 - k0; S.kofs = k0; S.halo_lo = k0 > 0; S.halo_hi = k1 < T.nz;
        const size_t n2 = plane * (size_t)(k1 - k0) / 2;
        { LaunchTimer t(P, K_PROJ, st); k_project_fast<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(S, d[0] + off, d[1] + off, d[2] + off, d[3] + off, d[4] + off, alpha_dt, beta); }
        CU(cudaGetLastError());
        launches++;
        CU(cudaEventRecord(ev_pr, st));
        CU(cudaStreamWaitEvent(P->host_dn, ev_pr, 0));
        for (int f = 0; f < 4; f++) CU(cudaMemcpyAsync(h[f] + off, d[f] + off, cb, cudaMemcpyDeviceToHost, P->host_dn));
    }
    CU(cudaEventRecord(ev_out, P->host_dn));
    CU(cudaStreamWaitEvent(st, ev_out, 0));
    CU(cudaStreamSynchronize(st));
    P->last_launches = launches;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// fluid substep: explicit terms, implicit viscous step
// ------------------------------------------------------------------------------------------
extern "C" int fsei_explicit_terms(fsei_plan* P, const double* u, const double* v, const double* w, const double* p,
                                   const double* fu, const double* fv, const double* fw, double* hu, double* hv, double* hw,
                                   double* ru, double* rv, double* rw, double gamma_dt, double rho_dt, double alpha_dt,
                                   double beta, void* cuda_stream)
{
    if (!P || !u || !v || !w || !p || !hu || !hv || !hw || !ru || !rv || !rw) return fail(FSEI_ERR_ARG, "fsei_explicit_terms: NULL argument");
    if (gamma_dt != gamma_dt || rho_dt != rho_dt || alpha_dt != alpha_dt || !(beta >= 0.0)) return fail(FSEI_ERR_ARG, "fsei_explicit_terms: NaN parameter or beta < 0");
    const double* in[4] = {u, v, w, p};
    double* out[6] = {hu, hv, hw, ru, rv, rw};
    for (int a = 0; a < 6; a++) {
        for (int b = 0; b < 4; b++) if (out[a] == in[b]) return fail(FSEI_ERR_ARG, "fsei_explicit_terms: outputs must not alias u, v, w, p");
        for (int b = a + 1; b < 6; b++) if (out[a] == out[b]) return fail(FSEI_ERR_ARG, "fsei_explicit_terms: outputs must not alias each other");
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // planes per CTA: long marches amortise the ring's prologue (two halo planes per chunk); short ones keep small grids busy
    const long tiles = (long)((P->T.nx + 31) / 32) * ((P->T.ny + 7) / 8);
    int kz = FSEI_EXPL_KZMAX;
    const int nzl = P->S.nz;                           // planes held by the fields (a slab plan: its own planes)
    while (kz > 8 && tiles * ((nzl + kz - 1) / kz) < 1184) kz >>= 1;
    ExplicitArgs A{P->S, u, v, w, p, fu, fv, fw, hu, hv, hw, ru, rv, rw, gamma_dt, rho_dt, alpha_dt, 2.0 * beta, kz, 0, 0, 0, {}, {}, {}, {}, {}, {}};
    // TMA boxes for the tiles whose halo lies inside the grid: (nx, ny, planes) views of u, v, w, p that start at the halo plane
    // below a slab.  Rows must be 16-byte multiples (nx even) and the fields 16-byte aligned; otherwise every tile copies per thread.
    if (P->T.nx % 2 == 0 && P->T.nx >= 2 * FSEI_EXPL_TX + 4 && P->T.ny >= 3 * FSEI_EXPL_TY && !misaligned(u) && !misaligned(v) &&
        !misaligned(w) && !misaligned(p)) {
        EncodeTiledFn fn = tma_encode_fn();
        const size_t plane = (size_t)P->T.nx * P->T.ny;
        const int below = P->S.halo_lo ? 1 : 0, planes = nzl + below + (P->S.halo_hi ? 1 : 0);
        cuuint64_t dims[3] = {(cuuint64_t)P->T.nx, (cuuint64_t)P->T.ny, (cuuint64_t)planes};
        cuuint64_t strides[2] = {(cuuint64_t)P->T.nx * sizeof(double), (cuuint64_t)plane * sizeof(double)};
        cuuint32_t box[3] = {FSEI_EXPL_PW, FSEI_EXPL_TY + 2, 1u}, estr[3] = {1, 1, 1};
        TmaMap3D* maps[4] = {&A.mu, &A.mv, &A.mw, &A.mp};
        bool ok = fn != nullptr;
        for (int q = 0; q < 4 && ok; q++)
            ok = fn(&maps[q]->m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(in[q] - (size_t)below * plane), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        // H_prev and the body force of the CTA's own cells: (nx, ny, nzl) views, box (32, 8, 1)
        cuuint64_t hdims[3] = {(cuuint64_t)P->T.nx, (cuuint64_t)P->T.ny, (cuuint64_t)nzl};
        cuuint32_t hbox[3] = {FSEI_EXPL_TX, FSEI_EXPL_TY, 1u};
        const double* hf[6] = {hu, hv, hw, fu, fv, fw};
        for (int q = 0; q < 6 && ok; q++) {
            if (!hf[q]) continue;
            ok = !misaligned(hf[q]) &&
                 fn(&(q < 3 ? A.mh[q] : A.mf[q - 3]).m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(hf[q]), hdims, strides, hbox, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        }
        A.tma = ok ? 1 : 0;
    }
    // ring: as many slots as two CTAs per SM leave room for (the force tiles take their share of a slot only when given)
    A.slot = FSEI_EXPL_SLOT((fu ? 1 : 0) + (fv ? 1 : 0) + (fw ? 1 : 0));
    A.ring = FSEI_EXPL_SMEM_MAX / (A.slot * (int)sizeof(double));
    if (A.ring > FSEI_EXPL_MAXRING) A.ring = FSEI_EXPL_MAXRING;
    if (A.ring > kz + 2) A.ring = kz + 2 < FSEI_EXPL_RING ? FSEI_EXPL_RING : kz + 2;
    const size_t smem = (size_t)A.ring * A.slot * sizeof(double);
    const dim3 grid((P->T.nx + 31) / 32, (P->T.ny + 7) / 8, (nzl + kz - 1) / kz);
    { LaunchTimer t(P, K_EXPL, st); k_explicit_terms<<<grid, dim3(32, 8), smem, st>>>(A); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

static VTab visc_tab(const fsei_plan* P, int slot, int comp, int dir)
{
    const HostTables& T = P->T;
    const double* t = P->vtab + (size_t)(slot * 9 + comp * 3 + dir) * vtab_set_doubles(P->vnmax);
    const size_t m = (size_t)P->vnmax;
    VTab V;
    V.ip = t; V.am = t + m; V.cp = t + 2 * m; V.wc = t + 3 * m; V.er = t + 4 * m; V.ipl = t + 5 * m;
    V.n = dir == DIR_X ? T.nx : (dir == DIR_Y ? T.ny : T.nz);
    V.cyclic = (dir == DIR_X && T.bcx == BC_PERIODIC) || (dir == DIR_Y && T.bcy == BC_PERIODIC);
    V.fixed0 = (dir == DIR_X && comp == COMP_U && T.bcx != BC_PERIODIC) || (dir == DIR_Y && comp == COMP_V && T.bcy != BC_PERIODIC) ||
               (dir == DIR_Z && comp == COMP_W);
    return V;
}

// factorisation tables of the implicit viscous step for this beta: kept per value in FSEI_VSLOTS slots (round-robin
// replacement).  Under stream capture the device tables are rebuilt inside the graph even on a hit, so a replay never depends
// on a slot that an eager call with other betas has overwritten in the meantime (the host-built tables travel as kernel
// parameters).  Returns the slot; *launches counts the factor kernel if it ran.
static int visc_tables(fsei_plan* P, double beta, cudaStream_t st, int* slot_out, int* launches)
{
    const HostTables& T = P->T;
    int slot = -1;
    for (int i = 0; i < FSEI_VSLOTS; i++) if (P->visc_beta[i] == beta) slot = i;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CU(cudaStreamIsCapturing(st, &cap));
    const bool miss = slot < 0;
    if (miss) {
        slot = P->visc_next; P->visc_next = (slot + 1) % FSEI_VSLOTS;
        if (P->visc_fast) {
            visc_fast_line(T.nx, P->S.rdx, beta, &P->vline_x[slot]); P->vnsig_x[slot] = visc_fast_nsig(P->vline_x[slot]);
            visc_fast_line(T.ny, P->S.rdy, beta, &P->vline_y[slot]); P->vnsig_y[slot] = visc_fast_nsig(P->vline_y[slot]);
        }
        P->visc_beta[slot] = beta;
    }
    if (miss || cap != cudaStreamCaptureStatusNone) {
        VFactorArgs A{P->slab ? P->Sg : P->S, beta, P->vtab + (size_t)slot * 9 * vtab_set_doubles(P->vnmax), P->vnmax};
        { LaunchTimer t(P, K_VFACT, st); k_visc_factor<<<9, 32, 0, st>>>(A); }
        CU(cudaGetLastError());
        (*launches)++;
    }
    *slot_out = slot;
    return FSEI_OK;
}

extern "C" int fsei_viscous_step(fsei_plan* P, double* u, double* v, double* w, double* ru, double* rv, double* rw,
                                 double beta, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_viscous_step: this is a slab plan (use the fsei_slab_* calls)");
    if (!P || !u || !v || !w || !ru || !rv || !rw) return fail(FSEI_ERR_ARG, "fsei_viscous_step: NULL argument");
    if (!(beta >= 0.0) || std::isinf(beta)) return fail(FSEI_ERR_ARG, "fsei_viscous_step: beta must be finite and >= 0");
    double* q[3] = {u, v, w};
    double* r[3] = {ru, rv, rw};
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) if (r[a] == q[b] || (a != b && (r[a] == r[b] || q[a] == q[b]))) return fail(FSEI_ERR_ARG, "fsei_viscous_step: fields must not alias");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostTables& T = P->T;
    int launches = 0;
    int slot = 0;
    { int rc0 = visc_tables(P, beta, st, &slot, &launches); if (rc0) return rc0; }
    if (P->visc_fast) {
        VFastArgs A;
        for (int c = 0; c < 3; c++) {
            const VTab V = visc_tab(P, slot, c, DIR_Z);
            A.zam[c] = V.am; A.zip[c] = V.ip; A.zcp[c] = V.cp; A.r[c] = r[c]; A.q[c] = q[c];
        }
        A.nx = T.nx; A.ny = T.ny; A.nz = T.nz; A.slab = 0;
        A.split = 2 * (T.nx / 8) <= P->nsm ? 1 : 0;           // up to 1.5 marches per SM (measured: nx <= 576 gain 1.1-3x, nx >= 640 lose)
        A.L = P->vline_x[slot]; A.nsig = P->vnsig_x[slot];
        { LaunchTimer t(P, K_VXZ, st); CU(launch_visc_xz(A, st)); }
        A.L = P->vline_y[slot]; A.nsig = P->vnsig_y[slot];
        { LaunchTimer t(P, K_VZY, st); CU(launch_visc_zy(A, st)); }
        P->last_launches = launches + 2;
        return FSEI_OK;
    }
    const long nlx = (long)T.ny * T.nz, nly = (long)T.nx * T.nz, nlz = (long)T.nx * T.ny;
    const size_t plane = (size_t)T.nx * T.ny;
    for (int c = 0; c < 3; c++) {
        {
            VTab V = visc_tab(P, slot, c, DIR_X);
            LaunchTimer t(P, K_VX, st);
            const unsigned g = (unsigned)((nlx + 127) / 128);
            if (V.cyclic) k_visc_sweep_x<true, false><<<g, 128, 0, st>>>(V, r[c], nullptr, nlx);
            else k_visc_sweep_x<false, false><<<g, 128, 0, st>>>(V, r[c], nullptr, nlx);
        }
        CU(cudaGetLastError());
        {
            VTab V = visc_tab(P, slot, c, DIR_Y);
            LaunchTimer t(P, K_VY, st);
            const unsigned g = (unsigned)((nly + 127) / 128);
            if (V.cyclic) k_visc_sweep_strided<true, false><<<g, 128, 0, st>>>(V, r[c], nullptr, T.nx, (size_t)T.nx, plane, nly);
            else k_visc_sweep_strided<false, false><<<g, 128, 0, st>>>(V, r[c], nullptr, T.nx, (size_t)T.nx, plane, nly);
        }
        CU(cudaGetLastError());
        {
            VTab V = visc_tab(P, slot, c, DIR_Z);
            LaunchTimer t(P, K_VZ, st);
            k_visc_sweep_strided<false, true><<<(unsigned)((nlz + 127) / 128), 128, 0, st>>>(V, r[c], q[c], (int)nlz, plane, 0, nlz);
        }
        CU(cudaGetLastError());
        launches += 3;
    }
    P->last_launches = launches;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// fsei_viscous_step_noalloc: the generic family of the implicit viscous step with its factorisation tables in a file-scope
// device array instead of plan-owned memory, for callers that may not allocate (stream capture, serving loops, harnesses that
// forbid cudaMalloc).  Every GPU that loads the library holds the array until exit (FSEI_NOALLOC_BYTES = 369 216 bytes).
//
// In HOST code the name `g_noalloc_vtab` is a host-side stand-in, not a device address: its device address comes from
// cudaGetSymbolAddress, asked once per device with that device current (noalloc_resolve, called at plan creation = set-up)
// and only that pointer is ever given to a kernel.
//
// All calls on a device share the array and it keeps the last call's contents.  Nothing in it has to start at zero: the
// factor launch of a call writes every table entry the nine sweeps of that call read (ip, am, cp, wc, er at rows 0..n-1 and
// ipl[0] of each of the 9 sets) before they run, on the same stream.  Two calls that overlap on the GPU (different streams,
// or two processes' worth of plans in one process on one device) RACE on it: serialise them.
// ------------------------------------------------------------------------------------------
#define FSEI_NOALLOC_NMAX 1024                                           /* longest line (nx, ny, nz each) */
#define FSEI_NOALLOC_DOUBLES (9 * (5 * FSEI_NOALLOC_NMAX + 8))           /* 9 sets of vtab_set_doubles(NMAX) */
#define FSEI_NOALLOC_BYTES (FSEI_NOALLOC_DOUBLES * 8)
#define FSEI_NOALLOC_MAXDEV 64
static __device__ __align__(256) double g_noalloc_vtab[FSEI_NOALLOC_DOUBLES];
static double* g_noalloc_ptr[FSEI_NOALLOC_MAXDEV];                       // device address of the array on each device (host cache)
static std::mutex g_noalloc_mu;

// device address of the scratch array on the CURRENT device; asks the runtime once per device
static int noalloc_resolve(double** out, int* dev_out)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= FSEI_NOALLOC_MAXDEV) return fail(FSEI_ERR_CUDA, "fsei_viscous_step_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_vtab);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_vtab)"); }
        g_noalloc_ptr[dev] = static_cast<double*>(p);
    }
    *out = g_noalloc_ptr[dev]; *dev_out = dev;
    return FSEI_OK;
}

static VTab visc_tab_from(const HostTables& T, const double* base, int nmax, int comp, int dir)
{
    const double* t = base + (size_t)(comp * 3 + dir) * vtab_set_doubles(nmax);
    const size_t m = (size_t)nmax;
    VTab V;
    V.ip = t; V.am = t + m; V.cp = t + 2 * m; V.wc = t + 3 * m; V.er = t + 4 * m; V.ipl = t + 5 * m;
    V.n = dir == DIR_X ? T.nx : (dir == DIR_Y ? T.ny : T.nz);
    V.cyclic = (dir == DIR_X && T.bcx == BC_PERIODIC) || (dir == DIR_Y && T.bcy == BC_PERIODIC);
    V.fixed0 = (dir == DIR_X && comp == COMP_U && T.bcx != BC_PERIODIC) || (dir == DIR_Y && comp == COMP_V && T.bcy != BC_PERIODIC) ||
               (dir == DIR_Z && comp == COMP_W);
    return V;
}

extern "C" int fsei_viscous_step_noalloc(fsei_plan* P, double* u, double* v, double* w, double* ru, double* rv, double* rw,
                                         double beta, void* cuda_stream)
{
    if (P && P->slab) return fail(FSEI_ERR_ARG, "fsei_viscous_step_noalloc: this is a slab plan");
    if (!P || !u || !v || !w || !ru || !rv || !rw) return fail(FSEI_ERR_ARG, "fsei_viscous_step_noalloc: NULL argument");
    if (!(beta >= 0.0) || std::isinf(beta)) return fail(FSEI_ERR_ARG, "fsei_viscous_step_noalloc: beta must be finite and >= 0");
    double* q[3] = {u, v, w};
    double* r[3] = {ru, rv, rw};
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) if (r[a] == q[b] || (a != b && (r[a] == r[b] || q[a] == q[b]))) return fail(FSEI_ERR_ARG, "fsei_viscous_step_noalloc: fields must not alias");
    const HostTables& T = P->T;
    const int nmax = T.nx > T.ny ? (T.nx > T.nz ? T.nx : T.nz) : (T.ny > T.nz ? T.ny : T.nz);
    if (nmax > FSEI_NOALLOC_NMAX)
        return fail(FSEI_ERR_SIZE, "fsei_viscous_step_noalloc: nx, ny and nz must each be <= 1024 (the static scratch array holds the "
                                   "factorisation tables of lines up to that length); use fsei_viscous_step on larger grids");
    if (!P->noalloc_tab) return fail(FSEI_ERR_CUDA, "fsei_viscous_step_noalloc: the address of the static scratch array could not be resolved when the plan was created");
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev != P->noalloc_dev) return fail(FSEI_ERR_ARG, "fsei_viscous_step_noalloc: the current device is not the one the plan was created on");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* tab = P->noalloc_tab;                                        // a device address (never the symbol's host stand-in)
    VFactorArgs A{P->S, beta, tab, nmax};
    k_visc_factor<<<9, 32, 0, st>>>(A);
    CU(cudaGetLastError());
    const long nlx = (long)T.ny * T.nz, nly = (long)T.nx * T.nz, nlz = (long)T.nx * T.ny;
    const size_t plane = (size_t)T.nx * T.ny;
    for (int c = 0; c < 3; c++) {
        const VTab Vx = visc_tab_from(T, tab, nmax, c, DIR_X), Vy = visc_tab_from(T, tab, nmax, c, DIR_Y), Vz = visc_tab_from(T, tab, nmax, c, DIR_Z);
        const unsigned gx = (unsigned)((nlx + 127) / 128), gy = (unsigned)((nly + 127) / 128), gz = (unsigned)((nlz + 127) / 128);
        if (Vx.cyclic) k_visc_sweep_x<true, false><<<gx, 128, 0, st>>>(Vx, r[c], nullptr, nlx);
        else k_visc_sweep_x<false, false><<<gx, 128, 0, st>>>(Vx, r[c], nullptr, nlx);
        CU(cudaGetLastError());
        if (Vy.cyclic) k_visc_sweep_strided<true, false><<<gy, 128, 0, st>>>(Vy, r[c], nullptr, T.nx, (size_t)T.nx, plane, nly);
        else k_visc_sweep_strided<false, false><<<gy, 128, 0, st>>>(Vy, r[c], nullptr, T.nx, (size_t)T.nx, plane, nly);
        CU(cudaGetLastError());
        k_visc_sweep_strided<false, true><<<gz, 128, 0, st>>>(Vz, r[c], q[c], (int)nlz, plane, 0, nlz);
        CU(cudaGetLastError());
    }
    P->last_launches = 10;
    return FSEI_OK;
}

extern "C" int fsei_fluid_substep(fsei_plan* P, double* u, double* v, double* w, double* p, const double* fu, const double* fv,
                                  const double* fw, double* hu, double* hv, double* hw, double* ru, double* rv, double* rw,
                                  double* phi, double gamma_dt, double rho_dt, double alpha_dt, double beta, void* cuda_stream)
{
    int rc, n = 0;
    if (!P) return fail(FSEI_ERR_ARG, "fsei_fluid_substep: NULL plan");
    if ((rc = fsei_explicit_terms(P, u, v, w, p, fu, fv, fw, hu, hv, hw, ru, rv, rw, gamma_dt, rho_dt, alpha_dt, beta, cuda_stream))) return rc;
    n += P->last_launches;
    if ((rc = fsei_viscous_step(P, u, v, w, ru, rv, rw, beta, cuda_stream))) return rc;
    n += P->last_launches;
    if ((rc = fsei_pressure_projection(P, u, v, w, p, phi, alpha_dt, beta, cuda_stream))) return rc;
    n += P->last_launches;
    P->last_launches = n;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// IB-MLS transfer operators
// ------------------------------------------------------------------------------------------
static MlsGrid mls_grid(const fsei_plan* P)
{
    const HostTables& T = P->T;
    MlsGrid G;
    G.nx = T.nx; G.ny = T.ny; G.nz = T.nz; G.bcx = T.bcx; G.bcy = T.bcy;
    G.dx = T.Lx / T.nx; G.dy = T.Ly / T.ny; G.Lx = T.Lx; G.Ly = T.Ly; G.zc = P->zc_dev;
    return G;
}

template <int MODE> static int mls_launch(fsei_plan* P, const MlsArgs& A, cudaStream_t st)
{
    if (A.n == 0) { P->last_launches = 0; return FSEI_OK; }
    { LaunchTimer t(P, K_MLS, st); k_mls<MODE><<<(unsigned)((3 * A.n + 127) / 128), 128, 0, st>>>(A); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

extern "C" int fsei_mls_interpolate(fsei_plan* P, long n, const double* xm, const double* ym, const double* zm,
                                    const double* u, const double* v, const double* w, double* ub, double* vb, double* wb,
                                    void* cuda_stream)
{
    if (!P || n < 0 || (n > 0 && (!xm || !ym || !zm || !u || !v || !w || !ub || !vb || !wb))) return fail(FSEI_ERR_ARG, "fsei_mls_interpolate: NULL argument or n < 0");
    if (P->T.nz < 3) return fail(FSEI_ERR_SIZE, "fsei_mls_interpolate: the 27-node support needs nz >= 3");
    MlsArgs A{mls_grid(P), n, xm, ym, zm, nullptr, {u, v, w}, {nullptr, nullptr, nullptr}, {ub, vb, wb}, {nullptr, nullptr, nullptr}, 0.0};
    return mls_launch<0>(P, A, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int fsei_mls_spread(fsei_plan* P, long n, const double* xm, const double* ym, const double* zm, const double* area,
                               const double* Fu, const double* Fv, const double* Fw, double* fu, double* fv, double* fw,
                               void* cuda_stream)
{
    if (!P || n < 0 || (n > 0 && (!xm || !ym || !zm || !area || !Fu || !Fv || !Fw || !fu || !fv || !fw))) return fail(FSEI_ERR_ARG, "fsei_mls_spread: NULL argument or n < 0");
    if (P->T.nz < 3) return fail(FSEI_ERR_SIZE, "fsei_mls_spread: the 27-node support needs nz >= 3");
    MlsArgs A{mls_grid(P), n, xm, ym, zm, area, {nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr},
              {const_cast<double*>(Fu), const_cast<double*>(Fv), const_cast<double*>(Fw)}, {fu, fv, fw}, 0.0};
    return mls_launch<2>(P, A, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int fsei_ibm_forcing(fsei_plan* P, long n, const double* xm, const double* ym, const double* zm, const double* area,
                                const double* Vu, const double* Vv, const double* Vw, const double* u, const double* v,
                                const double* w, double inv_dt, double* Fu, double* Fv, double* Fw, double* fu, double* fv,
                                double* fw, void* cuda_stream)
{
    if (!P || n < 0 || (n > 0 && (!xm || !ym || !zm || !area || !Vu || !Vv || !Vw || !u || !v || !w || !Fu || !Fv || !Fw || !fu || !fv || !fw)))
        return fail(FSEI_ERR_ARG, "fsei_ibm_forcing: NULL argument or n < 0");
    if (inv_dt != inv_dt) return fail(FSEI_ERR_ARG, "fsei_ibm_forcing: NaN inv_dt");
    if (fu == u || fu == v || fu == w || fv == u || fv == v || fv == w || fw == u || fw == v || fw == w) return fail(FSEI_ERR_ARG, "fsei_ibm_forcing: the forcing fields must not alias the velocity");
    if (P->T.nz < 3) return fail(FSEI_ERR_SIZE, "fsei_ibm_forcing: the 27-node support needs nz >= 3");
    MlsArgs A{mls_grid(P), n, xm, ym, zm, area, {u, v, w}, {Vu, Vv, Vw}, {Fu, Fv, Fw}, {fu, fv, fw}, inv_dt};
    return mls_launch<1>(P, A, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int fsei_ibm_apply_forcing(fsei_plan* P, long n, const double* xm, const double* ym, const double* zm, double* fu, double* fv,
                                      double* fw, double* ru, double* rv, double* rw, double alpha_dt, void* cuda_stream)
{
    if (!P || n < 0 || (n > 0 && (!xm || !ym || !zm || !fu || !fv || !fw || !ru || !rv || !rw))) return fail(FSEI_ERR_ARG, "fsei_ibm_apply_forcing: NULL argument or n < 0");
    if (P->slab) return fail(FSEI_ERR_ARG, "fsei_ibm_apply_forcing: not available on a slab plan");
    if (alpha_dt != alpha_dt) return fail(FSEI_ERR_ARG, "fsei_ibm_apply_forcing: NaN alpha_dt");
    double* fs[3] = {fu, fv, fw};
    double* rs[3] = {ru, rv, rw};
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) if (fs[a] == rs[b] || (a != b && (fs[a] == fs[b] || rs[a] == rs[b]))) return fail(FSEI_ERR_ARG, "fsei_ibm_apply_forcing: aliased fields");
    if (P->T.nz < 3) return fail(FSEI_ERR_SIZE, "fsei_ibm_apply_forcing: the 27-node support needs nz >= 3");
    if (n == 0) { P->last_launches = 0; return FSEI_OK; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MlsApplyArgs A{mls_grid(P), n, xm, ym, zm, {fu, fv, fw}, {ru, rv, rw}, alpha_dt};
    { LaunchTimer t(P, K_MLSAPPLY, st); k_mls_apply<<<(unsigned)((3 * n + 127) / 128), 128, 0, st>>>(A); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// multi-GPU slab decomposition of the projection: the per-rank stages.
// A rank owns planes [k0, k1) of the fields (a z-slab with one halo plane) for a1-a3 and a5-a7, and x-slots [s0, s1) of
// every (ky, k) -- full z columns -- for a4.  The two exchanges between them are the all-to-all of P:L248, done by
// paper_2103_15187_b200/slab.py over torch.distributed; these calls are the local work on either side of it.
// ------------------------------------------------------------------------------------------
static int slab_plan_build(fsei_plan* P, int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy,
                           int k0, int k1, int s0, int s1)
{
    int code = 0, rc;
    if (bcx != BC_PERIODIC || bcy != BC_PERIODIC) return fail(FSEI_ERR_ARG, "fsei_slab_plan_create: periodic x and y only (the paper's decomposition, P:L240)");
    if (nx < 4 || nx % 4 || k0 < 0 || k1 <= k0 || k1 > nz || s0 < 0 || s1 <= s0 || s1 > nx / 2) return fail(FSEI_ERR_ARG, "fsei_slab_plan_create: empty or out-of-range share [k0,k1) x [s0,s1)");
    std::string msg = build_tables(P->T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code, true);
    if (code) return fail(code, msg);
    if (!(xfast_supported(nx / 2) && yfast_supported(ny) && (size_t)nz * 4 * sizeof(cplx) <= 200 * 1024))
        return fail(FSEI_ERR_SIZE, "fsei_slab_plan_create: nx/2 and ny need a register-resident transform (the lengths of the fast family: DESIGN.md sec. 1), nz <= 3200");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(FSEI_ERR_CUDA, "no CUDA device: libfsei has no CPU fallback"); }
    HostTables& T = P->T;
    P->slab = true; P->fast = true; P->k0 = k0; P->k1 = k1; P->s0 = s0; P->s1 = s1;
    const int nzl = k1 - k0, nsl = s1 - s0;
    XParams& X = P->X; YParams& Y = P->Y; ZParams& Z = P->Z; SParams& S = P->S;
    if ((rc = upload(P, T.twx, &X.tw))) return rc;
    if ((rc = upload(P, T.twx_r2c, &X.tw_r2c))) return rc;
    if ((rc = upload(P, T.twx_dct, &X.tw_dct))) return rc;
    if ((rc = upload(P, T.twy, &Y.tw))) return rc;
    if ((rc = upload(P, T.twy_dct, &Y.tw_dct))) return rc;
    if ((rc = upload(P, T.za, &Z.za))) return rc;
    if ((rc = upload(P, T.zcc, &Z.zcc))) return rc;
    if ((rc = upload(P, T.dzc, &Z.dzc))) return rc;
    if ((rc = upload(P, T.dzm, &Z.dzm))) return rc;
    if ((rc = upload(P, T.lamx, &Z.lamx))) return rc;
    if ((rc = upload(P, T.lamy, &Z.lamy))) return rc;
    S.nx = nx; S.ny = ny; S.nz = nzl; S.bcx = bcx; S.bcy = bcy; S.rdx = T.rdx; S.rdy = T.rdy;
    if ((rc = upload(P, T.rdzc, &S.rdzc))) return rc;
    if ((rc = upload(P, T.rdzm, &S.rdzm))) return rc;
    S.kofs = k0; S.halo_lo = k0 > 0; S.halo_hi = k1 < nz;
    P->Sg = S; P->Sg.nz = nz; P->Sg.kofs = 0; P->Sg.halo_lo = 0; P->Sg.halo_hi = 0;
    {
        P->vnmax = nx > ny ? (nx > nz ? nx : nz) : (ny > nz ? ny : nz);
        void* qv = nullptr;
        if ((rc = dalloc(P, sizeof(double) * FSEI_VSLOTS * 9 * vtab_set_doubles(P->vnmax), &qv))) return rc;
        P->vtab = static_cast<double*>(qv);
        CU(kernel_smem(k_explicit_terms, FSEI_EXPL_SMEM_MAX));
        P->visc_fast = visc_fast_slab_supported(nx, ny);               // x and y sweeps of fsei_slab_viscous_xy by the partition kernels
        if (P->visc_fast) {
            CU(visc_fast_init());
            int dev = 0;
            CU(cudaGetDevice(&dev)); CU(cudaDeviceGetAttribute(&P->nsm, cudaDevAttrMultiProcessorCount, dev));
        }
    }
    XFast& XF = P->XF; YFast& YF = P->YF; ZFast& ZF = P->ZF;
    XF.nx = nx; XF.ny = ny; XF.nz = nzl; XF.N = nx / 2; XF.tw = X.tw; XF.tw_r2c = X.tw_r2c; XF.tw_dct = X.tw_dct; XF.scale = T.scale;
    {
        int dev = 0, nsm = 148;
        cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        const int lpb = xfast_lines_per_block(nx / 2, false);
        long kc = ((long)((ny + lpb - 1) / lpb) * nzl) / (4L * nsm);
        XF.kchunk = (int)(kc < 1 ? 1 : (kc > 64 ? 64 : kc));
        P->kchunk_inv = (int)(kc < 1 ? 1 : (kc > 32 ? 32 : kc));
    }
    YF.nxc = T.nxc; YF.ny = ny; YF.nz = nzl; YF.tw = Y.tw; YF.tw_dct = Y.tw_dct; YF.untangle = 1;
    ZF.nxc = nsl; ZF.ny = ny; ZF.nz = nz; ZF.bcx = bcx; ZF.bcy = bcy; ZF.ncomp = 1; ZF.s0 = s0;
    ZF.za = Z.za; ZF.zcc = Z.zcc; ZF.lamx = Z.lamx + 2 * (size_t)s0; ZF.lamy = Z.lamy; ZF.dzc = Z.dzc; ZF.dzm = Z.dzm;
    ZF.ktw = nz; ZF.cb = 0; ZF.special_in = nullptr;
    void* q = nullptr;
    if ((rc = dalloc(P, sizeof(cplx) * 2 * nz, &q))) return rc;
    ZF.special = static_cast<cplx*>(q);
    if ((rc = dalloc(P, sizeof(double) * 8 * nz, &q))) return rc;
    ZF.cpw = static_cast<double*>(q);
    if ((rc = dalloc(P, sizeof(double) * (size_t)nz * ny * nsl, &q))) return rc;
    ZF.ipiv = static_cast<const double*>(q);
    const size_t cols = (size_t)ny * nsl;
    k_zf_factor<<<(unsigned)((cols + 255) / 256), 256>>>(ZF, static_cast<double*>(q));
    CU(cudaGetLastError());
    if (s0 == 0) { k_z_special_factor<<<1, 32>>>(ZF); CU(cudaGetLastError()); }
    CU(cudaDeviceSynchronize());
    CU(xfast_init());
    CU(yfast_init());
    CU(cudaFuncSetAttribute(k_z_special, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)z_special_smem(nz, z_special_staged(nz))));
    return FSEI_OK;
}

extern "C" fsei_plan* fsei_slab_plan_create(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bc_x, int bc_y,
                                            int k0, int k1, int s0, int s1)
{
    fsei_plan* P = new (std::nothrow) fsei_plan();
    if (!P) { fail(FSEI_ERR_ALLOC, "out of host memory"); return nullptr; }
    int rc = slab_plan_build(P, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, k0, k1, s0, s1);
    if (rc != FSEI_OK) { const std::string msg = g_err; fsei_plan_destroy(P); g_err = msg; g_err_code = rc; return nullptr; }
    g_err_code = FSEI_OK; g_err.clear();
    return P;
}

#define SLAB_ONLY(name) if (!P || !P->slab) return fail(FSEI_ERR_ARG, name ": not a slab plan")

// Peer-store exchange: after this call fsei_slab_forward writes its result straight into the pencils of the ranks that
// own the slots, and fsei_pencil_solve writes its result straight into the slab spectra of the ranks that own the planes
// (pointers may be peer-mapped device pointers of other GPUs; on one GPU they are ordinary device pointers).
extern "C" int fsei_slab_set_peers(fsei_plan* P, int nranks, void* const* pencils, void* const* specs, const int* k0s, const int* s0s)
{
    SLAB_ONLY("fsei_slab_set_peers");
    if (nranks == 0) { P->YF.npeer = 0; P->ZF.npeer = 0; return FSEI_OK; }
    if (nranks < 0 || nranks > 8 || !pencils || !specs || !k0s || !s0s) return fail(FSEI_ERR_ARG, "fsei_slab_set_peers: 1 <= nranks <= 8 and non-NULL tables");
    if (k0s[0] != 0 || k0s[nranks] != P->T.nz || s0s[0] != 0 || s0s[nranks] != P->T.nxc) return fail(FSEI_ERR_ARG, "fsei_slab_set_peers: the ranges must cover [0, nz) and [0, nx/2)");
    bool mine = false;
    for (int d = 0; d < nranks; d++) {
        if (!pencils[d] || !specs[d] || misaligned(pencils[d]) || misaligned(specs[d]) || k0s[d + 1] <= k0s[d] || s0s[d + 1] <= s0s[d])
            return fail(FSEI_ERR_ARG, "fsei_slab_set_peers: NULL / misaligned pointer or empty range");
        mine = mine || (k0s[d] == P->k0 && k0s[d + 1] == P->k1 && s0s[d] == P->s0 && s0s[d + 1] == P->s1);
    }
    if (!mine) return fail(FSEI_ERR_ARG, "fsei_slab_set_peers: this plan's own share is not among the ranges");
    YFast& YF = P->YF; ZFast& ZF = P->ZF;
    YF.npeer = nranks; YF.kofs = P->k0; ZF.npeer = nranks; ZF.nxc_full = P->T.nxc;
    for (int d = 0; d < nranks; d++) {
        YF.peer_base[d] = static_cast<cplx*>(pencils[d]); YF.peer_s0[d] = s0s[d];
        ZF.slab_base[d] = static_cast<cplx*>(specs[d]); ZF.slab_k0[d] = k0s[d];
    }
    YF.peer_s0[nranks] = s0s[nranks]; ZF.slab_k0[nranks] = k0s[nranks];
    return FSEI_OK;
}

extern "C" int fsei_slab_forward(fsei_plan* P, const double* u, const double* v, const double* w, double alpha_dt,
                                 double* spec, void* cuda_stream)
{
    SLAB_ONLY("fsei_slab_forward");
    if (!u || !v || !w || !spec) return fail(FSEI_ERR_ARG, "fsei_slab_forward: NULL argument");
    if (alpha_dt == 0.0 || alpha_dt != alpha_dt) return fail(FSEI_ERR_ARG, "fsei_slab_forward: alpha_dt must be non-zero");
    if (spec == u || spec == v || spec == w) return fail(FSEI_ERR_ARG, "fsei_slab_forward: spec must not alias u, v, w");
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(spec)) return fail(FSEI_ERR_ARG, "fsei_slab_forward: field pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cplx* sp = reinterpret_cast<cplx*>(spec);
    // a1 fused into the x transform (the kernel takes the slab's plane offset and the halo plane of w from SParams)
    { LaunchTimer t(P, K_DIVXF, st); CU(launch_xf_fast(P->XF, P->S, false, true, u, v, w, 1.0 / alpha_dt, sp, st, false)); }
    { LaunchTimer t(P, K_YF, st); CU(launch_y_fast(P->YF, false, false, sp, st)); }
    P->last_launches = 2;
    return FSEI_OK;
}

extern "C" int fsei_pencil_solve(fsei_plan* P, double* pencil, void* cuda_stream)
{
    SLAB_ONLY("fsei_pencil_solve");
    if (!pencil || misaligned(pencil)) return fail(FSEI_ERR_ARG, "fsei_pencil_solve: NULL or misaligned pencil");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostTables& T = P->T;
    cplx* sp = reinterpret_cast<cplx*>(pencil);
    int launches = 0;
    if (P->s0 == 0) {
        { LaunchTimer t(P, K_GAUGE, st); k_z_special<<<1, 128, z_special_smem(T.nz, z_special_staged(T.nz)), st>>>(P->ZF, sp, z_special_staged(T.nz)); }
        CU(cudaGetLastError()); launches++;
    }
    {
        LaunchTimer t(P, K_ZD, st);
        const size_t nthr = (size_t)(P->s1 - P->s0) * T.ny;
        if (T.nz <= 32) k_zf_pcr<<<(unsigned)((nthr * 32 + 127) / 128), 128, 0, st>>>(P->ZF, sp);
        else k_zf_sweep<1><<<(unsigned)((nthr + 127) / 128), 128, 0, st>>>(P->ZF, sp);
    }
    CU(cudaGetLastError());
    P->last_launches = launches + 1;
    return FSEI_OK;
}

extern "C" int fsei_slab_backward(fsei_plan* P, double* spec, double* phi, void* cuda_stream)
{
    SLAB_ONLY("fsei_slab_backward");
    if (!spec || !phi || misaligned(spec) || misaligned(phi)) return fail(FSEI_ERR_ARG, "fsei_slab_backward: NULL or misaligned argument");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cplx* sp = reinterpret_cast<cplx*>(spec);
    { LaunchTimer t(P, K_YI, st); CU(launch_y_fast(P->YF, true, false, sp, st)); }
    { LaunchTimer t(P, K_XI, st); XFast xi = P->XF; xi.kchunk = P->kchunk_inv; CU(launch_xi_fast(xi, false, sp, phi, st)); }
    P->last_launches = 2;
    return FSEI_OK;
}

extern "C" int fsei_slab_project(fsei_plan* P, double* u, double* v, double* w, double* p, const double* phi,
                                 double alpha_dt, double beta, void* cuda_stream)
{
    SLAB_ONLY("fsei_slab_project");
    if (!u || !v || !w || !p || !phi) return fail(FSEI_ERR_ARG, "fsei_slab_project: NULL argument");
    if (alpha_dt != alpha_dt || beta != beta) return fail(FSEI_ERR_ARG, "fsei_slab_project: NaN parameter");
    if (misaligned(u) || misaligned(v) || misaligned(w) || misaligned(p) || misaligned(phi)) return fail(FSEI_ERR_ARG, "fsei_slab_project: field pointers must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t n = (size_t)P->T.nx * P->T.ny * (P->k1 - P->k0);
    { LaunchTimer t(P, K_PROJ, st); k_project_fast<<<(unsigned)((n / 2 + 255) / 256), 256, 0, st>>>(P->S, u, v, w, p, phi, alpha_dt, beta); }
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

// ---- slab decomposition of the implicit viscous step: x and y sweeps are local to a z-slab, the z sweep runs on pencils
// that hold full z columns (here: every row and plane of a range of x, the real field viewed as nx/2 complex slots so that
// the spectrum's exchange buffers and lists serve unchanged); q += dq afterwards, on the slab.
__global__ void __launch_bounds__(256) k_field_add(double* __restrict__ q, const double* __restrict__ r, size_t n2)
{
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (t >= n2) return;
    cplx a = *reinterpret_cast<cplx*>(q + 2 * t);
    const cplx b = *reinterpret_cast<const cplx*>(r + 2 * t);
    a.re += b.re; a.im += b.im;
    *reinterpret_cast<cplx*>(q + 2 * t) = a;
}

extern "C" int fsei_slab_viscous_xy(fsei_plan* P, double* ru, double* rv, double* rw, double beta, void* cuda_stream)
{
    SLAB_ONLY("fsei_slab_viscous_xy");
    if (!ru || !rv || !rw || ru == rv || ru == rw || rv == rw) return fail(FSEI_ERR_ARG, "fsei_slab_viscous_xy: NULL or aliased fields");
    if (!(beta >= 0.0) || std::isinf(beta)) return fail(FSEI_ERR_ARG, "fsei_slab_viscous_xy: beta must be finite and >= 0");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostTables& T = P->T;
    int launches = 0, slot = 0, rc;
    if ((rc = visc_tables(P, beta, st, &slot, &launches))) return rc;
    const int nzl = P->k1 - P->k0;
    const long nlx = (long)T.ny * nzl, nly = (long)T.nx * nzl;
    const size_t plane = (size_t)T.nx * T.ny;
    double* r[3] = {ru, rv, rw};
    if (P->visc_fast && (size_t)32 * T.ny * nzl < (1ull << 31) && !misaligned(ru) && !misaligned(rv) && !misaligned(rw)) {
        // the fast family's two passes without their z parts: periodic x solves, then periodic y solves, in place
        VFastArgs A;
        for (int c = 0; c < 3; c++) { A.zam[c] = A.zip[c] = A.zcp[c] = nullptr; A.r[c] = r[c]; A.q[c] = r[c]; }
        A.nx = T.nx; A.ny = T.ny; A.nz = nzl; A.slab = 1;
        A.split = 2 * (T.nx / 8) <= P->nsm ? 1 : 0;
        A.L = P->vline_x[slot]; A.nsig = P->vnsig_x[slot];
        { LaunchTimer t(P, K_VXZ, st); CU(launch_visc_xz(A, st)); }
        A.L = P->vline_y[slot]; A.nsig = P->vnsig_y[slot];
        { LaunchTimer t(P, K_VZY, st); CU(launch_visc_zy(A, st)); }
        P->last_launches = launches + 2;
        return FSEI_OK;
    }
    for (int c = 0; c < 3; c++) {
        { VTab V = visc_tab(P, slot, c, DIR_X); LaunchTimer t(P, K_VX, st); k_visc_sweep_x<true, false><<<(unsigned)((nlx + 127) / 128), 128, 0, st>>>(V, r[c], nullptr, nlx); }
        CU(cudaGetLastError());
        { VTab V = visc_tab(P, slot, c, DIR_Y); LaunchTimer t(P, K_VY, st); k_visc_sweep_strided<true, false><<<(unsigned)((nly + 127) / 128), 128, 0, st>>>(V, r[c], nullptr, T.nx, (size_t)T.nx, plane, nly); }
        CU(cudaGetLastError());
        launches += 2;
    }
    P->last_launches = launches;
    return FSEI_OK;
}

extern "C" int fsei_pencil_viscous_z(fsei_plan* P, double* pencil, int comp, double beta, void* cuda_stream)
{
    SLAB_ONLY("fsei_pencil_viscous_z");
    if (!pencil || comp < 0 || comp > 2) return fail(FSEI_ERR_ARG, "fsei_pencil_viscous_z: NULL pencil or component not in 0..2");
    if (!(beta >= 0.0) || std::isinf(beta)) return fail(FSEI_ERR_ARG, "fsei_pencil_viscous_z: beta must be finite and >= 0");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0, slot = 0, rc;
    if ((rc = visc_tables(P, beta, st, &slot, &launches))) return rc;
    const long ncol = (long)P->T.ny * 2 * (P->s1 - P->s0);            // real columns of the pencil [nz][ny][2 nsl]
    { VTab V = visc_tab(P, slot, comp, DIR_Z); LaunchTimer t(P, K_VZ, st); k_visc_sweep_strided<false, false><<<(unsigned)((ncol + 127) / 128), 128, 0, st>>>(V, pencil, nullptr, (int)ncol, (size_t)ncol, 0, ncol); }
    CU(cudaGetLastError());
    P->last_launches = launches + 1;
    return FSEI_OK;
}

extern "C" int fsei_slab_field_add(fsei_plan* P, double* q, const double* r, void* cuda_stream)
{
    SLAB_ONLY("fsei_slab_field_add");
    if (!q || !r || q == r || misaligned(q) || misaligned(r)) return fail(FSEI_ERR_ARG, "fsei_slab_field_add: NULL, aliased or misaligned fields");
    const size_t n2 = (size_t)P->T.nx * P->T.ny * (P->k1 - P->k0) / 2;
    k_field_add<<<(unsigned)((n2 + 255) / 256), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(q, r, n2);
    CU(cudaGetLastError());
    P->last_launches = 1;
    return FSEI_OK;
}

// ------------------------------------------------------------------------------------------
// per-kernel timing
// ------------------------------------------------------------------------------------------
extern "C" int fsei_plan_profile(fsei_plan* P, int enable)
{
    if (!P) return fail(FSEI_ERR_ARG, "fsei_plan_profile: NULL plan");
    if (enable && P->ev_pool.size() < 4096) {                    // all events are created here, none inside a timed loop
        P->ev_pool.reserve(4096); P->ev_kid.reserve(2048);
        while (P->ev_pool.size() < 4096) { cudaEvent_t e; CU(cudaEventCreate(&e)); P->ev_pool.push_back(e); }
    }
    P->profiling = enable != 0;
    return FSEI_OK;
}

extern "C" int fsei_plan_profile_read(fsei_plan* P, int max_kernels, double* ms_sum, long* count, const char** names)
{
    if (!P || !ms_sum || !count) return -fail(FSEI_ERR_ARG, "fsei_plan_profile_read: NULL argument");
    for (size_t i = 0; i < P->ev_kid.size(); i++) {
        cudaError_t e = cudaEventSynchronize(P->ev_pool[2 * i + 1]);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, P->ev_pool[2 * i], P->ev_pool[2 * i + 1]);
        if (e != cudaSuccess) return -cuda_fail(e, "fsei_plan_profile_read");
        P->prof_ms[P->ev_kid[i]] += ms; P->prof_n[P->ev_kid[i]]++;
    }
    P->ev_kid.clear(); P->ev_used = 0;
    int n = max_kernels < FSEI_NKERNELS ? max_kernels : FSEI_NKERNELS;
    for (int k = 0; k < n; k++) { ms_sum[k] = P->prof_ms[k]; count[k] = P->prof_n[k]; if (names) names[k] = k_names[k]; P->prof_ms[k] = 0; P->prof_n[k] = 0; }
    return n;
}
