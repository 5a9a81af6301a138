// emu_fast.cpp -- HOST HARNESS for the fast-path kernels of libfsei (test infrastructure).
//
// The fast-path kernels (xfast.cuh, yfast.cuh, zfast.cuh, stencil_fast.cuh) are written against the
// macros of kernel_env.cuh; here they are compiled by g++ with cuda_shim.hpp standing in for the CUDA
// execution model (a CTA = a team of host threads with a barrier) and run on the same launch shapes
// as libfsei uses, so that their index arithmetic (Stockham passes, padded tiles, pair steps, split
// y-spectra, special z columns) is checked against the oracle in this GPU-less container.
#include <cstdio>
#include <cstring>
#include <vector>
#include "cuda_shim.hpp"
#include "../../paper_2103_15187_b200/csrc/plan_host.hpp"
#include "../../paper_2103_15187_b200/csrc/fast_configs.hpp"
#include "../../paper_2103_15187_b200/csrc/xfast.cuh"
#include "../../paper_2103_15187_b200/csrc/yfast.cuh"
#include "../../paper_2103_15187_b200/csrc/yzfused.cuh"
#include "../../paper_2103_15187_b200/csrc/zfast.cuh"
#include "../../paper_2103_15187_b200/csrc/stencil_fast.cuh"

using namespace fsei;

namespace {

bool x_ok(int N) { switch (N) {
#define X(n, a, b, c) case n:
    FSEI_X_CONFIGS(X)
#undef X
    return true; default: return false; } }
bool y_ok(int N) { switch (N) {
#define X(n, a, b, c, cy) case n:
    FSEI_Y_CONFIGS(X)
#undef X
    return true; default: return false; } }

template <class C, bool NEU> void xf_one(const XFast& P, const SParams& S, bool fused, const double* u, const double* v, const double* w,
                                         double inv_adt, cplx* spec)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    if (fused) cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, [&] { k_xf_fast<C, LPB, NEU, true>(P, S, u, v, w, inv_adt, spec); });
    else cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, [&] { k_xf_fast<C, LPB, NEU, false>(P, S, u, v, w, inv_adt, spec); });
}
void xf(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v, const double* w, double inv_adt, cplx* spec)
{
    switch (P.N) {
#define X(n, a, b, c) case n: if (neu) xf_one<FftCfg<n, a, b, c>, true>(P, S, fused, u, v, w, inv_adt, spec); \
                              else xf_one<FftCfg<n, a, b, c>, false>(P, S, fused, u, v, w, inv_adt, spec); break;
        FSEI_X_CONFIGS(X)
#undef X
    }
}
template <class C, bool NEU> void xi_one(const XFast& P, const cplx* spec, double* phi)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    TmaMap3D none{};
    cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, [&] { k_xi_fast<C, LPB, NEU>(P, none, spec, phi); });
}
void xi(const XFast& P, bool neu, const cplx* spec, double* phi)
{
    switch (P.N) {
#define X(n, a, b, c) case n: if (neu) xi_one<FftCfg<n, a, b, c>, true>(P, spec, phi); else xi_one<FftCfg<n, a, b, c>, false>(P, spec, phi); break;
        FSEI_X_CONFIGS(X)
#undef X
    }
}
template <class C, int CY> void y_one(const YFast& P, bool inv, bool neu, cplx* spec)
{
    const int gx = (P.nxc + CY - 1) / CY;
    int gy = P.nz < 3 ? P.nz : 3;                      // fewer blocks than planes: exercises the plane loop
    dim3 grid(gx, gy);
    const int nt = C::T * CY;
    const size_t b0 = YSmemLayout<C, CY, false>::BYTES, b1 = YSmemLayout<C, CY, true>::BYTES;
    TmaMap2D map{reinterpret_cast<const unsigned char*>(spec), (size_t)P.nxc * sizeof(cplx), (unsigned)sizeof(double), 2u * CY,
                 (unsigned)y_box_rows(C::N)};
    if (!inv && !neu) cuda_shim::launch(grid, nt, b0, [&] { k_y_fast<C, CY, false, false>(P, map, spec); });
    else if (inv && !neu) cuda_shim::launch(grid, nt, b0, [&] { k_y_fast<C, CY, true, false>(P, map, spec); });
    else if (!inv && neu) cuda_shim::launch(grid, nt, b1, [&] { k_y_fast<C, CY, false, true>(P, map, spec); });
    else cuda_shim::launch(grid, nt, b1, [&] { k_y_fast<C, CY, true, true>(P, map, spec); });
}
void yf(const YFast& P, bool inv, bool neu, cplx* spec)
{
    switch (P.ny) {
#define X(n, a, b, c, cy) case n: y_one<FftCfg<n, a, b, c>, cy>(P, inv, neu, spec); break;
        FSEI_Y_CONFIGS(X)
#undef X
    }
}

// ---- fused path: blocked spectrum layout, z-marching y kernels ------------------------------------------
bool xb_ok(int N) { switch (N) {
#define X(n, a, b, c) case n:
    FSEI_XB_CONFIGS(X)
#undef X
    return true; default: return false; } }
bool yz_ok(int N) { switch (N) {
#define X(n, a, b, c) case n:
    FSEI_YZ_CONFIGS(X)
#undef X
    return true; default: return false; } }

template <class C, bool NEU> void xfb_one(const XFast& P, const SParams& S, bool fused, const double* u, const double* v, const double* w,
                                          double inv_adt, cplx* spec)
{
    constexpr int LPB = XShape<C, NEU>::LPB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    if (fused) cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, 4 * LPB + 1>::BYTES, [&] { k_xf_fast<C, LPB, NEU, true, FSEI_CB>(P, S, u, v, w, inv_adt, spec); });
    else cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, [&] { k_xf_fast<C, LPB, NEU, false, FSEI_CB>(P, S, u, v, w, inv_adt, spec); });
}
void xfb(const XFast& P, const SParams& S, bool neu, bool fused, const double* u, const double* v, const double* w, double inv_adt, cplx* spec)
{
    switch (P.N) {
#define X(n, a, b, c) case n: if (neu) xfb_one<FftCfg<n, a, b, c>, true>(P, S, fused, u, v, w, inv_adt, spec); \
                              else xfb_one<FftCfg<n, a, b, c>, false>(P, S, fused, u, v, w, inv_adt, spec); break;
        FSEI_XB_CONFIGS(X)
#undef X
    }
}
template <class C, bool NEU> void xib_one(const XFast& P, const cplx* spec, double* phi)
{
    constexpr int LPB = XShape<C, NEU>::LPB, CB = FSEI_CB, NXT = C::N / CB;
    dim3 grid((P.ny + LPB - 1) / LPB, (P.nz + P.kchunk - 1) / P.kchunk);
    // the view make_xi_blocked_map (fast_x.cu) encodes: (2 ny CB doubles, nz, N / CB), boxes (2 LPB CB, 1, xi_box_tiles)
    TmaMap3D map{reinterpret_cast<const unsigned char*>(spec), (size_t)P.ny * CB * sizeof(cplx), (size_t)P.nz * P.ny * CB * sizeof(cplx),
                 (unsigned)sizeof(double), 2u * P.ny * CB, (unsigned)P.nz, (unsigned)NXT, 2u * LPB * CB, 1u, (unsigned)xi_box_tiles(NXT)};
    cuda_shim::launch(grid, C::T * LPB, XSmemLayout<C, LPB, NEU, LPB>::BYTES, [&] { k_xi_fast<C, LPB, NEU, FSEI_CB>(P, map, spec, phi); });
}
void xib(const XFast& P, bool neu, const cplx* spec, double* phi)
{
    switch (P.N) {
#define X(n, a, b, c) case n: if (neu) xib_one<FftCfg<n, a, b, c>, true>(P, spec, phi); else xib_one<FftCfg<n, a, b, c>, false>(P, spec, phi); break;
        FSEI_XB_CONFIGS(X)
#undef X
    }
}
template <class C, bool NEU, int NCOMP> void yz_variant(const YZFused& P, bool backward, cplx* spec)
{
    using L = YZSmem<C, FSEI_CB, NEU, NCOMP>;
    const dim3 grid(P.nxc / FSEI_CB, P.ktw < P.nz ? 2 : 1);
    const unsigned nt = C::T * FSEI_CB;
    if (!backward) cuda_shim::launch(grid, nt, L::FWD, [&] { k_yz_forward<C, FSEI_CB, NEU, NCOMP>(P, spec); });
    else cuda_shim::launch(grid, nt, L::BWD, [&] { k_yz_backward<C, FSEI_CB, NEU, NCOMP>(P, spec); });
}
void yz(const YZFused& P, bool backward, bool neu, int ncomp, cplx* spec)
{
    switch (P.ny) {
#define X(n, a, b, c) case n: if (neu) yz_variant<FftCfg<n, a, b, c>, true, 2>(P, backward, spec); \
                              else if (ncomp == 1) yz_variant<FftCfg<n, a, b, c>, false, 1>(P, backward, spec); \
                              else yz_variant<FftCfg<n, a, b, c>, false, 2>(P, backward, spec); break;
        FSEI_YZ_CONFIGS(X)
#undef X
    }
}

struct Ctx {
    HostTables T;
    SParams S; XFast XF; YFast YF; ZFast ZF;
    std::vector<double> ipiv, cpw;
    std::vector<cplx> special, special_in, mid;
};

void setup(Ctx& c, bool blocked = false, bool twist = false)
{
    HostTables& T = c.T;
    c.S.nx = T.nx; c.S.ny = T.ny; c.S.nz = T.nz; c.S.bcx = T.bcx; c.S.bcy = T.bcy; c.S.rdx = T.rdx; c.S.rdy = T.rdy;
    c.S.rdzc = T.rdzc.data(); c.S.rdzm = T.rdzm.data();
    XFast& XF = c.XF; YFast& YF = c.YF; ZFast& ZF = c.ZF;
    XF.nx = T.nx; XF.ny = T.ny; XF.nz = T.nz; XF.N = T.nx / 2; XF.tw = T.twx.data(); XF.tw_r2c = T.twx_r2c.data();
    XF.tw_dct = T.twx_dct.data(); XF.scale = T.scale; XF.kchunk = T.nz < 3 ? T.nz : 3;
    YF.nxc = T.nxc; YF.ny = T.ny; YF.nz = T.nz; YF.tw = T.twy.data(); YF.tw_dct = T.twy_dct.data();
    YF.untangle = (T.bcy == BC_PERIODIC) ? (T.bcx == BC_PERIODIC ? 1 : T.nxc) : 0;
    ZF.nxc = T.nxc; ZF.ny = T.ny; ZF.nz = T.nz; ZF.bcx = T.bcx; ZF.bcy = T.bcy;
    ZF.ncomp = (T.bcx == BC_PERIODIC && T.bcy == BC_PERIODIC) ? 1 : 2;
    ZF.za = T.za.data(); ZF.zcc = T.zcc.data(); ZF.lamx = T.lamx.data(); ZF.lamy = T.lamy.data(); ZF.dzc = T.dzc.data(); ZF.dzm = T.dzm.data();
    c.special.assign(2 * (size_t)T.nz, cmake(0, 0)); ZF.special = c.special.data();
    c.cpw.assign(8 * (size_t)T.nz, 0.0); ZF.cpw = c.cpw.data();
    ZF.cb = blocked ? FSEI_CB : 0; ZF.special_in = nullptr;
    ZF.ktw = (twist && T.nz >= 4) ? T.nz / 2 : T.nz;
    if (blocked) { c.special_in.assign(2 * (size_t)T.nz, cmake(0, 0)); ZF.special_in = c.special_in.data(); }
    c.ipiv.assign((size_t)T.nz * T.ny * T.nxc * ZF.ncomp, 0.0); ZF.ipiv = c.ipiv.data();
    size_t cols = (size_t)T.ny * T.nxc * ZF.ncomp;
    cuda_shim::launch((unsigned)((cols + 255) / 256), 256, 0, [&] { k_zf_factor(ZF, c.ipiv.data()); });
    cuda_shim::launch(1, 32, 0, [&] { k_z_special_factor(ZF); });
}

// pcr: short columns through the warp-shuffle PCR kernel (as libfsei does for nz <= 32); the shuffle emulation costs
// two host barriers per call, so the harness uses it on request only
void spectral_solve(Ctx& c, cplx* spec, bool pcr = false)
{
    const HostTables& T = c.T;
    const bool yneu = T.bcy == BC_NEUMANN;
    yf(c.YF, false, yneu, spec);
    cuda_shim::launch(1, 128, z_special_smem(T.nz, z_special_staged(T.nz)), [&] { k_z_special(c.ZF, spec, z_special_staged(T.nz)); });
    size_t nthr = (size_t)T.nxc * T.ny;
    if (pcr && T.nz <= 32) cuda_shim::launch((unsigned)((nthr * 32 + 127) / 128), 128, 0, [&] { k_zf_pcr(c.ZF, spec); });
    else if (c.ZF.ncomp == 1) cuda_shim::launch((unsigned)((nthr + 127) / 128), 128, 0, [&] { k_zf_sweep<1>(c.ZF, spec); });
    else cuda_shim::launch((unsigned)((nthr + 127) / 128), 128, 0, [&] { k_zf_sweep<2>(c.ZF, spec); });
    yf(c.YF, true, yneu, spec);
    xi(c.XF, T.bcx == BC_NEUMANN, spec, reinterpret_cast<double*>(spec));
}

// a3 .. a6 of the fused path: work = blocked spectrum, phi receives the result
void fused_spectral_solve(Ctx& c, cplx* work, double* phi)
{
    const HostTables& T = c.T;
    YZFused YZ;
    YZ.nxc = T.nxc; YZ.ny = T.ny; YZ.nz = T.nz; YZ.untangle = c.YF.untangle;
    YZ.pp = (T.bcx == BC_PERIODIC && T.bcy == BC_PERIODIC) ? 1 : 0;
    YZ.tw = T.twy.data(); YZ.tw_dct = T.twy_dct.data(); YZ.za = T.za.data(); YZ.zcc = T.zcc.data(); YZ.ip = c.ipiv.data();
    YZ.special_in = c.special_in.data(); YZ.special = c.special.data();
    YZ.tile_shift[0] = 3 % (T.nxc / FSEI_CB); YZ.tile_shift[1] = 5 % (T.nxc / FSEI_CB);
    YZ.ktw = c.ZF.ktw; c.mid.assign((size_t)T.nxc * T.ny * 2, cmake(0, 0)); YZ.mid = c.mid.data();
    const bool yneu = T.bcy == BC_NEUMANN;
    yz(YZ, false, yneu, c.ZF.ncomp, work);
    cuda_shim::launch(1, 128, z_special_smem(T.nz, z_special_staged(T.nz)), [&] { k_z_special(c.ZF, work, z_special_staged(T.nz)); });
    yz(YZ, true, yneu, c.ZF.ncomp, work);
    xib(c.XF, T.bcx == BC_NEUMANN, work, phi);
}
}  // namespace

extern "C" {

int emu_fused_supported(int nx, int ny) { return nx >= 4 && nx % 2 == 0 && xb_ok(nx / 2) && yz_ok(ny) && (nx / 2) % FSEI_CB == 0; }

// whole projection through the fused-path kernels (blocked spectrum in a workspace field)
int emu_fused_pressure_projection(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy,
                                  double* u, double* v, double* w, double* p, double* phi, double alpha_dt, double beta, int split)
{
    if (!emu_fused_supported(nx, ny)) return -1;
    Ctx c; int code = 0;
    std::string msg = build_tables(c.T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code, true);
    if (code) { std::fprintf(stderr, "emu: %s\n", msg.c_str()); return code; }
    setup(c, true, (split & 4) != 0);                      // split & 4: twisted factorisation (two CTAs per tile)
    const size_t n = (size_t)nx * ny * nz;
    const unsigned gpairs = (unsigned)((n / 2 + 255) / 256);
    std::vector<cplx> work(n / 2);
    const bool xneu = bcx == BC_NEUMANN;
    if (split & 1) {
        cuda_shim::launch(gpairs, 256, 0, [&] { k_divergence_fast(c.S, u, v, w, 1.0 / alpha_dt, phi); });
        xfb(c.XF, c.S, xneu, false, phi, nullptr, nullptr, 0.0, work.data());
    } else {
        xfb(c.XF, c.S, xneu, true, u, v, w, 1.0 / alpha_dt, work.data());
    }
    fused_spectral_solve(c, work.data(), phi);
    cuda_shim::launch(gpairs, 256, 0, [&] { k_project_fast(c.S, u, v, w, p, phi, alpha_dt, beta); });
    return 0;
}

int emu_fast_supported(int nx, int ny) { return nx >= 4 && nx % 2 == 0 && x_ok(nx / 2) && y_ok(ny); }

// whole projection through the fast-path kernels.  split & 1: divergence kernel + non-fused x-forward;
// split & 2: z-solve by the PCR kernel (nz <= 32).
int emu_fast_pressure_projection(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy,
                                 double* u, double* v, double* w, double* p, double* phi, double alpha_dt, double beta, int split)
{
    if (!emu_fast_supported(nx, ny)) return -1;
    Ctx c; int code = 0;
    std::string msg = build_tables(c.T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code, true);
    if (code) { std::fprintf(stderr, "emu: %s\n", msg.c_str()); return code; }
    setup(c);
    const size_t n = (size_t)nx * ny * nz;
    const unsigned gpairs = (unsigned)((n / 2 + 255) / 256);
    cplx* spec = reinterpret_cast<cplx*>(phi);
    const bool xneu = bcx == BC_NEUMANN;
    if (split & 1) {
        cuda_shim::launch(gpairs, 256, 0, [&] { k_divergence_fast(c.S, u, v, w, 1.0 / alpha_dt, phi); });
        xf(c.XF, c.S, xneu, false, phi, nullptr, nullptr, 0.0, spec);
    } else {
        xf(c.XF, c.S, xneu, true, u, v, w, 1.0 / alpha_dt, spec);
    }
    spectral_solve(c, spec, (split & 2) != 0);
    cuda_shim::launch(gpairs, 256, 0, [&] { k_project_fast(c.S, u, v, w, p, phi, alpha_dt, beta); });
    return 0;
}
}
