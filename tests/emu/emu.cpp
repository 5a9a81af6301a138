// emu.cpp -- HOST STEPPING HARNESS for the device code of libfsei (test infrastructure).
//
// The kernels of paper_2103_15187_b200/csrc are written as sequences of per-thread phases
// (__host__ __device__ functions taking (tid, nthreads)) separated by block barriers.  This
// file includes those same headers and steps through the phases thread by thread on the
// host, so that the index arithmetic (digit-reversed in-place passes, packed half spectrum,
// DCT reorder, paired z-columns) is checked against the oracle in this GPU-less container
// before a GPU run.  It is built and used by tests/ only; the product never loads it.
#include <cstdio>
#include <cstring>
#include <vector>
#include "../../paper_2103_15187_b200/csrc/plan_host.hpp"
#include "../../paper_2103_15187_b200/csrc/xfft.cuh"
#include "../../paper_2103_15187_b200/csrc/yfft.cuh"
#include "../../paper_2103_15187_b200/csrc/zsolve.cuh"
#include "../../paper_2103_15187_b200/csrc/stencil.cuh"

using namespace fsei;

namespace {
struct Ctx {
    HostTables T;
    XParams X; YParams Y; ZParams Z; SParams S;
    std::vector<double> ipiv, gauge, cpw;
};

void setup(Ctx& c)
{
    HostTables& T = c.T;
    c.X.n = T.nx; c.X.N = T.nx / 2; c.X.bc = T.bcx; c.X.pitch = padx(T.nx / 2) + 1; c.X.f = T.fx;
    c.X.tw = T.twx.data(); c.X.pos = T.posx.data(); c.X.tw_r2c = T.twx_r2c.data(); c.X.tw_dct = T.twx_dct.data(); c.X.scale = T.scale;
    c.Y.N = T.ny; c.Y.bc = T.bcy; c.Y.f = T.fy; c.Y.tw = T.twy.data(); c.Y.pos = T.posy.data(); c.Y.tw_dct = T.twy_dct.data();
    c.Z.nxc = T.nxc; c.Z.ny = T.ny; c.Z.nz = T.nz; c.Z.ncomp = T.ncomp; c.Z.za = T.za.data(); c.Z.zcc = T.zcc.data();
    c.Z.lamx = T.lamx.data(); c.Z.lamy = T.lamy.data(); c.Z.posy = T.posy.data(); c.Z.dzc = T.dzc.data(); c.Z.dzm = T.dzm.data();
    c.gauge.assign(T.nz, 0.0); c.Z.gauge = c.gauge.data();
    c.S.nx = T.nx; c.S.ny = T.ny; c.S.nz = T.nz; c.S.bcx = T.bcx; c.S.bcy = T.bcy; c.S.rdx = T.rdx; c.S.rdy = T.rdy;
    c.S.rdzc = T.rdzc.data(); c.S.rdzm = T.rdzm.data();
    if (!T.paired_all) {
        c.ipiv.assign((size_t)T.nz * T.ny * T.nxc * T.ncomp, 0.0);
        c.Z.ipiv = c.ipiv.data();
        for (int row = 0; row < T.ny; row++)
            for (int slot = 0; slot < T.nxc; slot++)
                for (int comp = 0; comp < T.ncomp; comp++) {
                    bool zero = (row == 0 && slot == 0 && comp == 0) || (T.paired_slot0 && slot == 0);
                    z_factor_column(c.Z, c.ipiv.data(), row, slot, comp, zero);
                }
    }
    size_t npairs = (size_t)(T.ny / 2 + 1) * (T.paired_all ? T.nxc : 1);
    c.cpw.assign((size_t)T.nz * npairs * 2, 0.0); c.Z.cpw = c.cpw.data();
}

template <bool INV> void run_x_passes(const XParams& X, cplx* sm, int lines, int nt)
{
    int Ns[8]; int n = X.N;
    for (int s = 0; s < X.f.npass; s++) { Ns[s] = n; n /= X.f.radix[s]; }
    for (int i = 0; i < X.f.npass; i++) {
        int s = INV ? X.f.npass - 1 - i : i;
        for (int tid = 0; tid < nt; tid++) x_pass_dispatch<INV>(X, sm, lines, X.f.radix[s], Ns[s], tid, nt);
    }
}
template <bool INV, bool NEU> void run_y_passes(const YParams& Y, cplx* sm, int C, int nt)
{
    int Ns[8]; int n = Y.N;
    for (int s = 0; s < Y.f.npass; s++) { Ns[s] = n; n /= Y.f.radix[s]; }
    for (int i = 0; i < Y.f.npass; i++) {
        int s = INV ? Y.f.npass - 1 - i : i;
        for (int tid = 0; tid < nt; tid++) y_pass_dispatch<INV, NEU>(Y, sm, C, Y.f.radix[s], Ns[s], tid, nt);
    }
}

void poisson(Ctx& c, const double* rhs, double* phi)
{
    const HostTables& T = c.T;
    const int nt = 64, LX = 3;                       // odd tile height on purpose: exercises the ragged last tile
    const long nlines = (long)T.ny * T.nz;
    std::vector<cplx> sm((size_t)LX * c.X.pitch);
    cplx* spec = reinterpret_cast<cplx*>(phi);
    // a2: x forward
    for (long l0 = 0; l0 < nlines; l0 += LX) {
        int lines = (int)((nlines - l0 < LX) ? nlines - l0 : LX);
        for (int t = 0; t < nt; t++) x_load_real(c.X, sm.data(), rhs + (size_t)l0 * T.nx, lines, t, nt);
        run_x_passes<false>(c.X, sm.data(), lines, nt);
        for (int t = 0; t < nt; t++) x_post_forward(c.X, sm.data(), lines, t, nt);
        for (int t = 0; t < nt; t++) x_store_spec(c.X, sm.data(), spec + (size_t)l0 * T.nxc, lines, t, nt);
    }
    // a3: y forward
    int C = (T.nxc % 4 == 0) ? 4 : 2;
    std::vector<cplx> ty((size_t)T.ny * C);
    for (int k = 0; k < T.nz; k++)
        for (int c0 = 0; c0 < T.nxc; c0 += C) {
            cplx* g = spec + (size_t)k * T.ny * T.nxc + c0;
            for (int t = 0; t < nt; t++) y_load(ty.data(), g, T.nxc, T.ny, C, t, nt);
            if (T.bcy == BC_NEUMANN) {
                run_y_passes<false, true>(c.Y, ty.data(), C, nt);
                for (int t = 0; t < nt; t++) y_post_forward_dct(c.Y, ty.data(), C, t, nt);
            } else run_y_passes<false, false>(c.Y, ty.data(), C, nt);
            for (int t = 0; t < nt; t++) y_store(ty.data(), g, T.nxc, T.ny, C, t, nt);
        }
    // a4: gauge column first (reads d), then the tridiagonal solves
    {
        std::vector<double> d(T.nz);
        for (int k = 0; k < T.nz; k++) d[k] = spec[zidx(c.Z, k, 0, 0)].re;
        z_gauge_serial(c.Z, d.data(), c.gauge.data());
    }
    if (T.paired_all) {
        size_t np = (size_t)(T.ny / 2 + 1) * T.nxc;
        for (int q = 0; q <= T.ny / 2; q++)
            for (int slot = 0; slot < T.nxc; slot++) z_paired_column(c.Z, spec, slot, q, (size_t)q * T.nxc + slot, np);
    } else {
        int s0 = T.paired_slot0 ? 1 : 0;
        for (int row = 0; row < T.ny; row++)
            for (int slot = s0; slot < T.nxc; slot++) {
                bool g = (row == 0 && slot == 0);
                if (T.ncomp == 1) z_direct_column<1>(c.Z, spec, row, slot, g); else z_direct_column<2>(c.Z, spec, row, slot, g);
            }
        if (T.paired_slot0) {
            size_t np = (size_t)(T.ny / 2 + 1);
            for (int q = 0; q <= T.ny / 2; q++) z_paired_column(c.Z, spec, 0, q, (size_t)q, np);
        }
    }
    // a5: y inverse
    for (int k = 0; k < T.nz; k++)
        for (int c0 = 0; c0 < T.nxc; c0 += C) {
            cplx* g = spec + (size_t)k * T.ny * T.nxc + c0;
            for (int t = 0; t < nt; t++) y_load(ty.data(), g, T.nxc, T.ny, C, t, nt);
            if (T.bcy == BC_NEUMANN) {
                for (int t = 0; t < nt; t++) y_pre_inverse_dct(c.Y, ty.data(), C, t, nt);
                run_y_passes<true, true>(c.Y, ty.data(), C, nt);
            } else run_y_passes<true, false>(c.Y, ty.data(), C, nt);
            for (int t = 0; t < nt; t++) y_store(ty.data(), g, T.nxc, T.ny, C, t, nt);
        }
    // a6: x inverse
    for (long l0 = 0; l0 < nlines; l0 += LX) {
        int lines = (int)((nlines - l0 < LX) ? nlines - l0 : LX);
        for (int t = 0; t < nt; t++) x_load_spec(c.X, sm.data(), spec + (size_t)l0 * T.nxc, lines, t, nt);
        for (int t = 0; t < nt; t++) x_pre_inverse(c.X, sm.data(), lines, t, nt);
        run_x_passes<true>(c.X, sm.data(), lines, nt);
        for (int t = 0; t < nt; t++) x_store_real(c.X, sm.data(), phi + (size_t)l0 * T.nx, lines, t, nt);
    }
}
}  // namespace

extern "C" {

// whole projection through the stepped device phases; returns 0 or the plan error code
int emu_pressure_projection(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy,
                            double* u, double* v, double* w, double* p, double* phi, double alpha_dt, double beta)
{
    Ctx c; int code = 0;
    std::string msg = build_tables(c.T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code);
    if (code) { std::fprintf(stderr, "emu: %s\n", msg.c_str()); return code; }
    setup(c);
    const double inv_adt = 1.0 / alpha_dt;
    for (int k = 0; k < nz; k++) for (int j = 0; j < ny; j++) for (int i = 0; i < nx; i++)
        phi[sidx(c.S, i, j, k)] = div_at(c.S, u, v, w, i, j, k, inv_adt);
    poisson(c, phi, phi);
    for (int k = 0; k < nz; k++) for (int j = 0; j < ny; j++) for (int i = 0; i < nx; i++)
        project_at(c.S, u, v, w, p, phi, i, j, k, alpha_dt, beta);
    return 0;
}

int emu_poisson_solve(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy,
                      const double* rhs, double* phi)
{
    Ctx c; int code = 0;
    std::string msg = build_tables(c.T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code);
    if (code) { std::fprintf(stderr, "emu: %s\n", msg.c_str()); return code; }
    setup(c);
    if (rhs != phi) std::memcpy(phi, rhs, sizeof(double) * (size_t)nx * ny * nz);
    poisson(c, phi, phi);
    return 0;
}

// table checks used by the CPU tests
int emu_plan_radices(int N, int* radix) { FftPlan1D f = make_fft_plan(N); for (int i = 0; i < f.npass; i++) radix[i] = f.radix[i]; return f.npass; }
int emu_plan_check(int nx, int ny, int nz, double Lx, double Ly, const double* zc, int bcx, int bcy)
{
    HostTables T; int code = 0; build_tables(T, nx, ny, nz, Lx, Ly, zc, bcx, bcy, code); return code;
}
}
