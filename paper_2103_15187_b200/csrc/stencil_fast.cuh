// stencil_fast.cuh -- vectorised kernels of steps a1 (divergence / (alpha dt)) and a7 (velocity correction
// + pressure update): one thread per pair of x-adjacent cells, 128-bit loads and stores.  The per-cell
// arithmetic is that of stencil.cuh (same operations in the same order, every one individually rounded),
// so the results are bit-identical to the definition (R20).  P:L87.
#pragma once
#include "kernel_env.cuh"
#include "stencil.cuh"

namespace fsei {

FSEI_HD cplx sld2(const double* p) { return *reinterpret_cast<const cplx*>(p); }
FSEI_HD void sst2(double* p, cplx v) { *reinterpret_cast<cplx*>(p) = v; }

// p + (c0 - beta * L phi) at one cell from its neighbours (0 / flags false on wall faces)
FSEI_HD double pressure_cell(const SParams& S, double p, double c0, double pxm, double pxp, double pym, double pyp,
                             double pzm, double pzp, bool xlo, bool xhi, bool ylo, bool yhi, bool zlo, bool zhi,
                             double rdzm_k, double rdzm_kp, double rdzc_k, double beta)
{
    double gxm = xlo ? FSEI_MUL(FSEI_SUB(c0, pxm), S.rdx) : 0.0;
    double gxp = xhi ? FSEI_MUL(FSEI_SUB(pxp, c0), S.rdx) : 0.0;
    double gym = ylo ? FSEI_MUL(FSEI_SUB(c0, pym), S.rdy) : 0.0;
    double gyp = yhi ? FSEI_MUL(FSEI_SUB(pyp, c0), S.rdy) : 0.0;
    double gzm = zlo ? FSEI_MUL(FSEI_SUB(c0, pzm), rdzm_k) : 0.0;
    double gzp = zhi ? FSEI_MUL(FSEI_SUB(pzp, c0), rdzm_kp) : 0.0;
    double l = lap_cell(gxm, gxp, gym, gyp, gzm, gzp, S.rdx, S.rdy, rdzc_k);
    return FSEI_ADD(p, FSEI_SUB(c0, FSEI_MUL(beta, l)));
}

// grid ceil(nx ny nz / 2 / 256), block 256
FSEI_GLOBAL(256, 1) k_divergence_fast(SParams S, const double* __restrict__ u, const double* __restrict__ v,
                                      const double* __restrict__ w, double inv_adt, double* __restrict__ rhs)
{
    const int hx = S.nx >> 1;
    const size_t npair = (size_t)hx * S.ny * S.nz;
    const size_t pr = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (pr >= npair) return;
    const int t = (int)(pr % hx); const size_t r = pr / hx; const int j = (int)(r % S.ny), k = (int)(r / S.ny);
    const size_t line = r * S.nx, c = line + 2 * t, plane = (size_t)S.nx * S.ny;
    cplx uu = sld2(u + c);
    double un = (2 * t + 2 < S.nx) ? u[c + 2] : (S.bcx == BC_PERIODIC ? u[line] : 0.0);
    cplx vv = sld2(v + c);
    cplx vp = (j + 1 < S.ny) ? sld2(v + c + S.nx) : (S.bcy == BC_PERIODIC ? sld2(v + c - (size_t)(S.ny - 1) * S.nx) : cmake(0.0, 0.0));
    cplx ww = sld2(w + c);
    cplx wp = (k + 1 < S.nz || S.halo_hi) ? sld2(w + c + plane) : cmake(0.0, 0.0);
    const double rdz = S.rdzc[k + S.kofs];
    sst2(rhs + c, cmake(div_cell(uu.re, uu.im, vv.re, vp.re, ww.re, wp.re, S.rdx, S.rdy, rdz, inv_adt),
                        div_cell(uu.im, un, vv.im, vp.im, ww.im, wp.im, S.rdx, S.rdy, rdz, inv_adt)));
}

// grid ceil(nx ny nz / 2 / 256), block 256
FSEI_GLOBAL(256, 4) k_project_fast(SParams S, double* __restrict__ u, double* __restrict__ v, double* __restrict__ w,
                                   double* __restrict__ p, const double* __restrict__ phi, double adt, double beta)
{
    const int hx = S.nx >> 1;
    const size_t npair = (size_t)hx * S.ny * S.nz;
    const size_t pr = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (pr >= npair) return;
    const int t = (int)(pr % hx); const size_t r = pr / hx; const int j = (int)(r % S.ny), k = (int)(r / S.ny);
    const size_t line = r * S.nx, c = line + 2 * t, plane = (size_t)S.nx * S.ny;
    const bool xper = S.bcx == BC_PERIODIC, yper = S.bcy == BC_PERIODIC;
    const bool xlo0 = (t > 0) || xper, ylo = (j > 0) || yper, zlo = k > 0 || S.halo_lo;
    const cplx z0 = cmake(0.0, 0.0);

    const cplx c0 = sld2(phi + c);
    const double pxm = (t > 0) ? phi[c - 1] : (xper ? phi[line + S.nx - 1] : 0.0);
    const cplx pym = ylo ? sld2(phi + (j > 0 ? c - S.nx : c + (size_t)(S.ny - 1) * S.nx)) : z0;
    const cplx pzm = zlo ? sld2(phi + c - plane) : z0;
    cplx uu = sld2(u + c), vv = sld2(v + c), ww = sld2(w + c), pp = sld2(p + c);
    const double rzm = S.rdzm[k + S.kofs];

    if (xlo0) uu.re = corr_face(uu.re, c0.re, pxm, S.rdx, adt);
    uu.im = corr_face(uu.im, c0.im, c0.re, S.rdx, adt);
    if (ylo) { vv.re = corr_face(vv.re, c0.re, pym.re, S.rdy, adt); vv.im = corr_face(vv.im, c0.im, pym.im, S.rdy, adt); }
    if (zlo) { ww.re = corr_face(ww.re, c0.re, pzm.re, rzm, adt); ww.im = corr_face(ww.im, c0.im, pzm.im, rzm, adt); }
    if (beta == 0.0) {
        pp.re = FSEI_ADD(pp.re, c0.re); pp.im = FSEI_ADD(pp.im, c0.im);
    } else {
        const bool xhi1 = (2 * t + 2 < S.nx) || xper, yhi = (j + 1 < S.ny) || yper, zhi = k + 1 < S.nz || S.halo_hi;
        const double pxp = (2 * t + 2 < S.nx) ? phi[c + 2] : (xper ? phi[line] : 0.0);
        const cplx pyp = yhi ? sld2(phi + (j + 1 < S.ny ? c + S.nx : c - (size_t)(S.ny - 1) * S.nx)) : z0;
        const cplx pzp = zhi ? sld2(phi + c + plane) : z0;
        const double rzp = zhi ? S.rdzm[k + 1 + S.kofs] : 0.0, rzc = S.rdzc[k + S.kofs];
        pp.re = pressure_cell(S, pp.re, c0.re, pxm, c0.im, pym.re, pyp.re, pzm.re, pzp.re, xlo0, true, ylo, yhi, zlo, zhi, rzm, rzp, rzc, beta);
        pp.im = pressure_cell(S, pp.im, c0.im, c0.re, pxp, pym.im, pyp.im, pzm.im, pzp.im, true, xhi1, ylo, yhi, zlo, zhi, rzm, rzp, rzc, beta);
    }
    sst2(u + c, uu); sst2(v + c, vv); sst2(w + c, ww); sst2(p + c, pp);
}

}  // namespace fsei
