// stencil.cuh -- per-cell arithmetic of steps a1 (divergence / (alpha dt)) and a7 (velocity
// correction + pressure update).  P:L87 (staggered second-order differences)
// (fractional step).  The operation order is the one DESIGN.md R20 fixes, every operation
// individually rounded (no FMA contraction), so the result is bit-identical to the definition.
#pragma once
#include "plan_types.cuh"

namespace fsei {

#if defined(__CUDA_ARCH__)
#define FSEI_MUL(a, b) __dmul_rn((a), (b))
#define FSEI_ADD(a, b) __dadd_rn((a), (b))
#define FSEI_SUB(a, b) __dsub_rn((a), (b))
#else   // host stepping harness: compiled with -ffp-contract=off
#define FSEI_MUL(a, b) ((a) * (b))
#define FSEI_ADD(a, b) ((a) + (b))
#define FSEI_SUB(a, b) ((a) - (b))
#endif

// ((du*rdx + dv*rdy) + dw*rdz) * inv_adt
FSEI_HD double div_cell(double u0, double up, double v0, double vp, double w0, double wp,
                        double rdx, double rdy, double rdz, double inv_adt)
{
    double du = FSEI_SUB(up, u0), dv = FSEI_SUB(vp, v0), dw = FSEI_SUB(wp, w0);
    return FSEI_MUL(FSEI_ADD(FSEI_ADD(FSEI_MUL(du, rdx), FSEI_MUL(dv, rdy)), FSEI_MUL(dw, rdz)), inv_adt);
}

// q - adt*((c0 - pm)*r)
FSEI_HD double corr_face(double q, double c0, double pm, double r, double adt)
{
    return FSEI_SUB(q, FSEI_MUL(adt, FSEI_MUL(FSEI_SUB(c0, pm), r)));
}

// L phi at a cell from its six face gradients (0 on wall faces):
// ((gxp-gxm)*rdx + (gyp-gym)*rdy) + (gzp-gzm)*rdzc
FSEI_HD double lap_cell(double gxm, double gxp, double gym, double gyp, double gzm, double gzp,
                        double rdx, double rdy, double rdzc)
{
    return FSEI_ADD(FSEI_ADD(FSEI_MUL(FSEI_SUB(gxp, gxm), rdx), FSEI_MUL(FSEI_SUB(gyp, gym), rdy)),
                    FSEI_MUL(FSEI_SUB(gzp, gzm), rdzc));
}

FSEI_HD size_t sidx(const SParams& S, int i, int j, int k) { return ((size_t)k * S.ny + j) * S.nx + i; }

// reference-shaped per-cell versions (used by the simple kernels and by the host harness)
FSEI_HD double div_at(const SParams& S, const double* u, const double* v, const double* w,
                      int i, int j, int k, double inv_adt)
{
    double up = (i + 1 < S.nx) ? u[sidx(S, i + 1, j, k)] : (S.bcx == BC_PERIODIC ? u[sidx(S, 0, j, k)] : 0.0);
    double vp = (j + 1 < S.ny) ? v[sidx(S, i, j + 1, k)] : (S.bcy == BC_PERIODIC ? v[sidx(S, i, 0, k)] : 0.0);
    double wp = (k + 1 < S.nz) ? w[sidx(S, i, j, k + 1)] : 0.0;
    size_t c = sidx(S, i, j, k);
    return div_cell(u[c], up, v[c], vp, w[c], wp, S.rdx, S.rdy, S.rdzc[k], inv_adt);
}

FSEI_HD void project_at(const SParams& S, double* u, double* v, double* w, double* p, const double* phi,
                        int i, int j, int k, double adt, double beta)
{
    const size_t c = sidx(S, i, j, k);
    const double c0 = phi[c];
    const bool xlo = (i > 0) || S.bcx == BC_PERIODIC, ylo = (j > 0) || S.bcy == BC_PERIODIC;
    double pxm = xlo ? phi[sidx(S, i > 0 ? i - 1 : S.nx - 1, j, k)] : 0.0;
    double pym = ylo ? phi[sidx(S, i, j > 0 ? j - 1 : S.ny - 1, k)] : 0.0;
    double pzm = (k > 0) ? phi[sidx(S, i, j, k - 1)] : 0.0;
    if (xlo) u[c] = corr_face(u[c], c0, pxm, S.rdx, adt);
    if (ylo) v[c] = corr_face(v[c], c0, pym, S.rdy, adt);
    if (k > 0) w[c] = corr_face(w[c], c0, pzm, S.rdzm[k], adt);
    if (beta == 0.0) {
        p[c] = FSEI_ADD(p[c], c0);
    } else {
        const bool xhi = (i + 1 < S.nx) || S.bcx == BC_PERIODIC, yhi = (j + 1 < S.ny) || S.bcy == BC_PERIODIC;
        double pxp = xhi ? phi[sidx(S, i + 1 < S.nx ? i + 1 : 0, j, k)] : 0.0;
        double pyp = yhi ? phi[sidx(S, i, j + 1 < S.ny ? j + 1 : 0, k)] : 0.0;
        double gxm = xlo ? FSEI_MUL(FSEI_SUB(c0, pxm), S.rdx) : 0.0;
        double gxp = xhi ? FSEI_MUL(FSEI_SUB(pxp, c0), S.rdx) : 0.0;
        double gym = ylo ? FSEI_MUL(FSEI_SUB(c0, pym), S.rdy) : 0.0;
        double gyp = yhi ? FSEI_MUL(FSEI_SUB(pyp, c0), S.rdy) : 0.0;
        double gzm = (k > 0) ? FSEI_MUL(FSEI_SUB(c0, pzm), S.rdzm[k]) : 0.0;
        double gzp = (k + 1 < S.nz) ? FSEI_MUL(FSEI_SUB(phi[sidx(S, i, j, k + 1)], c0), S.rdzm[k + 1]) : 0.0;
        double l = lap_cell(gxm, gxp, gym, gyp, gzm, gzp, S.rdx, S.rdy, S.rdzc[k]);
        p[c] = FSEI_ADD(p[c], FSEI_SUB(c0, FSEI_MUL(beta, l)));
    }
}

}  // namespace fsei
