// zsolve.cuh -- per-thread work of step a4: one real tridiagonal system per wavenumber pair,
//   a_k x_{k-1} + (-(a_k + c_k) + lambda) x_k + c_k x_{k+1} = d_k,   lambda = lambda_x + lambda_y,
// solved by Thomas' algorithm along z, in place in the spectrum, and the singular
// (0,0) column by two prefix sums + volume-weighted zero mean (R7, R8).
//
// The matrix depends only on the grid, so its factorisation (reciprocal pivots) is computed
// once per plan (z_factor_column); the per-call sweeps then hold no division.
#pragma once
#include "plan_types.cuh"

namespace fsei {

FSEI_HD size_t zidx(const ZParams& Z, int k, int row, int slot) { return ((size_t)k * Z.ny + row) * Z.nxc + slot; }

// plan time: reciprocal pivots of column (row, slot), component comp.  zero_it: column unused
// by the direct kernel (gauge component, or a slot the paired kernel owns).
FSEI_HD void z_factor_column(const ZParams& Z, double* ipiv, int row, int slot, int comp, bool zero_it)
{
    const double lam = Z.lamx[2 * slot + comp] + Z.lamy[row];
    double cp = 0.0;
    for (int k = 0; k < Z.nz; k++) {
        double a = Z.za[k], c = Z.zcc[k];
        double piv = (-(a + c) + lam) - a * cp;
        double ip = zero_it ? 0.0 : 1.0 / piv;
        ipiv[zidx(Z, k, row, slot) * Z.ncomp + comp] = ip;
        cp = c * ip;
    }
}

// direct kernel: one thread per (row, slot); Re and Im are two right-hand sides.
// NCOMP = 1: they share the factorisation; NCOMP = 2: each has its own (lambda differs).
template <int NCOMP>
FSEI_HD void z_direct_column(const ZParams& Z, cplx* S, int row, int slot, bool gauge_re)
{
    const int nz = Z.nz;
    cplx prev = cmake(0.0, 0.0);
    for (int k = 0; k < nz; k++) {
        size_t i = zidx(Z, k, row, slot);
        cplx d = S[i];
        double ipr = Z.ipiv[i * NCOMP], ipi = Z.ipiv[i * NCOMP + (NCOMP - 1)];
        double a = Z.za[k];
        prev = cmake((d.re - a * prev.re) * ipr, (d.im - a * prev.im) * ipi);
        S[i] = prev;
    }
    cplx next = cmake(0.0, 0.0);
    for (int k = nz - 1; k >= 0; k--) {
        size_t i = zidx(Z, k, row, slot);
        cplx dp = S[i];
        double ipr = Z.ipiv[i * NCOMP], ipi = Z.ipiv[i * NCOMP + (NCOMP - 1)];
        double c = Z.zcc[k];
        next = cmake(dp.re - (c * ipr) * next.re, dp.im - (c * ipi) * next.im);
        if (gauge_re) next.re = Z.gauge[k];
        S[i] = next;
        if (gauge_re) next.re = 0.0;
    }
}

// paired kernel (y periodic, Re and Im of the slot are two packed real x-sequences A, B whose
// y-spectra are Hermitian): pair q = ky in [0, ny/2] owns rows r1 = pos[ky], r2 = pos[ny-ky].
//   A(ky) = (P1 + conj P2)/2,  B(ky) = (P1 - conj P2)/(2i);  solve each with its own lambda;
//   P1 <- A^ + i B^,  P2 <- conj(A^) + i conj(B^).
// Self-paired rows (ky = 0, ny/2) carry real A, B in one slot.  Factorisation on the fly,
// c' kept in Z.cpw[(k*npairs + pairidx)*2 + {0,1}].
FSEI_HD void z_paired_column(const ZParams& Z, cplx* S, int slot, int q, size_t pairidx, size_t npairs)
{
    const int nz = Z.nz, ny = Z.ny;
    const int r1 = Z.posy[q], r2 = Z.posy[(ny - q) % ny];
    const bool self = (r1 == r2);
    const bool gaugeA = (slot == 0 && q == 0);
    const double lamA = Z.lamx[2 * slot] + Z.lamy[r1], lamB = Z.lamx[2 * slot + 1] + Z.lamy[r1];
    cplx pa = cmake(0, 0), pb = cmake(0, 0);
    double cpa = 0.0, cpb = 0.0;
    for (int k = 0; k < nz; k++) {
        size_t i1 = zidx(Z, k, r1, slot), i2 = zidx(Z, k, r2, slot);
        cplx p1 = S[i1], p2 = self ? p1 : S[i2];
        cplx A = cmake(0.5 * (p1.re + p2.re), 0.5 * (p1.im - p2.im));
        cplx D = cmake(p1.re - p2.re, p1.im + p2.im);
        cplx B = cmake(0.5 * D.im, -0.5 * D.re);
        double a = Z.za[k], c = Z.zcc[k];
        double ipa = gaugeA ? 0.0 : 1.0 / ((-(a + c) + lamA) - a * cpa);
        double ipb = 1.0 / ((-(a + c) + lamB) - a * cpb);
        cpa = c * ipa; cpb = c * ipb;
        pa = cmake((A.re - a * pa.re) * ipa, (A.im - a * pa.im) * ipa);
        pb = cmake((B.re - a * pb.re) * ipb, (B.im - a * pb.im) * ipb);
        Z.cpw[((size_t)k * npairs + pairidx) * 2] = cpa;
        Z.cpw[((size_t)k * npairs + pairidx) * 2 + 1] = cpb;
        if (self) S[i1] = cmake(pa.re, pb.re);
        else { S[i1] = pa; S[i2] = pb; }
    }
    cplx xa = cmake(0, 0), xb = cmake(0, 0);
    for (int k = nz - 1; k >= 0; k--) {
        size_t i1 = zidx(Z, k, r1, slot), i2 = zidx(Z, k, r2, slot);
        cplx da, db;
        if (self) { cplx t = S[i1]; da = cmake(t.re, 0.0); db = cmake(t.im, 0.0); }
        else { da = S[i1]; db = S[i2]; }
        double ca = Z.cpw[((size_t)k * npairs + pairidx) * 2], cb = Z.cpw[((size_t)k * npairs + pairidx) * 2 + 1];
        xa = cmake(da.re - ca * xa.re, da.im - ca * xa.im);
        xb = cmake(db.re - cb * xb.re, db.im - cb * xb.im);
        if (gaugeA) xa = cmake(Z.gauge[k], 0.0);
        if (self) S[i1] = cmake(xa.re, xb.re);
        else {
            S[i1] = cmake(xa.re - xb.im, xa.im + xb.re);
            S[i2] = cmake(xa.re + xb.im, -xa.im + xb.re);
        }
        if (gaugeA) xa = cmake(0.0, 0.0);
    }
}

// the (0,0) column: d_k = Re S(k, row 0, slot 0).  Serial definition (R7):
//   F_k = F_{k-1} + d_{k-1} dzc[k-1],  x_0 = 0,  x_k = x_{k-1} + F_k dzm[k],  x -= sum x dzc / sum dzc
FSEI_HD void z_gauge_serial(const ZParams& Z, const double* d, double* x)
{
    double F = 0.0, acc = 0.0, vol = 0.0;
    x[0] = 0.0;
    for (int k = 1; k < Z.nz; k++) {
        F += d[k - 1] * Z.dzc[k - 1];
        x[k] = x[k - 1] + F * Z.dzm[k];
    }
    for (int k = 0; k < Z.nz; k++) { acc += x[k] * Z.dzc[k]; vol += Z.dzc[k]; }
    double mean = acc / vol;
    for (int k = 0; k < Z.nz; k++) x[k] -= mean;
}

}  // namespace fsei
