// zfast.cuh -- step a4 on the fast path: one real tridiagonal system per wavenumber pair and component,
//   a_k x_{k-1} + (-(a_k + c_k) + lambda) x_k + c_k x_{k+1} = d_k
// solved by Thomas' algorithm along z, in place in the spectrum (natural-order layout of
// xfast.cuh / yfast.cuh), and the singular (0,0) column by two prefix sums + volume-weighted zero mean
// (R7, R8).
#pragma once
#include "kernel_env.cuh"
#include "plan_types.cuh"

namespace fsei {

struct ZFast {
    int nxc, ny, nz;
    int ncomp;            // reciprocal-pivot components per column in `ipiv` (1: Re and Im share lambda)
    int bcx, bcy;
    const double* za;     // a_k  (a_0 = 0)
    const double* zcc;    // c_k  (c_{nz-1} = 0)
    const double* lamx;   // [nxc][2]  lambda_x of the Re part, of the Im part, per slot
    const double* lamy;   // [ny]      lambda_y per row (natural order)
    const double* dzc;    // [nz]
    const double* dzm;    // [nz] (dzm[0] unused)
    const double* ipiv;   // [nz][ny][nxc][ncomp] reciprocal pivots (plan time)
    cplx* special;        // [2][nz] solved special columns: (row 0, slot 0) and, on (P,P), (row ny/2, slot 0)
    int ktw;              // twist plane: nz = plain Thomas (pivots eliminated from k = 0 upwards); < nz = twisted
                          // factorisation (fused path, few tiles): planes [0, ktw) from below, planes [ktw, nz) from above
    int cb;               // spectrum / pivot-table layout: 0 = natural, else blocked by tiles of cb slots (xfast.cuh)
    const cplx* special_in;   // fused path: [2][nz] right-hand sides of the special columns (else read from the spectrum)
    double* cpw;          // [8][nz] plan-time factorisation of the special columns: c'_k of component t at [t][k],
                          // reciprocal pivots at [4 + t][k]   (t = 2 col + comp; k_z_special_factor)
    int s0 = 0;           // pencil view (slab.py): local slot s is global slot s + s0 (lamx already points at slot s0)
    // peer-store exchange (slab.py): when npeer > 0 the solved column does not go back into the pencil but straight into the
    // slab spectra of the ranks that own the planes: (k, row, slot) -> slab_base[d][((k - slab_k0[d]) ny + row) nxc_full + s0 + slot]
    int npeer = 0, nxc_full = 0;
    cplx* slab_base[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int slab_k0[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
};

FSEI_HD size_t zf_idx(const ZFast& Z, int k, int row, int slot);
// final store of a solved element: the pencil itself, or (peer-store exchange) the slab spectrum of the plane's owner
FSEI_HD void zf_store_out(const ZFast& Z, cplx* S, int k, int row, int slot, cplx v)
{
    if (Z.npeer == 0) { S[zf_idx(Z, k, row, slot)] = v; return; }
    int d = 0;
    while (d + 1 < Z.npeer && k >= Z.slab_k0[d + 1]) d++;
    Z.slab_base[d][((size_t)(k - Z.slab_k0[d]) * Z.ny + row) * Z.nxc_full + Z.s0 + slot] = v;
}

FSEI_HD size_t zf_idx(const ZFast& Z, int k, int row, int slot)
{
    if (Z.cb == 0) return ((size_t)k * Z.ny + row) * Z.nxc + slot;
    return (((size_t)(slot / Z.cb) * Z.nz + k) * Z.ny + row) * Z.cb + slot % Z.cb;
}

// lambda of component comp (0 = Re, 1 = Im) of column (row, slot).  Periodic y: columns that the y-forward
// kernel split (yfast.cuh) hold A^(ky) in rows 1..ny/2-1 and B^(ky) in rows ny-ky, both parts of a row
// belonging to the same x-sequence.
FSEI_HD double z_lambda(const ZFast& Z, int row, int slot, int comp)
{
    int cx = comp;
    if (Z.bcy == BC_PERIODIC && (slot + Z.s0 == 0 || Z.bcx == BC_NEUMANN)) {
        const int h = Z.ny >> 1;
        if (row != 0 && row != h) cx = (row < h) ? 0 : 1;
    }
    return Z.lamx[2 * slot + cx] + Z.lamy[row];
}

// special columns: index into Z.special (or -1) and the mask of components taken from there.
// (P,P): the table has one component per column, so the two columns whose parts differ in lambda --
// (row 0, slot 0) = (gauge, (N_x, 0)) and (row ny/2, slot 0) -- are solved by k_z_special entirely;
// otherwise only the gauge component (row 0, slot 0, Re) is.
FSEI_HD int z_special(const ZFast& Z, int row, int slot, int& mask)
{
    mask = 0;
    if (slot + Z.s0 != 0) return -1;
    const bool pp = (Z.bcx == BC_PERIODIC && Z.bcy == BC_PERIODIC);
    if (row == 0) { mask = pp ? 3 : 1; return 0; }
    if (pp && row == (Z.ny >> 1)) { mask = 3; return 1; }
    return -1;
}

// plan time: reciprocal pivots of one component of one column.  Planes [0, ktw): piv_k = b_k - a_k (c_{k-1} / piv_{k-1});
// planes [ktw, nz) (twisted): piv_k = b_k - c_k (a_{k+1} / piv_{k+1}), eliminated from the top wall downwards.
FSEI_HD void zf_factor_column(const ZFast& Z, double* ipiv, int row, int slot, int comp)
{
    int mask; z_special(Z, row, slot, mask);
    const bool zero_it = (Z.ncomp == 1) ? (mask != 0) : ((mask >> comp) & 1);
    const double lam = z_lambda(Z, row, slot, comp);
    double cp = 0.0;
    for (int k = 0; k < Z.ktw; k++) {
        double a = Z.za[k], c = Z.zcc[k];
        double piv = (-(a + c) + lam) - a * cp;
        double ip = zero_it ? 0.0 : 1.0 / piv;
        ipiv[zf_idx(Z, k, row, slot) * Z.ncomp + comp] = ip;
        cp = c * ip;
    }
    double ap = 0.0;
    for (int k = Z.nz - 1; k >= Z.ktw; k--) {
        double a = Z.za[k], c = Z.zcc[k];
        double piv = (-(a + c) + lam) - c * ap;
        double iq = zero_it ? 0.0 : 1.0 / piv;
        ipiv[zf_idx(Z, k, row, slot) * Z.ncomp + comp] = iq;
        ap = a * iq;
    }
}

// one thread per column: forward elimination then back substitution, in place (two passes over the column).
// Planes are taken in chunks of ZSW: all loads of a chunk are issued before its dependent chain and its stores (the
// compiler cannot move the loads of plane k+1 over the store of plane k, and a chain of exposed L2 latencies is what
// this kernel would otherwise be).
#define FSEI_ZSW 8
template <int NCOMP>
FSEI_HD void zf_sweep_column(const ZFast& Z, cplx* S, int row, int slot)
{
    const int nz = Z.nz;
    int mask; const int sp = z_special(Z, row, slot, mask);
    cplx prev = cmake(0.0, 0.0);
    for (int k0 = 0; k0 < nz; k0 += FSEI_ZSW) {
        cplx d[FSEI_ZSW]; double ip[FSEI_ZSW][2], a[FSEI_ZSW];
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) {
            const int k = (k0 + j < nz) ? k0 + j : nz - 1;
            const size_t i = zf_idx(Z, k, row, slot);
            d[j] = S[i]; ip[j][0] = Z.ipiv[i * NCOMP]; ip[j][1] = Z.ipiv[i * NCOMP + (NCOMP - 1)]; a[j] = Z.za[k];
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) {
            if (k0 + j < nz) { prev = cmake((d[j].re - a[j] * prev.re) * ip[j][0], (d[j].im - a[j] * prev.im) * ip[j][1]); d[j] = prev; }
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) if (k0 + j < nz) S[zf_idx(Z, k0 + j, row, slot)] = d[j];
    }
    cplx next = cmake(0.0, 0.0);
    for (int k1 = nz - 1; k1 >= 0; k1 -= FSEI_ZSW) {
        cplx d[FSEI_ZSW], sv[FSEI_ZSW]; double ip[FSEI_ZSW][2], c[FSEI_ZSW];
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) {
            const int k = (k1 - j >= 0) ? k1 - j : 0;
            const size_t i = zf_idx(Z, k, row, slot);
            d[j] = S[i]; ip[j][0] = Z.ipiv[i * NCOMP]; ip[j][1] = Z.ipiv[i * NCOMP + (NCOMP - 1)]; c[j] = Z.zcc[k];
            sv[j] = (sp >= 0) ? Z.special[(size_t)sp * nz + k] : cmake(0.0, 0.0);
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) {
            if (k1 - j >= 0) {
                next = cmake(d[j].re - (c[j] * ip[j][0]) * next.re, d[j].im - (c[j] * ip[j][1]) * next.im);
                cplx o = next;
                if (sp >= 0) {
                    if (mask & 1) o.re = sv[j].re;
                    if (mask & 2) o.im = sv[j].im;
                }
                d[j] = o;
            }
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZSW; j++) if (k1 - j >= 0) zf_store_out(Z, S, k1 - j, row, slot, d[j]);
    }
}

// the (0,0) component: serial definition (R7):
//   F_k = F_{k-1} + d_{k-1} dzc[k-1],  x_0 = 0,  x_k = x_{k-1} + F_k dzm[k],  x -= sum x dzc / sum dzc
// d, x: arrays of cplx; comp selects the part (stride 2 doubles).  Chunks of ZCH planes: all loads of a chunk are
// issued before its dependent chain (the compiler cannot reorder loads over the stores of x itself).
#define FSEI_ZCH 16
// Returns the volume-weighted mean; the caller subtracts it from x (in parallel).
FSEI_HD double zf_gauge_serial(const ZFast& Z, const double* FSEI_RESTRICT d, double* FSEI_RESTRICT x,
                               const double* FSEI_RESTRICT dzc, const double* FSEI_RESTRICT dzm)
{
    const int nz = Z.nz;
    double F = 0.0, acc = 0.0, vol = 0.0, xp = 0.0;
    x[0] = 0.0;
    for (int k0 = 1; k0 < nz; k0 += FSEI_ZCH) {
        double dd[FSEI_ZCH], wc[FSEI_ZCH], wm[FSEI_ZCH];
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) {
            const int k = (k0 + j < nz) ? k0 + j : nz - 1;
            dd[j] = d[2 * (k - 1)]; wc[j] = dzc[k - 1]; wm[j] = dzm[k];
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) {
            if (k0 + j < nz) { F += dd[j] * wc[j]; xp = xp + F * wm[j]; dd[j] = xp; }
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k0 + j < nz) x[2 * (k0 + j)] = dd[j];
    }
    for (int k0 = 0; k0 < nz; k0 += FSEI_ZCH) {
        double xx[FSEI_ZCH], wc[FSEI_ZCH];
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) {
            const int k = (k0 + j < nz) ? k0 + j : nz - 1;
            xx[j] = x[2 * k]; wc[j] = dzc[k];
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k0 + j < nz) { acc += xx[j] * wc[j]; vol += wc[j]; }
    }
    return acc / vol;
}

// plan time: factorisation of one component of a special column (same recurrence as zf_factor_column)
FSEI_HD void zf_special_factor(const ZFast& Z, double lam, double* cp, double* ip)
{
    double cprev = 0.0;
    for (int k = 0; k < Z.nz; k++) {
        double a = Z.za[k], c = Z.zcc[k];
        double r = 1.0 / ((-(a + c) + lam) - a * cprev);
        ip[k] = r; cprev = c * r; cp[k] = cprev;
    }
}

// Thomas on one component of a column held in shared memory, factorisation from the plan's tables
FSEI_HD void zf_thomas_serial(const ZFast& Z, const double* FSEI_RESTRICT d, double* FSEI_RESTRICT x,
                              const double* FSEI_RESTRICT cp, const double* FSEI_RESTRICT ip, const double* FSEI_RESTRICT za)
{
    const int nz = Z.nz;
    double prev = 0.0;
    for (int k0 = 0; k0 < nz; k0 += FSEI_ZCH) {
        double dd[FSEI_ZCH], aa[FSEI_ZCH], ii[FSEI_ZCH];
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) {
            const int k = (k0 + j < nz) ? k0 + j : nz - 1;
            dd[j] = d[2 * k]; aa[j] = za[k]; ii[j] = ip[k];
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k0 + j < nz) { prev = (dd[j] - aa[j] * prev) * ii[j]; dd[j] = prev; }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k0 + j < nz) x[2 * (k0 + j)] = dd[j];
    }
    double next = 0.0;
    for (int k1 = nz - 1; k1 >= 0; k1 -= FSEI_ZCH) {
        double xx[FSEI_ZCH], cc[FSEI_ZCH];
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) {
            const int k = (k1 - j >= 0) ? k1 - j : 0;
            xx[j] = x[2 * k]; cc[j] = cp[k];
        }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k1 - j >= 0) { next = xx[j] - cc[j] * next; xx[j] = next; }
#pragma unroll
        for (int j = 0; j < FSEI_ZCH; j++) if (k1 - j >= 0) x[2 * (k1 - j)] = xx[j];
    }
}

// dynamic shared memory of k_z_special: the columns (4 nz cplx + 16) and, when `staged`, the tables of the serial chains
// (dzc, dzm, za and the 8 rows of cpw: 11 nz doubles) -- a chain that reads its coefficients from L2 spends most of its
// time waiting for them
FSEI_HD size_t z_special_smem(int nz, bool staged) { return 4 * sizeof(cplx) * (size_t)nz + 16 + (staged ? 11 * sizeof(double) * (size_t)nz : 0); }
FSEI_HD bool z_special_staged(int nz) { return z_special_smem(nz, true) <= 200 * 1024; }

// grid 1, block 128: gathers the special columns, solves them (one thread per component), leaves them in Z.special
FSEI_GLOBAL(128, 1) k_z_special(ZFast Z, const cplx* spec, int staged)
{
    FSEI_DYN_SMEM(smraw);
    cplx* d = reinterpret_cast<cplx*>(smraw);            // [2][nz]
    cplx* x = d + 2 * Z.nz;                              // [2][nz]
    double* mean = reinterpret_cast<double*>(x + 2 * Z.nz);
    double* tab = mean + 2;                              // [11][nz] when staged
    const int nz = Z.nz, tid = threadIdx.x;
    const bool pp = (Z.bcx == BC_PERIODIC && Z.bcy == BC_PERIODIC);
    const int ncol = pp ? 2 : 1;
    for (int i = tid; i < ncol * nz; i += 128) {
        int col = i / nz, k = i - col * nz;
        d[i] = Z.special_in ? Z.special_in[i] : spec[zf_idx(Z, k, col == 0 ? 0 : (Z.ny >> 1), 0)];
        x[i] = cmake(0.0, 0.0);
    }
    const double *dzc = Z.dzc, *dzm = Z.dzm, *za = Z.za, *cpw = Z.cpw;
    if (staged) {
        for (int i = tid; i < nz; i += 128) { tab[i] = Z.dzc[i]; tab[nz + i] = Z.dzm[i]; tab[2 * nz + i] = Z.za[i]; }
        if (pp) for (int i = tid; i < 8 * nz; i += 128) tab[3 * nz + i] = Z.cpw[i];
        dzc = tab; dzm = tab + nz; za = tab + 2 * nz; cpw = tab + 3 * nz;
    }
    FSEI_SYNC();
    if ((tid & 31) == 0 && (tid >> 5) < 2 * ncol) {          // component t on lane 0 of warp t: the four chains run side by side
        const int t = tid >> 5, col = t >> 1, comp = t & 1;
        const double* dd = reinterpret_cast<const double*>(d + col * nz) + comp;
        double* xx = reinterpret_cast<double*>(x + col * nz) + comp;
        if (t == 0) mean[0] = zf_gauge_serial(Z, dd, xx, dzc, dzm);
        else if (pp) zf_thomas_serial(Z, dd, xx, cpw + (size_t)t * nz, cpw + (size_t)(4 + t) * nz, za);
    }
    FSEI_SYNC();
    const double gm = mean[0];
    for (int i = tid; i < ncol * nz; i += 128) {
        cplx v = x[i];
        if (i < nz) v.re -= gm;                              // gauge: volume-weighted zero mean of the (0,0) component
        Z.special[i] = v;
    }
}

// plan time.  grid 1, block 32: tables of the special Thomas components (threads 1..3 on (P,P))
FSEI_GLOBAL(32, 1) k_z_special_factor(ZFast Z)
{
    const int tid = threadIdx.x;
    const bool pp = (Z.bcx == BC_PERIODIC && Z.bcy == BC_PERIODIC);
    if (!pp || tid < 1 || tid > 3) return;
    const int col = tid >> 1, comp = tid & 1;
    zf_special_factor(Z, z_lambda(Z, col == 0 ? 0 : (Z.ny >> 1), 0, comp), Z.cpw + (size_t)tid * Z.nz, Z.cpw + (size_t)(4 + tid) * Z.nz);
}

// plan time.  grid ceil(ny nxc ncomp / 256), block 256
FSEI_GLOBAL(256, 1) k_zf_factor(ZFast Z, double* ipiv)
{
    size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;
    size_t n = (size_t)Z.ny * Z.nxc * Z.ncomp;
    if (t >= n) return;
    int comp = (int)(t % Z.ncomp); size_t r = t / Z.ncomp; int slot = (int)(r % Z.nxc), row = (int)(r / Z.nxc);
    zf_factor_column(Z, ipiv, row, slot, comp);
}

// Short columns (nz <= 32): parallel cyclic reduction with the column spread over the lanes of ONE warp (lane = k).
// Step s = 1, 2, 4, 8, 16 eliminates the couplings to k - s and k + s:
//   al = -a_k / b_{k-s},  ga = -c_k / b_{k+s},
//   a_k <- al a_{k-s},  c_k <- ga c_{k+s},  b_k <- b_k + al c_{k-s} + ga a_{k+s},  d_k <- d_k + al d_{k-s} + ga d_{k+s}
// (rows outside [0, nz) are identity rows), after which x_k = d_k / b_k.  No factorisation table, log2(32) dependent
// steps instead of 2 nz.  Re and Im are two systems (same a, c; b differs when the parts have different lambda).
// The diagonal is carried as its excess over the off-diagonals, r_k = a_k + b_k + c_k (= lambda <= 0 at the start):
// r obeys the same recurrence as d, r_k <- r_k + al r_{k-s} + ga r_{k+s}, in which every term has the same sign, and
// b_k = r_k - (a_k + c_k) is again a sum of like-signed terms -- so the reduction never subtracts nearly equal numbers
// (updating b directly loses the 1e-5-relative lambda of the low modes to cancellation: 3x the Thomas residual).
struct PcrRow { double a, r, c, d; };
FSEI_DEV void pcr_reduce(PcrRow& w, int lane)
{
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        const bool lo = lane - s >= 0, hi = lane + s < 32;
        const double am = lane_up(w.a, s), rm = lane_up(w.r, s), cm = lane_up(w.c, s), dm = lane_up(w.d, s);
        const double ap = lane_down(w.a, s), rp = lane_down(w.r, s), cp = lane_down(w.c, s), dp = lane_down(w.d, s);
        const double al = lo ? -w.a / (rm - (am + cm)) : 0.0, ga = hi ? -w.c / (rp - (ap + cp)) : 0.0;
        w.r = w.r + al * (lo ? rm : 0.0) + ga * (hi ? rp : 0.0);
        w.d = w.d + al * (lo ? dm : 0.0) + ga * (hi ? dp : 0.0);
        w.a = al * (lo ? am : 0.0);
        w.c = ga * (hi ? cp : 0.0);
    }
}

// grid ceil(32 ny nxc / 128), block 128: warp w of the grid owns column (row w / nxc, slot w % nxc).  nz <= 32.
// Every thread runs the whole kernel (uniform control flow: the host harness emulates the shuffles with barriers).
FSEI_GLOBAL(128, 1) k_zf_pcr(ZFast Z, cplx* spec)
{
    const size_t t = (size_t)blockIdx.x * 128 + threadIdx.x;
    const int lane = (int)(t & 31);
    const size_t w = t >> 5, ncol = (size_t)Z.nxc * Z.ny;
    const bool col_ok = w < ncol;
    const int slot = col_ok ? (int)(w % Z.nxc) : 0, row = col_ok ? (int)(w / Z.nxc) : 0;
    const bool on = col_ok && lane < Z.nz;
    int mask; const int sp = z_special(Z, row, slot, mask);
    const size_t i = on ? zf_idx(Z, lane, row, slot) : 0;
    const cplx d = on ? spec[i] : cmake(0.0, 0.0);
    const double a = on ? Z.za[lane] : 0.0, c = on ? Z.zcc[lane] : 0.0;
    PcrRow re, im;
    re.a = a; re.c = c; re.d = d.re; re.r = on ? z_lambda(Z, row, slot, 0) : 1.0;
    im.a = a; im.c = c; im.d = d.im; im.r = on ? z_lambda(Z, row, slot, 1) : 1.0;
    pcr_reduce(re, lane);
    pcr_reduce(im, lane);
    if (on) {
        cplx o = cmake(re.d / (re.r - (re.a + re.c)), im.d / (im.r - (im.a + im.c)));
        if (sp >= 0) {                                      // singular / separately solved parts: selected, not mixed
            const cplx s = Z.special[(size_t)sp * Z.nz + lane];
            if (mask & 1) o.re = s.re;
            if (mask & 2) o.im = s.im;
        }
        zf_store_out(Z, spec, lane, row, slot, o);
    }
}

// grid ceil(ny nxc / 128), block 128: slot fastest across the warp (coalesced 16-byte accesses)
template <int NCOMP>
FSEI_GLOBAL(128, 1) k_zf_sweep(ZFast Z, cplx* spec)
{
    size_t t = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (t >= (size_t)Z.nxc * Z.ny) return;
    int slot = (int)(t % Z.nxc), row = (int)(t / Z.nxc);
    zf_sweep_column<NCOMP>(Z, spec, row, slot);
}

}  // namespace fsei
