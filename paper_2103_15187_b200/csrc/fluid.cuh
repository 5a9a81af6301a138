// fluid.cuh -- the two steps that precede the pressure projection in one fluid substep:
//
//   explicit terms (Eq. 3):  H = -div(u u) + f,
//        rhs_q = ((gdt H + rdt Hprev) - adt G p) + 2 beta lap q,   Hprev <- H
//   implicit viscous step:    q += [(1 - beta dxx)(1 - beta dyy)(1 - beta dzz)]^-1 rhs_q
//        "approximate factorization yielding tridiagonal matrices (one for each direction) inverted using Thomas'
//        algorithm with a Sherman-Morrison perturbation in the two periodic dimensions"
//
// Discrete operators: readings V1..V12 of DESIGN.md sec. 3.  The explicit terms are stencils evaluated in IEEE double
// in one fixed order, every operation individually rounded (FSEI_MUL/ADD/SUB), so they match the definition bit for
// bit.  The implicit step here is the GENERIC kernel family (any size, any bc): plan-independent factorisation tables
// built on the device for the beta of the call, one thread per line for the strided directions (y, z: coalesced across
// lines), warp-transposed 32 x 32 tiles for the contiguous x lines.  A periodic line is solved as a BORDERED
// tridiagonal system (the last unknown is the border): one forward and one backward pass, the same arithmetic count
// as Thomas + Sherman-Morrison without the third pass over the line that the rank-one correction needs.
#pragma once
#include "kernel_env.cuh"
#include "stencil.cuh"

namespace fsei {

enum { COMP_U = 0, COMP_V = 1, COMP_W = 2, DIR_X = 0, DIR_Y = 1, DIR_Z = 2 };

// ---------------------------------------------------------------------------------------------------------------
// implicit step: factorisation tables of one (component, direction)
// ---------------------------------------------------------------------------------------------------------------
struct VTab {
    const double* ip;     // [n] reciprocal pivots
    const double* am;     // [n] sub-diagonal a_m of (1 - beta d2)
    const double* cp;     // [n] c_m / piv_m
    const double* wc;     // [n] border column after elimination (periodic lines)
    const double* er;     // [n] border row multipliers (periodic lines)
    const double* ipl;    // [1] reciprocal pivot of the border unknown
    int n, cyclic, fixed0;
};

struct VFactorArgs {
    SParams S;
    double beta;
    double* tab;          // 9 sets x (5 n_max + 1) doubles
    int nmax;
};

FSEI_HD size_t vtab_set_doubles(int nmax) { return (size_t)5 * nmax + 8; }

// rows of d2 of component comp along dir (reading V3-V6): lo, di, up at row m; *fixed: row m is a wall face
FSEI_HD void visc_row(const SParams& S, int comp, int dir, int m, double& lo, double& di, double& up, bool& fixed)
{
    fixed = false;
    if (dir != DIR_Z) {
        const int n = dir == DIR_X ? S.nx : S.ny;
        const int bc = dir == DIR_X ? S.bcx : S.bcy;
        const double r = dir == DIR_X ? S.rdx : S.rdy, r2 = r * r;
        lo = r2; up = r2; di = -2.0 * r2;
        if (bc == BC_PERIODIC) return;
        const bool normal = (dir == DIR_X && comp == COMP_U) || (dir == DIR_Y && comp == COMP_V);
        if (normal) {
            if (m == 0) { fixed = true; lo = up = di = 0.0; }
            if (m == 1) lo = 0.0;
            if (m == n - 1) up = 0.0;
        } else {
            if (m == 0) { lo = 0.0; di = -3.0 * r2; }
            if (m == n - 1) { up = 0.0; di = (n == 1) ? -4.0 * r2 : -3.0 * r2; }
        }
        return;
    }
    const int nz = S.nz;
    if (comp != COMP_W) {
        const double rc = S.rdzc[m];
        lo = (m > 0) ? S.rdzm[m] * rc : 0.0;
        up = (m + 1 < nz) ? S.rdzm[m + 1] * rc : 0.0;
        const double wl = (m == 0) ? 2.0 * rc * rc : 0.0, wu = (m == nz - 1) ? 2.0 * rc * rc : 0.0;
        di = -(lo + up + wl + wu);
    } else {
        if (m == 0) { fixed = true; lo = up = di = 0.0; return; }
        const double l = S.rdzc[m - 1] * S.rdzm[m], u = S.rdzc[m] * S.rdzm[m];
        lo = (m > 1) ? l : 0.0; up = (m + 1 < nz) ? u : 0.0; di = -(l + u);
    }
}

// one thread per (component, direction): the serial factorisation recurrences (n <= 8192 steps, once per call)
FSEI_GLOBAL(32, 1) k_visc_factor(VFactorArgs A)
{
    if (threadIdx.x != 0) return;
    const int set = blockIdx.x, comp = set / 3, dir = set % 3;
    const SParams& S = A.S;
    const int n = dir == DIR_X ? S.nx : (dir == DIR_Y ? S.ny : S.nz);
    const bool cyc = (dir == DIR_X && S.bcx == BC_PERIODIC) || (dir == DIR_Y && S.bcy == BC_PERIODIC);
    double* t = A.tab + (size_t)set * vtab_set_doubles(A.nmax);
    double *ip = t, *am = t + A.nmax, *cp = t + 2 * (size_t)A.nmax, *wc = t + 3 * (size_t)A.nmax, *er = t + 4 * (size_t)A.nmax;
    double* ipl = t + 5 * (size_t)A.nmax;
    const double beta = A.beta;
    const int nn = cyc ? n - 1 : n;          // rows of the tridiagonal core
    double lo, di, up; bool fx;
    // border data of a periodic line: a_0 couples row 0 to the border unknown, c_{n-2} row n-2; border row: c_{n-1} x_0 + a_{n-1} x_{n-2} + b x_{n-1}
    double cpm = 0.0, wcm = 0.0, e = 0.0, bl = 0.0, a_last = 0.0;
    if (cyc) { visc_row(S, comp, dir, n - 1, lo, di, up, fx); e = -beta * up; a_last = -beta * lo; bl = 1.0 - beta * di; }
    for (int m = 0; m < nn; m++) {
        visc_row(S, comp, dir, m, lo, di, up, fx);
        double a = fx ? 0.0 : -beta * lo, b = fx ? 1.0 : 1.0 - beta * di, c = fx ? 0.0 : -beta * up;
        double wsrc = 0.0;                   // entry of this row in the border column before elimination
        if (cyc && m == 0) { wsrc = a; a = 0.0; }
        if (cyc && m == nn - 1) { wsrc += c; c = 0.0; }
        const double piv = b - a * cpm, r = 1.0 / piv;
        cpm = c * r;
        wcm = (wsrc - a * wcm) * r;
        ip[m] = r; am[m] = a; cp[m] = cpm; wc[m] = wcm;
        if (cyc) {
            const double em = (m == nn - 1) ? e + a_last : e;
            er[m] = em;
            bl -= em * wcm;
            e = -e * cpm;
        } else er[m] = 0.0;
    }
    if (cyc) { ip[n - 1] = 0.0; am[n - 1] = 0.0; cp[n - 1] = 0.0; wc[n - 1] = 0.0; er[n - 1] = 0.0; ipl[0] = 1.0 / bl; }
    else ipl[0] = 0.0;
}

// ---------------------------------------------------------------------------------------------------------------
// strided directions (y, z): one thread per line, neighbouring threads on neighbouring x -> coalesced
//   line of thread t: i = t % ni, o = t / ni, elements at o*outer_stride + i + m*stride
//   LAST: the result is added to q instead of being written back (the last of the three sweeps)
// ---------------------------------------------------------------------------------------------------------------
template <bool CYC, bool LAST>
FSEI_GLOBAL(128, 1) k_visc_sweep_strided(VTab T, double* __restrict__ f, double* __restrict__ q, int ni, size_t stride,
                                         size_t outer_stride, long nlines)
{
    const long t = (long)blockIdx.x * 128 + threadIdx.x;
    if (t >= nlines) return;
    const size_t base = (size_t)(t / ni) * outer_stride + (size_t)(t % ni);
    const int n = T.n, nn = CYC ? n - 1 : n;
    double dp = 0.0, g = 0.0;
#pragma unroll 4
    for (int m = 0; m < nn; m++) {
        double d = f[base + m * stride];
        if (m == 0 && T.fixed0) d = 0.0;
        dp = (d - T.am[m] * dp) * T.ip[m];
        if (CYC) g += T.er[m] * dp;
        f[base + m * stride] = dp;
    }
    double xl = 0.0, xn = 0.0;
    if (CYC) {
        xl = (f[base + (size_t)(n - 1) * stride] - g) * T.ipl[0];
        if (LAST) q[base + (size_t)(n - 1) * stride] += xl; else f[base + (size_t)(n - 1) * stride] = xl;
    }
#pragma unroll 4
    for (int m = nn - 1; m >= 0; m--) {
        double x = f[base + m * stride] - T.cp[m] * xn;
        if (CYC) x -= T.wc[m] * xl;
        if (LAST) q[base + m * stride] += x; else f[base + m * stride] = x;
        xn = x;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// contiguous direction (x): a warp owns 32 consecutive lines (lane = line) and walks along x in chunks of 32
// columns: coalesced 256-byte row reads into a warp-private 32 x 33 tile, each lane eliminates its own row of the
// tile, coalesced write back.  4 warps per CTA.
// ---------------------------------------------------------------------------------------------------------------
template <bool CYC, bool LAST>
FSEI_GLOBAL(128, 1) k_visc_sweep_x(VTab T, double* __restrict__ f, double* __restrict__ q, long nlines)
{
    __shared__ double tile_all[4][32 * 33];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double* tile = tile_all[wid];
    const long l0 = ((long)blockIdx.x * 4 + wid) * 32;
    if (l0 >= nlines) return;
    const int nl = (int)((nlines - l0 < 32) ? nlines - l0 : 32);
    const int n = T.n, nn = CYC ? n - 1 : n;
    double* fb = f + (size_t)l0 * n;
    double* qb = LAST ? q + (size_t)l0 * n : nullptr;
    double dp = 0.0, g = 0.0;
    for (int c0 = 0; c0 < n; c0 += 32) {
        const int nc = (n - c0 < 32) ? n - c0 : 32;
        for (int r = 0; r < nl; r++) if (lane < nc) tile[r * 33 + lane] = fb[(size_t)r * n + c0 + lane];
        __syncwarp();
        if (lane < nl)
            for (int c = 0; c < nc; c++) {
                const int m = c0 + c;
                if (m >= nn) break;
                double d = tile[lane * 33 + c];
                if (m == 0 && T.fixed0) d = 0.0;
                dp = (d - T.am[m] * dp) * T.ip[m];
                if (CYC) g += T.er[m] * dp;
                tile[lane * 33 + c] = dp;
            }
        __syncwarp();
        for (int r = 0; r < nl; r++) if (lane < nc) fb[(size_t)r * n + c0 + lane] = tile[r * 33 + lane];
        __syncwarp();
    }
    double xl = 0.0, xn = 0.0;
    if (CYC && lane < nl) xl = (fb[(size_t)lane * n + n - 1] - g) * T.ipl[0];      // the border entry was copied through unchanged
    const int cl = ((n - 1) / 32) * 32;
    for (int c0 = cl; c0 >= 0; c0 -= 32) {
        const int nc = (n - c0 < 32) ? n - c0 : 32;
        for (int r = 0; r < nl; r++) if (lane < nc) tile[r * 33 + lane] = fb[(size_t)r * n + c0 + lane];
        __syncwarp();
        if (lane < nl)
            for (int c = nc - 1; c >= 0; c--) {
                const int m = c0 + c;
                double x;
                if (CYC && m == n - 1) x = xl;
                else {
                    x = tile[lane * 33 + c] - T.cp[m] * xn;
                    if (CYC) x -= T.wc[m] * xl;
                    xn = x;
                }
                tile[lane * 33 + c] = x;
            }
        __syncwarp();
        for (int r = 0; r < nl; r++)
            if (lane < nc) {
                const size_t a = (size_t)r * n + c0 + lane;
                if (LAST) qb[a] += tile[r * 33 + lane]; else fb[a] = tile[r * 33 + lane];
            }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// explicit terms: one thread per cell, every operation individually rounded in the order of the definition
// ---------------------------------------------------------------------------------------------------------------
template <int COMP> FSEI_DEV double vfetch(const SParams& S, const double* __restrict__ q, int i, int j, int k)
{
    bool neg = false;
    if (i < 0 || i >= S.nx) {
        if (S.bcx == BC_PERIODIC) i = i < 0 ? i + S.nx : i - S.nx;
        else if (COMP == COMP_U) return 0.0;
        else { i = i < 0 ? 0 : S.nx - 1; neg = !neg; }
    }
    if (j < 0 || j >= S.ny) {
        if (S.bcy == BC_PERIODIC) j = j < 0 ? j + S.ny : j - S.ny;
        else if (COMP == COMP_V) return 0.0;
        else { j = j < 0 ? 0 : S.ny - 1; neg = !neg; }
    }
    if (k < 0 || k >= S.nz) {
        if (COMP == COMP_W) return 0.0;
        k = k < 0 ? 0 : S.nz - 1; neg = !neg;
    }
    const double val = q[sidx(S, i, j, k)];
    return neg ? -val : val;
}

FSEI_DEV double avg2(double a, double b) { return FSEI_MUL(0.5, FSEI_ADD(a, b)); }
FSEI_DEV bool xwall(const SParams& S, int i) { return S.bcx != BC_PERIODIC && (i <= 0 || i >= S.nx); }
FSEI_DEV bool ywall(const SParams& S, int j) { return S.bcy != BC_PERIODIC && (j <= 0 || j >= S.ny); }
FSEI_DEV bool zwall(const SParams& S, int k) { return k <= 0 || k >= S.nz; }

template <int COMP> FSEI_DEV bool wall_row(const SParams& S, int i, int j, int k)
{
    return (COMP == COMP_U && S.bcx != BC_PERIODIC && i == 0) || (COMP == COMP_V && S.bcy != BC_PERIODIC && j == 0) ||
           (COMP == COMP_W && k == 0);
}

// lap q = (dxx q + dyy q) + dzz q, second differences as differences of face gradients
template <int COMP> FSEI_DEV double vel_lap(const SParams& S, const double* __restrict__ q, int i, int j, int k)
{
    const double c0 = q[sidx(S, i, j, k)];
    double gp = FSEI_MUL(FSEI_SUB(vfetch<COMP>(S, q, i + 1, j, k), c0), S.rdx), gm = FSEI_MUL(FSEI_SUB(c0, vfetch<COMP>(S, q, i - 1, j, k)), S.rdx);
    const double dxx = FSEI_MUL(FSEI_SUB(gp, gm), S.rdx);
    gp = FSEI_MUL(FSEI_SUB(vfetch<COMP>(S, q, i, j + 1, k), c0), S.rdy); gm = FSEI_MUL(FSEI_SUB(c0, vfetch<COMP>(S, q, i, j - 1, k)), S.rdy);
    const double dyy = FSEI_MUL(FSEI_SUB(gp, gm), S.rdy);
    double dzz;
    if (COMP != COMP_W) {
        const double rc = S.rdzc[k];
        gp = (k + 1 < S.nz) ? FSEI_MUL(FSEI_SUB(q[sidx(S, i, j, k + 1)], c0), S.rdzm[k + 1]) : FSEI_MUL(FSEI_SUB(0.0, c0), FSEI_MUL(2.0, rc));
        gm = (k > 0) ? FSEI_MUL(FSEI_SUB(c0, q[sidx(S, i, j, k - 1)]), S.rdzm[k]) : FSEI_MUL(FSEI_SUB(c0, 0.0), FSEI_MUL(2.0, rc));
        dzz = FSEI_MUL(FSEI_SUB(gp, gm), rc);
    } else {
        const double wp = (k + 1 < S.nz) ? q[sidx(S, i, j, k + 1)] : 0.0;
        gp = FSEI_MUL(FSEI_SUB(wp, c0), S.rdzc[k]); gm = FSEI_MUL(FSEI_SUB(c0, q[sidx(S, i, j, k - 1)]), S.rdzc[k - 1]);
        dzz = FSEI_MUL(FSEI_SUB(gp, gm), S.rdzm[k]);
    }
    return FSEI_ADD(FSEI_ADD(dxx, dyy), dzz);
}

FSEI_DEV double neg3(double fx, double fy, double fz) { return -FSEI_ADD(FSEI_ADD(fx, fy), fz); }

FSEI_DEV double conv_u(const SParams& S, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w, int i, int j, int k)
{
    const double c0 = u[sidx(S, i, j, k)];
    const double ucp = avg2(c0, vfetch<COMP_U>(S, u, i + 1, j, k)), ucm = avg2(vfetch<COMP_U>(S, u, i - 1, j, k), c0);
    const double fx = FSEI_MUL(FSEI_SUB(FSEI_MUL(ucp, ucp), FSEI_MUL(ucm, ucm)), S.rdx);
    const double fa = ywall(S, j + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_U>(S, u, i, j + 1, k)), avg2(vfetch<COMP_V>(S, v, i - 1, j + 1, k), vfetch<COMP_V>(S, v, i, j + 1, k)));
    const double fb = ywall(S, j) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_U>(S, u, i, j - 1, k), c0), avg2(vfetch<COMP_V>(S, v, i - 1, j, k), vfetch<COMP_V>(S, v, i, j, k)));
    const double fy = FSEI_MUL(FSEI_SUB(fa, fb), S.rdy);
    const double ga = zwall(S, k + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_U>(S, u, i, j, k + 1)), avg2(vfetch<COMP_W>(S, w, i - 1, j, k + 1), vfetch<COMP_W>(S, w, i, j, k + 1)));
    const double gb = zwall(S, k) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_U>(S, u, i, j, k - 1), c0), avg2(vfetch<COMP_W>(S, w, i - 1, j, k), vfetch<COMP_W>(S, w, i, j, k)));
    const double fz = FSEI_MUL(FSEI_SUB(ga, gb), S.rdzc[k]);
    return neg3(fx, fy, fz);
}
FSEI_DEV double conv_v(const SParams& S, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w, int i, int j, int k)
{
    const double c0 = v[sidx(S, i, j, k)];
    const double fa = xwall(S, i + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_V>(S, v, i + 1, j, k)), avg2(vfetch<COMP_U>(S, u, i + 1, j - 1, k), vfetch<COMP_U>(S, u, i + 1, j, k)));
    const double fb = xwall(S, i) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_V>(S, v, i - 1, j, k), c0), avg2(vfetch<COMP_U>(S, u, i, j - 1, k), vfetch<COMP_U>(S, u, i, j, k)));
    const double fx = FSEI_MUL(FSEI_SUB(fa, fb), S.rdx);
    const double vcp = avg2(c0, vfetch<COMP_V>(S, v, i, j + 1, k)), vcm = avg2(vfetch<COMP_V>(S, v, i, j - 1, k), c0);
    const double fy = FSEI_MUL(FSEI_SUB(FSEI_MUL(vcp, vcp), FSEI_MUL(vcm, vcm)), S.rdy);
    const double ga = zwall(S, k + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_V>(S, v, i, j, k + 1)), avg2(vfetch<COMP_W>(S, w, i, j - 1, k + 1), vfetch<COMP_W>(S, w, i, j, k + 1)));
    const double gb = zwall(S, k) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_V>(S, v, i, j, k - 1), c0), avg2(vfetch<COMP_W>(S, w, i, j - 1, k), vfetch<COMP_W>(S, w, i, j, k)));
    const double fz = FSEI_MUL(FSEI_SUB(ga, gb), S.rdzc[k]);
    return neg3(fx, fy, fz);
}
FSEI_DEV double conv_w(const SParams& S, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w, int i, int j, int k)
{
    const double c0 = w[sidx(S, i, j, k)];
    const double fa = xwall(S, i + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_W>(S, w, i + 1, j, k)), avg2(vfetch<COMP_U>(S, u, i + 1, j, k - 1), vfetch<COMP_U>(S, u, i + 1, j, k)));
    const double fb = xwall(S, i) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_W>(S, w, i - 1, j, k), c0), avg2(vfetch<COMP_U>(S, u, i, j, k - 1), vfetch<COMP_U>(S, u, i, j, k)));
    const double fx = FSEI_MUL(FSEI_SUB(fa, fb), S.rdx);
    const double ga = ywall(S, j + 1) ? 0.0 : FSEI_MUL(avg2(c0, vfetch<COMP_W>(S, w, i, j + 1, k)), avg2(vfetch<COMP_V>(S, v, i, j + 1, k - 1), vfetch<COMP_V>(S, v, i, j + 1, k)));
    const double gb = ywall(S, j) ? 0.0 : FSEI_MUL(avg2(vfetch<COMP_W>(S, w, i, j - 1, k), c0), avg2(vfetch<COMP_V>(S, v, i, j, k - 1), vfetch<COMP_V>(S, v, i, j, k)));
    const double fy = FSEI_MUL(FSEI_SUB(ga, gb), S.rdy);
    const double wcp = avg2(c0, vfetch<COMP_W>(S, w, i, j, k + 1)), wcm = avg2(vfetch<COMP_W>(S, w, i, j, k - 1), c0);
    const double fz = FSEI_MUL(FSEI_SUB(FSEI_MUL(wcp, wcp), FSEI_MUL(wcm, wcm)), S.rdzm[k]);
    return neg3(fx, fy, fz);
}

struct ExplicitArgs {
    SParams S;
    const double *u, *v, *w, *p, *fu, *fv, *fw;     // fu, fv, fw may be null (no body force)
    double *hu, *hv, *hw;                           // in: H of the previous substep, out: H of this one
    double *ru, *rv, *rw;                           // out: right-hand sides of the implicit step
    double gdt, rdt, adt, tb;                       // gamma dt, rho dt, alpha dt, 2 beta
};

FSEI_DEV double rhs_assemble(double H, double Hp, double gp, double lap, const ExplicitArgs& A)
{
    return FSEI_ADD(FSEI_SUB(FSEI_ADD(FSEI_MUL(A.gdt, H), FSEI_MUL(A.rdt, Hp)), FSEI_MUL(A.adt, gp)), FSEI_MUL(A.tb, lap));
}

// grid ceil(nx ny nz / 256), block 256, x fastest
FSEI_GLOBAL(256, 1) k_explicit_terms(ExplicitArgs A)
{
    const SParams& S = A.S;
    const size_t t = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (t >= (size_t)S.nx * S.ny * S.nz) return;
    const int i = (int)(t % S.nx); const size_t r = t / S.nx; const int j = (int)(r % S.ny), k = (int)(r / S.ny);
    const double c0 = A.p[t];
    if (wall_row<COMP_U>(S, i, j, k)) { A.hu[t] = 0.0; A.ru[t] = 0.0; }
    else {
        double H = conv_u(S, A.u, A.v, A.w, i, j, k);
        if (A.fu) H = FSEI_ADD(H, A.fu[t]);
        const double gp = FSEI_MUL(FSEI_SUB(c0, A.p[sidx(S, i > 0 ? i - 1 : S.nx - 1, j, k)]), S.rdx);
        A.ru[t] = rhs_assemble(H, A.hu[t], gp, vel_lap<COMP_U>(S, A.u, i, j, k), A);
        A.hu[t] = H;
    }
    if (wall_row<COMP_V>(S, i, j, k)) { A.hv[t] = 0.0; A.rv[t] = 0.0; }
    else {
        double H = conv_v(S, A.u, A.v, A.w, i, j, k);
        if (A.fv) H = FSEI_ADD(H, A.fv[t]);
        const double gp = FSEI_MUL(FSEI_SUB(c0, A.p[sidx(S, i, j > 0 ? j - 1 : S.ny - 1, k)]), S.rdy);
        A.rv[t] = rhs_assemble(H, A.hv[t], gp, vel_lap<COMP_V>(S, A.v, i, j, k), A);
        A.hv[t] = H;
    }
    if (wall_row<COMP_W>(S, i, j, k)) { A.hw[t] = 0.0; A.rw[t] = 0.0; }
    else {
        double H = conv_w(S, A.u, A.v, A.w, i, j, k);
        if (A.fw) H = FSEI_ADD(H, A.fw[t]);
        const double gp = FSEI_MUL(FSEI_SUB(c0, A.p[sidx(S, i, j, k - 1)]), S.rdzm[k]);
        A.rw[t] = rhs_assemble(H, A.hw[t], gp, vel_lap<COMP_W>(S, A.w, i, j, k), A);
        A.hw[t] = H;
    }
}

}  // namespace fsei
