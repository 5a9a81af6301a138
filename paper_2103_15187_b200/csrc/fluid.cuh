// fluid.cuh -- the two steps that precede the pressure projection in one fluid substep:
//
//   explicit terms (Eq. 3):  H = -div(u u),
//        rhs_q = ((gdt H + rdt Hprev) - adt G p) + 2 beta lap q (+ adt f),   Hprev <- H
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
// explicit terms.  CTA = 32 x 8 threads on a tile of 32 x-cells by 8 y-rows, marching KZ planes along z (2.5-D
// blocking): the (34 x 10) halo tiles of u, v, w, p of plane k+3 are on their way to a four-slot shared-memory ring
// (cp.async, 8-byte copies, one commit group per plane) while plane k is evaluated from slots k, k+1 and from registers
// carried along the march (everything it needs of plane k-1, and what it already read of plane k one iteration ago) -- so the bytes in flight per SM do not depend on how many registers a thread can spare, every
// input plane is read from L2/DRAM once per CTA (+ halo), and the only global accesses of the compute phase are the six
// coalesced stores.  Every floating-point operation is individually rounded in the order of the definition
// (V10 states it), so the results are bit-identical.
//
// Boundary conventions (V7): periodic wrap (by the loader's source index); beyond a wall the wall-normal
// component is 0 (face n) and a tangential component is its ghost -q (no slip, wall midway); a convective flux through
// a wall face is 0; wall-face rows (u at i = 0, v at j = 0 on a wall-bounded box; w at k = 0) get H = rhs = 0.
// ---------------------------------------------------------------------------------------------------------------
FSEI_DEV double avg2(double a, double b) { return FSEI_MUL(0.5, FSEI_ADD(a, b)); }
FSEI_DEV double sq_diff(double a, double b, double r) { return FSEI_MUL(FSEI_SUB(FSEI_MUL(a, a), FSEI_MUL(b, b)), r); }
FSEI_DEV double d2_grad(double qp, double c0, double qm, double r) { return FSEI_MUL(FSEI_SUB(FSEI_MUL(FSEI_SUB(qp, c0), r), FSEI_MUL(FSEI_SUB(c0, qm), r)), r); }
FSEI_DEV double neg3(double fx, double fy, double fz) { return -FSEI_ADD(FSEI_ADD(fx, fy), fz); }

struct ExplicitArgs {
    SParams S;
    const double *u, *v, *w, *p, *fu, *fv, *fw;     // fu, fv, fw may be null (no body force)
    double *hu, *hv, *hw;                           // in: H of the previous substep, out: H of this one
    double *ru, *rv, *rw;                           // out: right-hand sides of the implicit step
    double gdt, rdt, adt, tb;                       // gamma dt, rho dt, alpha dt, 2 beta
    int kz;                                         // planes per CTA (host: 64 on large grids, fewer when the grid would not fill the GPU)
    int ring, slot;                                 // ring slots (>= FSEI_EXPL_RING) and doubles per slot, sized by the host to two CTAs per SM
    int tma;                                        // the four maps below are valid (nx even, encode succeeded)
    TmaMap3D mu, mv, mw, mp;                        // (nx, ny, planes incl. slab halos) fp64, box (PW, TY + 2, 1)
    TmaMap3D mh[3], mf[3];                          // (nx, ny, planes) views of H_prev and of the body force, box (TX, TY, 1)
};

FSEI_DEV double rhs_assemble(double H, double Hp, double gp, double lap, const ExplicitArgs& A)
{
    return FSEI_ADD(FSEI_SUB(FSEI_ADD(FSEI_MUL(A.gdt, H), FSEI_MUL(A.rdt, Hp)), FSEI_MUL(A.adt, gp)), FSEI_MUL(A.tb, lap));
}

#ifndef FSEI_EXPL_MINB
#define FSEI_EXPL_MINB 2
#endif
#define FSEI_EXPL_KZMAX 64             // most planes a CTA marches (ExplicitArgs::kz)
#define FSEI_EXPL_TX 32
#define FSEI_EXPL_TY 8
#ifndef FSEI_EXPL_AHEAD
#define FSEI_EXPL_AHEAD 2              // planes in flight beyond k+1
#endif
#define FSEI_EXPL_RING (2 + FSEI_EXPL_AHEAD)    // planes k, k+1 being read + AHEAD in flight (plane k-1 lives in registers)
#define FSEI_EXPL_PW (FSEI_EXPL_TX + 4)                             // columns i0-2 .. i0+33: the box starts on a 16-byte boundary
#define FSEI_EXPL_TILE_ELEMS (FSEI_EXPL_PW * (FSEI_EXPL_TY + 2))
#define FSEI_EXPL_TILE ((FSEI_EXPL_TILE_ELEMS + 15) / 16 * 16)      // tile pitch: every tile starts 128-byte aligned (TMA destination)
// doubles per ring slot: four halo tiles (u, v, w, p); H_prev of the next plane waits in three registers
#define FSEI_EXPL_CELLS (FSEI_EXPL_TX * FSEI_EXPL_TY)
// doubles per ring slot: four halo tiles (u, v, w, p) + the CTA's cells of H_prev and of the body force (TMA tiles; rim tiles
// prefetch those into registers)
#define FSEI_EXPL_SLOT(nforce) (4 * FSEI_EXPL_TILE + (3 + (nforce)) * FSEI_EXPL_CELLS)
#define FSEI_EXPL_MAXRING 6
#define FSEI_EXPL_SMEM_MAX (110 * 1024)            // two CTAs per SM

#if defined(__CUDACC__)
__device__ __forceinline__ void cp_async8(uint32_t sdst, const double* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// what a thread carries along the z march instead of reading it again from shared memory: the values of plane k+1 it
// used at plane k are plane k's at the next iteration (cur), and plane k's become the plane below (bel)
struct ExplicitCarry {
    double u00, v00, w00, wM0, w0M;                  // plane k     : u, v, w at the cell, w at i-1 and at j-1
    double u_km, v_km, w_km, p_km, uP_km, v0P_km;    // plane k - 1 : u, v, w, p at the cell, u at i+1, v at j+1 (0 beyond a wall)
};

// one cell of the three components from the ring slots of planes k (s0), k+1 (sp) and the carried registers.  EDGE = false: a
// cell with no wall or z boundary among its neighbours (every cell of a periodic box except on its bottom and top planes): the
// wall selects compile away.  The arithmetic of the two variants is the same, operation for operation.
template <bool EDGE>
__device__ __forceinline__ void explicit_cell(const ExplicitArgs& A, const double* __restrict__ s0, ExplicitCarry& C,
                                              const double* __restrict__ sp, int c, const double (&hprev)[3], const double (&fb3)[3], const double (&zm4)[4], size_t t,
                                              bool xlo, bool xhi, bool ylo, bool yhi, bool zlo, bool zhi)
{
    constexpr int PW = FSEI_EXPL_PW, TILE = FSEI_EXPL_TILE;
    const SParams& S = A.S;
    const double rdx = S.rdx, rdy = S.rdy;
    const double *U0 = s0, *V0 = s0 + TILE, *W0 = s0 + 2 * TILE, *P0 = s0 + 3 * TILE;
    const double *Up = sp, *Vp = sp + TILE, *Wp = sp + 2 * TILE;
    const double u00 = C.u00, v00 = C.v00, w00 = C.w00, p00 = P0[c];
    const double uP0 = (EDGE && xhi) ? 0.0 : U0[c + 1], uM0 = U0[c - 1], uPM = U0[c - PW + 1];
    double u0P = U0[c + PW], u0M = U0[c - PW];
    double vP0 = V0[c + 1], vM0 = V0[c - 1];
    const double v0P = (EDGE && yhi) ? 0.0 : V0[c + PW], v0M = V0[c - PW], vMP = V0[c + PW - 1];
    double wP0 = W0[c + 1], w0P = W0[c + PW], wM0 = C.wM0, w0M = C.w0M;
    const double pM0 = P0[c - 1], p0M = P0[c - PW];
    // plane above (fluxes through the upper face; never used on the top plane) and below (never used on the bottom one)
    const double u_kp = Up[c], v_kp = Vp[c], w_kp = (EDGE && zhi) ? 0.0 : Wp[c], wM_kp = Wp[c - 1], w0M_kp = Wp[c - PW];
    const double u_km = C.u_km, v_km = C.v_km, w_km = C.w_km, p_km = C.p_km, uP_km = C.uP_km, v0P_km = C.v0P_km;
    // the next plane's carry (the ghosts below overwrite only local copies)
    C.u_km = u00; C.v_km = v00; C.w_km = w00; C.p_km = p00; C.uP_km = uP0; C.v0P_km = v0P;
    C.u00 = u_kp; C.v00 = v_kp; C.w00 = w_kp; C.wM0 = wM_kp; C.w0M = w0M_kp;
    if (EDGE) {                                      // ghosts of the tangential components beyond a wall
        if (ylo) u0M = -u00; if (yhi) u0P = -u00;
        if (xlo) vM0 = -v00; if (xhi) vP0 = -v00;
        if (xlo) wM0 = -w00; if (xhi) wP0 = -w00;
        if (ylo) w0M = -w00; if (yhi) w0P = -w00;
    }
    const double rc = zm4[1], rm = zm4[2], rm_up = zm4[3], rc_dn = zm4[0];      // rdzc[k], rdzm[k], rdzm[k+1], rdzc[k-1]

    // ---- u
    if (EDGE && xlo) { A.hu[t] = 0.0; A.ru[t] = 0.0; }
    else {
        const double fx = sq_diff(avg2(u00, uP0), avg2(uM0, u00), rdx);
        const double fa = (EDGE && yhi) ? 0.0 : FSEI_MUL(avg2(u00, u0P), avg2(vMP, v0P));
        const double fb = (EDGE && ylo) ? 0.0 : FSEI_MUL(avg2(u0M, u00), avg2(vM0, v00));
        const double ga = (EDGE && zhi) ? 0.0 : FSEI_MUL(avg2(u00, u_kp), avg2(wM_kp, w_kp));
        const double gb = (EDGE && zlo) ? 0.0 : FSEI_MUL(avg2(u_km, u00), avg2(wM0, w00));
        const double H = neg3(fx, FSEI_MUL(FSEI_SUB(fa, fb), rdy), FSEI_MUL(FSEI_SUB(ga, gb), rc));
        const double gzp = (EDGE && zhi) ? FSEI_MUL(FSEI_SUB(0.0, u00), FSEI_MUL(2.0, rc)) : FSEI_MUL(FSEI_SUB(u_kp, u00), rm_up);
        const double gzm = (EDGE && zlo) ? FSEI_MUL(FSEI_SUB(u00, 0.0), FSEI_MUL(2.0, rc)) : FSEI_MUL(FSEI_SUB(u00, u_km), rm);
        const double lap = FSEI_ADD(FSEI_ADD(d2_grad(uP0, u00, uM0, rdx), d2_grad(u0P, u00, u0M, rdy)), FSEI_MUL(FSEI_SUB(gzp, gzm), rc));
        const double r_ = rhs_assemble(H, hprev[0], FSEI_MUL(FSEI_SUB(p00, pM0), rdx), lap, A);
        A.ru[t] = A.fu ? FSEI_ADD(r_, FSEI_MUL(A.adt, fb3[0])) : r_;
        A.hu[t] = H;
    }
    // ---- v
    if (EDGE && ylo) { A.hv[t] = 0.0; A.rv[t] = 0.0; }
    else {
        const double fa = (EDGE && xhi) ? 0.0 : FSEI_MUL(avg2(v00, vP0), avg2(uPM, uP0));
        const double fb = (EDGE && xlo) ? 0.0 : FSEI_MUL(avg2(vM0, v00), avg2(u0M, u00));
        const double fy = sq_diff(avg2(v00, v0P), avg2(v0M, v00), rdy);
        const double ga = (EDGE && zhi) ? 0.0 : FSEI_MUL(avg2(v00, v_kp), avg2(w0M_kp, w_kp));
        const double gb = (EDGE && zlo) ? 0.0 : FSEI_MUL(avg2(v_km, v00), avg2(w0M, w00));
        const double H = neg3(FSEI_MUL(FSEI_SUB(fa, fb), rdx), fy, FSEI_MUL(FSEI_SUB(ga, gb), rc));
        const double gzp = (EDGE && zhi) ? FSEI_MUL(FSEI_SUB(0.0, v00), FSEI_MUL(2.0, rc)) : FSEI_MUL(FSEI_SUB(v_kp, v00), rm_up);
        const double gzm = (EDGE && zlo) ? FSEI_MUL(FSEI_SUB(v00, 0.0), FSEI_MUL(2.0, rc)) : FSEI_MUL(FSEI_SUB(v00, v_km), rm);
        const double lap = FSEI_ADD(FSEI_ADD(d2_grad(vP0, v00, vM0, rdx), d2_grad(v0P, v00, v0M, rdy)), FSEI_MUL(FSEI_SUB(gzp, gzm), rc));
        const double r_ = rhs_assemble(H, hprev[1], FSEI_MUL(FSEI_SUB(p00, p0M), rdy), lap, A);
        A.rv[t] = A.fv ? FSEI_ADD(r_, FSEI_MUL(A.adt, fb3[1])) : r_;
        A.hv[t] = H;
    }
    // ---- w
    if (EDGE && zlo) { A.hw[t] = 0.0; A.rw[t] = 0.0; }
    else {
        const double fa = (EDGE && xhi) ? 0.0 : FSEI_MUL(avg2(w00, wP0), avg2(uP_km, uP0));
        const double fb = (EDGE && xlo) ? 0.0 : FSEI_MUL(avg2(wM0, w00), avg2(u_km, u00));
        const double ga = (EDGE && yhi) ? 0.0 : FSEI_MUL(avg2(w00, w0P), avg2(v0P_km, v0P));
        const double gb = (EDGE && ylo) ? 0.0 : FSEI_MUL(avg2(w0M, w00), avg2(v_km, v00));
        const double fz = sq_diff(avg2(w00, w_kp), avg2(w_km, w00), rm);
        const double H = neg3(FSEI_MUL(FSEI_SUB(fa, fb), rdx), FSEI_MUL(FSEI_SUB(ga, gb), rdy), fz);
        const double gzp = FSEI_MUL(FSEI_SUB(w_kp, w00), rc), gzm = FSEI_MUL(FSEI_SUB(w00, w_km), rc_dn);
        const double lap = FSEI_ADD(FSEI_ADD(d2_grad(wP0, w00, wM0, rdx), d2_grad(w0P, w00, w0M, rdy)), FSEI_MUL(FSEI_SUB(gzp, gzm), rm));
        const double r_ = rhs_assemble(H, hprev[2], FSEI_MUL(FSEI_SUB(p00, p_km), rm), lap, A);
        A.rw[t] = A.fw ? FSEI_ADD(r_, FSEI_MUL(A.adt, fb3[2])) : r_;
        A.hw[t] = H;
    }
}

// grid (ceil(nx/32), ceil(ny/8), ceil(nz/kz)), block (32, 8), dynamic shared memory FSEI_EXPL_SMEM
// TMA_TILE: a tile whose halo lies inside the grid takes its planes as ONE TMA box per field (issued by one thread); tiles on the
// rim (periodic wrap or a wall in the halo; ragged edges) keep the per-thread copies, whose source index wraps / clamps.  The
// two variants are separate instantiations so that neither carries the other's loader state in registers.
template <bool TMA_TILE>
__device__ __forceinline__ void explicit_march(const ExplicitArgs& A, double* ring, uint64_t* bars, double* zc_s, double* zm_s)
{
    constexpr int TX = FSEI_EXPL_TX, TY = FSEI_EXPL_TY, PW = FSEI_EXPL_PW, TILE = FSEI_EXPL_TILE;
    constexpr bool tile_tma = TMA_TILE;
    // ring depth: TMA tiles use every slot the host could fit (planes k, k+1 being read, the rest in flight); rim tiles wait by
    // cp.async group counts, which are immediates: AHEAD planes in flight whatever the ring holds
    const int R = A.ring, SLOT = A.slot, ahead = tile_tma ? R - 2 : FSEI_EXPL_AHEAD;
    const int f_u = 3, f_v = f_u + (A.fu ? 1 : 0), f_w = f_v + (A.fv ? 1 : 0);      // the force tiles follow H_prev's, those given only
    const SParams& S = A.S;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, i = i0 + tx, j = j0 + ty;
    int in = i < S.nx && j < S.ny;
    asm volatile("" : "+r"(in));                     // kept in a register: recomputing it costs four S2R / LDC round trips per plane
    const bool xper = S.bcx == BC_PERIODIC, yper = S.bcy == BC_PERIODIC;
    const bool xlo = !xper && i == 0, xhi = !xper && i == S.nx - 1;      // x-face i / i+1 is a wall
    const bool ylo = !yper && j == 0, yhi = !yper && j == S.ny - 1;
    const bool xyedge = xlo || xhi || ylo || yhi;
    if (tile_tma && tid == 0)
        for (int q = 0; q < R; q++) abar_init(&bars[q]);
    const size_t plane = (size_t)S.nx * S.ny;
    const int k0 = blockIdx.z * A.kz, k1 = (k0 + A.kz < S.nz) ? k0 + A.kz : S.nz;

    // loader: tile elements e = tid and tid + 256 of the halo tiles (source index wrapped in a periodic direction, clamped at
    // a wall or a ragged edge) and this thread's own cell of the H_prev tiles; source pointers advance one plane per issue
    const int e1 = tid + 256;
    const bool has1 = e1 < FSEI_EXPL_TILE_ELEMS;
    auto srcidx = [&](int e) {
        const int jj = e / PW, ii = e - jj * PW;
        int gi = i0 + ii - 2, gj = j0 + jj - 1;
        if (xper) { gi = gi < 0 ? gi + S.nx : (gi >= S.nx ? gi - S.nx : gi); }
        gi = gi < 0 ? 0 : (gi >= S.nx ? S.nx - 1 : gi);
        if (yper) { gj = gj < 0 ? gj + S.ny : (gj >= S.ny ? gj - S.ny : gj); }
        gj = gj < 0 ? 0 : (gj >= S.ny ? S.ny - 1 : gj);
        return (size_t)gj * S.nx + gi;
    };
    const int kfirst = k0 - 1;                       // first plane the loader is asked for
    // planes the fields hold: [klo, khi) = [0, nz), widened by the halo planes of a z-slab (S.halo_lo / S.halo_hi)
    const int klo = S.halo_lo ? -1 : 0, khi = S.nz + (S.halo_hi ? 1 : 0);
    long long o0 = 0, o1 = 0;
    if (!tile_tma) {
        o0 = (long long)srcidx(tid) + (long long)(kfirst < klo ? klo : kfirst) * (long long)plane;
        o1 = (long long)srcidx(has1 ? e1 : tid) + (long long)(kfirst < klo ? klo : kfirst) * (long long)plane;
    }
    int kk = kfirst, slot = (kfirst + 2 * R) % R;
    uint32_t ring_tid = smem_u32(ring + tid);        // shared-window address of this thread's first element of slot 0
    asm volatile("" : "+r"(ring_tid));
    auto issue = [&]() {                             // next plane kk -> its ring slot (nothing for a plane outside the grid or beyond k1)
        if (tile_tma) {
            if (tid == 0 && kk >= klo && kk < khi && kk <= k1) {
                double* sl = ring + slot * SLOT;
                const int zc = kk + (S.halo_lo ? 1 : 0);
                const bool own = kk >= k0 && kk < k1;                  // a plane this CTA evaluates: its H_prev and force come along
                const unsigned nf = (A.fu ? 1u : 0u) + (A.fv ? 1u : 0u) + (A.fw ? 1u : 0u);
                abar_expect(&bars[slot], 4u * FSEI_EXPL_TILE_ELEMS * 8u + (own ? (3u + nf) * FSEI_EXPL_CELLS * 8u : 0u));
                if (own) {
                    double* hs = sl + 4 * TILE;
#pragma unroll
                    for (int q = 0; q < 3; q++) tma_load_3d(hs + q * FSEI_EXPL_CELLS, &A.mh[q], i0, j0, kk, &bars[slot]);
                    if (A.fu) tma_load_3d(hs + f_u * FSEI_EXPL_CELLS, &A.mf[0], i0, j0, kk, &bars[slot]);
                    if (A.fv) tma_load_3d(hs + f_v * FSEI_EXPL_CELLS, &A.mf[1], i0, j0, kk, &bars[slot]);
                    if (A.fw) tma_load_3d(hs + f_w * FSEI_EXPL_CELLS, &A.mf[2], i0, j0, kk, &bars[slot]);
                }
                tma_load_3d(sl, &A.mu, i0 - 2, j0 - 1, zc, &bars[slot]);
                tma_load_3d(sl + TILE, &A.mv, i0 - 2, j0 - 1, zc, &bars[slot]);
                tma_load_3d(sl + 2 * TILE, &A.mw, i0 - 2, j0 - 1, zc, &bars[slot]);
                tma_load_3d(sl + 3 * TILE, &A.mp, i0 - 2, j0 - 1, zc, &bars[slot]);
            }
        } else if (kk >= klo && kk < khi && kk <= k1) {
            const uint32_t sl = ring_tid + (uint32_t)(slot * SLOT * 8);
            cp_async8(sl, A.u + o0); cp_async8(sl + TILE * 8, A.v + o0);
            cp_async8(sl + 2 * TILE * 8, A.w + o0); cp_async8(sl + 3 * TILE * 8, A.p + o0);
            if (has1) {
                cp_async8(sl + 256 * 8, A.u + o1); cp_async8(sl + (TILE + 256) * 8, A.v + o1);
                cp_async8(sl + (2 * TILE + 256) * 8, A.w + o1); cp_async8(sl + (3 * TILE + 256) * 8, A.p + o1);
            }
            o0 += (long long)plane; o1 += (long long)plane;
        }
        if (!tile_tma) cp_async_commit();
        kk++; slot = slot + 1 == R ? 0 : slot + 1;
    };
    unsigned phases = 0;                             // TMA tiles: parity of the next phase of every slot's mbarrier
    auto landed = [&](int kq, int sq) {              // plane kq (in slot sq) is waited for exactly once, in plane order
        if (kq >= klo && kq < khi) {
            abar_wait(&bars[sq], (phases >> sq) & 1u);
            phases ^= 1u << sq;
        }
    };
    __syncthreads();                                 // the mbarriers are initialised
    for (int q = 0; q < ahead + 2; q++) issue();     // planes k0-1 .. k0+ahead
    const int c = (ty + 1) * PW + tx + 2;
    int sc = k0 % R;                                 // slot of plane k
    size_t t = (size_t)k0 * plane + (size_t)j * S.nx + i;
    // H_prev and the body force of the NEXT plane wait in registers (loaded one iteration ahead of their use)
    double hnext[3] = {0.0, 0.0, 0.0}, fnext[3] = {0.0, 0.0, 0.0};
    auto fetch_hf = [&](size_t tt) {
        hnext[0] = A.hu[tt]; hnext[1] = A.hv[tt]; hnext[2] = A.hw[tt];
        if (A.fu) fnext[0] = A.fu[tt];
        if (A.fv) fnext[1] = A.fv[tt];
        if (A.fw) fnext[2] = A.fw[tt];
    };
    if (!tile_tma && in) fetch_hf(t);
    // z metrics of planes k0-1 .. k1+1 staged in shared memory (they are warp-uniform: read from global memory in the loop
    // they end up in uniform registers, and the conversion waits out the full load latency every plane)
    for (int q = tid; q < k1 - k0 + 3; q += 256) {
        const int kq = k0 - 1 + q;                                  // slab view: the metric tables are global, hence + kofs
        const bool there = kq >= klo && kq < khi;
        zc_s[q] = there ? S.rdzc[kq + S.kofs] : 0.0;
        zm_s[q] = there ? S.rdzm[kq + S.kofs] : 0.0;
    }

    // the carried registers of the first plane: plane k0 and the plane below it (not there below the bottom: never used)
    ExplicitCarry C;
    if (tile_tma) { landed(kfirst, sc == 0 ? R - 1 : sc - 1); landed(k0, sc); }
    else cp_async_wait<FSEI_EXPL_AHEAD>();           // planes <= k0 have landed
    __syncthreads();
    {
        const double* s0 = ring + sc * SLOT;
        const double* sm = ring + (sc == 0 ? R - 1 : sc - 1) * SLOT;
        C.u00 = s0[c]; C.v00 = s0[TILE + c]; C.w00 = s0[2 * TILE + c]; C.wM0 = s0[2 * TILE + c - 1]; C.w0M = s0[2 * TILE + c - PW];
        const bool below = kfirst >= klo;
        C.u_km = below ? sm[c] : 0.0; C.v_km = below ? sm[TILE + c] : 0.0; C.w_km = below ? sm[2 * TILE + c] : 0.0;
        C.p_km = below ? sm[3 * TILE + c] : 0.0;
        C.uP_km = (below && !xhi) ? sm[c + 1] : 0.0; C.v0P_km = (below && !yhi) ? sm[TILE + c + PW] : 0.0;
    }

    for (int k = k0; k < k1; k++, t += plane) {
        double hprev[3] = {hnext[0], hnext[1], hnext[2]}, fb3[3] = {fnext[0], fnext[1], fnext[2]};
        if (tile_tma) {                              // plane k's slot landed one iteration ago
            const double* hs = ring + sc * SLOT + 4 * TILE + tid;
            hprev[0] = hs[0]; hprev[1] = hs[FSEI_EXPL_CELLS]; hprev[2] = hs[2 * FSEI_EXPL_CELLS];
            if (A.fu) fb3[0] = hs[f_u * FSEI_EXPL_CELLS];
            if (A.fv) fb3[1] = hs[f_v * FSEI_EXPL_CELLS];
            if (A.fw) fb3[2] = hs[f_w * FSEI_EXPL_CELLS];
        } else if (in && k + 1 < k1) fetch_hf(t + plane);
        const int kq = k - k0;                       // rdzc[k-1], rdzc[k], rdzm[k], rdzm[k+1]
        const double zm4[4] = {zc_s[kq], zc_s[kq + 1], zm_s[kq + 1], zm_s[kq + 2]};
        if (tile_tma) landed(k + 1, sc + 1 == R ? 0 : sc + 1);
        else cp_async_wait<FSEI_EXPL_AHEAD - 1>();   // everything but the newest AHEAD-1 groups: planes <= k+1 have landed
        __syncthreads();                             // ... for every thread; and every thread is done with slot (k-1) mod R
        issue();                                     // plane k+ahead+1 -> the slot plane k-1 was in (TMA tiles: slot (k-1) mod R)
        const int sp_ = sc + 1 == R ? 0 : sc + 1;
        if (in) {
            const double* s0 = ring + sc * SLOT;
            const double* sp = ring + sp_ * SLOT;
            const bool zlo = k == 0 && !S.halo_lo, zhi = k == S.nz - 1 && !S.halo_hi;     // a wall, not a slab boundary
            if (xyedge || zlo || zhi) explicit_cell<true>(A, s0, C, sp, c, hprev, fb3, zm4, t, xlo, xhi, ylo, yhi, zlo, zhi);
            else explicit_cell<false>(A, s0, C, sp, c, hprev, fb3, zm4, t, false, false, false, false, false, false);
        }
        sc = sp_;
    }
    if (!tile_tma) cp_async_wait<0>();
}

FSEI_GLOBAL(256, FSEI_EXPL_MINB) k_explicit_terms(const FSEI_GRID_CONSTANT ExplicitArgs A)
{
    FSEI_DYN_SMEM(smraw);
    __shared__ __align__(8) uint64_t bars[FSEI_EXPL_MAXRING];
    __shared__ double zc_s[FSEI_EXPL_KZMAX + 3], zm_s[FSEI_EXPL_KZMAX + 3];
    double* ring = reinterpret_cast<double*>(smraw);
    const int i0 = blockIdx.x * FSEI_EXPL_TX, j0 = blockIdx.y * FSEI_EXPL_TY;
    if (A.tma && i0 >= 2 && i0 + FSEI_EXPL_TX + 2 <= A.S.nx && j0 >= 1 && j0 + FSEI_EXPL_TY + 1 <= A.S.ny)
        explicit_march<true>(A, ring, bars, zc_s, zm_s);
    else
        explicit_march<false>(A, ring, bars, zc_s, zm_s);
}
#endif  // __CUDACC__

}  // namespace fsei
