/*
 * fsei_fluid_oracle.c -- CPU ORACLE for the two steps that precede the pressure projection
 * in one fluid substep of the paper's fractional-step scheme.  TEST INFRASTRUCTURE (same
 * rules as fsei_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may
 * load it; it shares no code, header, table or constant with paper_2103_15187_b200/).
 *
 * What it follows (P:Lnnn = /root/reference/PAPER.md line nnn):
 *   Eq. 3 (sec. 2.1):
 *     (u^{n+1}-u^n)/dt + [gamma div(uu)^n + rho div(uu)^{n-1}]
 *         = -grad p^{n+1} + (1/(2 Re)) lap(u^{n+1} + u^n) + f
 *   "explicit Adams-Bashforth method for the nonlinear convective term and an implicit
 *   Crank-Nicolson method for the viscous terms", gamma = 3/2, rho = -1/2; "a third order
 *   Runge-Kutta scheme is also implemented"
 *   "central second-order finite-differences discretized on a staggered mesh"
 *   "The viscous terms are treated implicitly yielding the solution of a large sparse matrix,
 *   which is avoided by an approximate factorization yielding tridiagonal matrices (one for
 *   each direction [13]) inverted using Thomas' algorithm with a Sherman-Morrison perturbation
 *   in the two periodic dimensions" (sec. 3.1)
 *   "a fractional-step method [18, 13] is used"
 * The paper prints nothing more; the discrete operators are the readings V1..V12 of DESIGN.md
 * sec. 3 (the second-order staggered scheme of the paper's refs [12],[13],[14]):
 *
 *   substep with weights gamma_l, rho_l, alpha_l = gamma_l + rho_l, beta = alpha_l dt/(2 Re):
 *     H^n   = -div(u u)^n                                                  (NEXT-2, explicit)
 *     rhs   = dt (gamma_l H^n + rho_l H^{n-1}) - alpha_l dt G p^n + 2 beta lap(q^n) + alpha_l dt f
 *             (f stands OUTSIDE the [gamma .. rho ..] bracket of Eq. 3: it carries the weight of the substep, alpha_l dt)
 *     (1 - beta dxx)(1 - beta dyy)(1 - beta dzz) dq = rhs                   (NEXT-1, implicit)
 *     q^    = q^n + dq          -> then the pressure projection of fsei_oracle.c
 *
 * Staggering: u[k][j][i] on the low x-face of cell (i,j,k), v low y-face,
 * w low z-face, p at the centre.  Periodic direction: face n == face 0.  Wall direction (z
 * always; x,y when bc = 1): stored face 0 is the wall (velocity 0, never modified), the high
 * wall face is not stored and is 0; a component TANGENTIAL to a wall sits half a cell away from
 * it and sees the no-slip wall through the ghost value q_ghost = -q_first (wall value 0 midway).
 *
 * The implicit step is computed in real_t (long double in the parity build); the explicit
 * terms are stencils and are ALWAYS computed in IEEE double in one fixed order with no FMA
 * contraction (-ffp-contract=off), so that a CUDA kernel keeping the order matches bit for bit.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real_t;
#else
typedef double real_t;
#endif

enum { BC_P = 0, BC_W = 1 };          /* periodic / wall-bounded (the projection's FSEI_BC_NEUMANN) */
enum { DIR_X = 0, DIR_Y = 1, DIR_Z = 2 };
enum { COMP_U = 0, COMP_V = 1, COMP_W = 2 };

#define IDX(i, j, k) (((size_t)(k) * (size_t)ny + (size_t)(j)) * (size_t)nx + (size_t)(i))

/* ------------------------------------------------------------------------- */
/* Thomas' algorithm:  a_k x_{k-1} + b_k x_k + c_k x_{k+1} = d_k.    */
/* ------------------------------------------------------------------------- */
static void thomas(int n, const real_t *a, const real_t *b, const real_t *c, const real_t *d, real_t *x, real_t *cp)
{
    real_t piv = b[0];
    cp[0] = c[0] / piv;
    x[0] = d[0] / piv;
    for (int k = 1; k < n; k++) {
        piv = b[k] - a[k] * cp[k - 1];
        cp[k] = c[k] / piv;
        x[k] = (d[k] - a[k] * x[k - 1]) / piv;
    }
    for (int k = n - 2; k >= 0; k--) x[k] -= cp[k] * x[k + 1];
}

/* ------------------------------------------------------------------------- */
/* Cyclic tridiagonal system by Thomas + Sherman-Morrison:           */
/*   a_k x_{k-1} + b_k x_k + c_k x_{k+1} = d_k  with indices modulo n,        */
/* i.e. A = T + p q^T with the corner entries A[0][n-1] = a_0, A[n-1][0] =    */
/* c_{n-1} moved into the rank-one term:  p = (g, 0, .., 0, c_{n-1})^T,       */
/* q = (1, 0, .., 0, a_0/g)^T, g = -b_0, T = A - p q^T tridiagonal with       */
/* T[0][0] = b_0 - g, T[n-1][n-1] = b_{n-1} - a_0 c_{n-1}/g.  Then            */
/*   T y = d,  T z = p,  x = y - z (q.y)/(1 + q.z).                           */
/* work: 5n.  n >= 3 (n = 1, 2 are handled as the small dense systems they are).*/
/* ------------------------------------------------------------------------- */
static void cyclic_thomas(int n, const real_t *a, const real_t *b, const real_t *c, const real_t *d, real_t *x,
                          real_t *work)
{
    if (n == 1) { x[0] = d[0] / (a[0] + b[0] + c[0]); return; }
    if (n == 2) {                       /* both neighbours of row k are the other unknown */
        real_t o0 = a[0] + c[0], o1 = a[1] + c[1], det = b[0] * b[1] - o0 * o1;
        x[0] = (d[0] * b[1] - o0 * d[1]) / det;
        x[1] = (b[0] * d[1] - o1 * d[0]) / det;
        return;
    }
    real_t *bb = work, *p = work + n, *y = work + 2 * n, *z = work + 3 * n, *cp = work + 4 * n;
    real_t g = -b[0];
    for (int k = 0; k < n; k++) { bb[k] = b[k]; p[k] = 0; }
    bb[0] = b[0] - g;
    bb[n - 1] = b[n - 1] - a[0] * c[n - 1] / g;
    p[0] = g; p[n - 1] = c[n - 1];
    thomas(n, a, bb, c, d, y, cp);
    thomas(n, a, bb, c, p, z, cp);
    real_t qy = y[0] + (a[0] / g) * y[n - 1];
    real_t qz = z[0] + (a[0] / g) * z[n - 1];
    real_t f = qy / (1 + qz);
    for (int k = 0; k < n; k++) x[k] = y[k] - f * z[k];
}

/* ------------------------------------------------------------------------- */
/* Wall-normal metrics, evaluated once in double exactly as every stencil     */
/* evaluates them (same convention as fsei_oracle.c, reading R5/R20).         */
/* ------------------------------------------------------------------------- */
static void zmetric_double(int nz, const double *zc, double *rdzc, double *rdzm)
{
    for (int k = 0; k < nz; k++) rdzc[k] = 1.0 / (zc[k + 1] - zc[k]);
    rdzm[0] = 0.0;
    for (int k = 1; k < nz; k++) rdzm[k] = 1.0 / (0.5 * (zc[k] + zc[k + 1]) - 0.5 * (zc[k - 1] + zc[k]));
}

/* ------------------------------------------------------------------------- */
/* Rows of the 1-D second-difference operator of component `comp` along       */
/* direction `dir` (readings V3-V6):                                          */
/*   (d2 q)_m = lo[m] q_{m-1} + di[m] q_m + up[m] q_{m+1}                     */
/* *cyclic = 1: indices modulo n (periodic direction).  fixed[m] = 1: row m   */
/* is a wall face of this component (value 0, never modified).               */
/*  - uniform periodic: (q_{m+1} - 2 q_m + q_{m-1})/h^2                       */
/*  - uniform wall direction, component NORMAL to the wall (u along x, v along*/
/*    y): face 0 fixed; faces 1..n-1 standard, the not-stored face n is 0     */
/*  - uniform wall direction, tangential component (cell-centred along it):   */
/*    ghost q_{-1} = -q_0, q_n = -q_{n-1}  ->  first/last diagonal -3/h^2     */
/*  - z, u and v (centres zm[k]): flux form on the stretched grid,            */
/*      [ (q_{k+1}-q_k)/dzm[k+1] - (q_k-q_{k-1})/dzm[k] ] / dzc[k];           */
/*    at the walls the one-sided gradient (q_0 - 0)/(dzc[0]/2), resp.         */
/*    (0 - q_{nz-1})/(dzc[nz-1]/2)                                            */
/*  - z, w (faces zc[k]): face 0 fixed; faces 1..nz-1                         */
/*      [ (w_{k+1}-w_k)/dzc[k] - (w_k-w_{k-1})/dzc[k-1] ] / dzm[k], w_nz = 0  */
/* ------------------------------------------------------------------------- */
static int visc_rows(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                     int comp, int dir, real_t *lo, real_t *di, real_t *up, int *fixed, int *cyclic)
{
    if (dir == DIR_X || dir == DIR_Y) {
        int n = dir == DIR_X ? nx : ny;
        int bc = dir == DIR_X ? bc_x : bc_y;
        double rh = 1.0 / ((dir == DIR_X ? Lx : Ly) / (double)n);          /* the stencils' own reciprocal */
        real_t r2 = (real_t)rh * (real_t)rh;
        int normal = (dir == DIR_X && comp == COMP_U) || (dir == DIR_Y && comp == COMP_V);
        for (int m = 0; m < n; m++) { lo[m] = r2; di[m] = -2 * r2; up[m] = r2; fixed[m] = 0; }
        *cyclic = (bc == BC_P);
        if (bc == BC_W) {
            if (normal) { fixed[0] = 1; lo[1] = 0; up[n - 1] = 0; }         /* q_0 = 0 (stored), q_n = 0 (not stored) */
            else { lo[0] = 0; di[0] = -3 * r2; up[n - 1] = 0; di[n - 1] = -3 * r2; if (n == 1) di[0] = -4 * r2; }
        }
        return n;
    }
    double *rc = malloc(sizeof(double) * nz), *rm = malloc(sizeof(double) * nz);
    zmetric_double(nz, zc, rc, rm);
    *cyclic = 0;
    if (comp != COMP_W) {
        for (int k = 0; k < nz; k++) {
            real_t l = (k > 0) ? (real_t)rm[k] * (real_t)rc[k] : 0;
            real_t u = (k + 1 < nz) ? (real_t)rm[k + 1] * (real_t)rc[k] : 0;
            real_t wl = (k == 0) ? 2 * (real_t)rc[k] * (real_t)rc[k] : 0;          /* wall half a cell below */
            real_t wu = (k == nz - 1) ? 2 * (real_t)rc[k] * (real_t)rc[k] : 0;     /* wall half a cell above */
            lo[k] = l; up[k] = u; di[k] = -(l + u + wl + wu); fixed[k] = 0;
        }
    } else {
        fixed[0] = 1; lo[0] = 0; di[0] = 0; up[0] = 0;
        for (int k = 1; k < nz; k++) {
            real_t l = (real_t)rc[k - 1] * (real_t)rm[k], u = (real_t)rc[k] * (real_t)rm[k];
            lo[k] = (k > 1) ? l : 0;                  /* w_0 = 0 */
            up[k] = (k + 1 < nz) ? u : 0;             /* w_nz = 0 */
            di[k] = -(l + u); fixed[k] = 0;
        }
    }
    free(rc); free(rm);
    return nz;
}

/* Solve (1 - beta d2) x = d along one line (in place in d): Thomas on a wall direction, */
/* Thomas + Sherman-Morrison on a periodic one.  Fixed (wall-face) rows give 0. */
static void visc_line_solve(int n, real_t beta, const real_t *lo, const real_t *di, const real_t *up,
                            const int *fixed, int cyclic, real_t *d, real_t *work /* 9n */)
{
    real_t *a = work, *b = work + n, *c = work + 2 * n, *x = work + 3 * n, *wk = work + 4 * n;
    for (int m = 0; m < n; m++) {
        if (fixed[m]) { a[m] = 0; b[m] = 1; c[m] = 0; d[m] = 0; }
        else { a[m] = -beta * lo[m]; b[m] = 1 - beta * di[m]; c[m] = -beta * up[m]; }
    }
    if (cyclic) cyclic_thomas(n, a, b, c, d, x, wk);
    else thomas(n, a, b, c, d, x, wk);
    for (int m = 0; m < n; m++) d[m] = x[m];
}

/* One directional sweep over a whole field held in real_t. */
static void visc_sweep(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                       int comp, int dir, real_t beta, real_t *f)
{
    int nmax = nx > ny ? nx : ny; if (nz > nmax) nmax = nz;
    real_t *lo = malloc(sizeof(real_t) * nmax), *di = malloc(sizeof(real_t) * nmax), *up = malloc(sizeof(real_t) * nmax);
    int *fixed = malloc(sizeof(int) * nmax), cyclic = 0;
    int n = visc_rows(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, comp, dir, lo, di, up, fixed, &cyclic);
    long nlines = (long)nx * ny * nz / n;
#pragma omp parallel
    {
        real_t *line = malloc(sizeof(real_t) * n), *work = malloc(sizeof(real_t) * 9 * n);
#pragma omp for schedule(static)
        for (long l = 0; l < nlines; l++) {
            size_t base, stride;
            if (dir == DIR_X) { base = (size_t)l * nx; stride = 1; }
            else if (dir == DIR_Y) { base = (size_t)(l / nx) * nx * ny + (size_t)(l % nx); stride = nx; }
            else { base = (size_t)l; stride = (size_t)nx * ny; }
            for (int m = 0; m < n; m++) line[m] = f[base + m * stride];
            visc_line_solve(n, beta, lo, di, up, fixed, cyclic, line, work);
            for (int m = 0; m < n; m++) f[base + m * stride] = line[m];
        }
        free(line); free(work);
    }
    free(lo); free(di); free(up); free(fixed);
}

/* ------------------------------------------------------------------------- */
/* NEXT-1: the implicit viscous step (Eq. 3), in place on u, v, w:    */
/*   q += [(1 - beta dxx)(1 - beta dyy)(1 - beta dzz)]^{-1} rhs_q             */
/* sweeps in the order x, y, z (reading V2; the three factors commute).       */
/* ------------------------------------------------------------------------- */
int oracle_viscous_step(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                        double *u, double *v, double *w, const double *ru, const double *rv, const double *rw,
                        double beta)
{
    if (nx < 1 || ny < 1 || nz < 2 || !(beta >= 0)) return 1;
    size_t N = (size_t)nx * ny * nz;
    real_t *f = malloc(sizeof(real_t) * N);
    if (!f) return 4;
    double *q[3] = {u, v, w};
    const double *r[3] = {ru, rv, rw};
    for (int comp = 0; comp < 3; comp++) {
        for (size_t t = 0; t < N; t++) f[t] = (real_t)r[comp][t];
        for (int dir = 0; dir < 3; dir++) visc_sweep(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, comp, dir, (real_t)beta, f);
        for (size_t t = 0; t < N; t++) q[comp][t] = (double)((real_t)q[comp][t] + f[t]);
    }
    free(f);
    return 0;
}

/* One sweep on a double field (exported so the tests can check each factor and the commutation). */
int oracle_viscous_sweep(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                         int comp, int dir, double beta, double *f)
{
    size_t N = (size_t)nx * ny * nz;
    real_t *g = malloc(sizeof(real_t) * N);
    if (!g) return 4;
    for (size_t t = 0; t < N; t++) g[t] = (real_t)f[t];
    visc_sweep(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, comp, dir, (real_t)beta, g);
    for (size_t t = 0; t < N; t++) f[t] = (double)g[t];
    free(g);
    return 0;
}

int oracle_cyclic_thomas(int n, const double *a, const double *b, const double *c, const double *d, double *x)
{
    real_t *m = malloc(sizeof(real_t) * 10 * (size_t)n);
    for (int k = 0; k < n; k++) { m[k] = a[k]; m[n + k] = b[k]; m[2 * n + k] = c[k]; m[3 * n + k] = d[k]; }
    cyclic_thomas(n, m, m + n, m + 2 * n, m + 3 * n, m + 4 * n, m + 5 * n);
    for (int k = 0; k < n; k++) x[k] = (double)m[4 * n + k];
    free(m);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* NEXT-2: explicit terms of Eq. 3, IEEE double, fixed order.      */
/*                                                                           */
/* Convective term in divergence form, second-order central, plain arithmetic */
/* averages to the flux positions (reading V8):                               */
/*  H_u(i,j,k) = -{ [ (u~x)^2|_{i} - (u~x)^2|_{i-1} ] /dx          (cell centres i, i-1)
 *               + [ (u~y v~x)|_{j+1} - (u~y v~x)|_{j} ] /dy        (x-face i, y-faces j+1, j)
 *               + [ (u~z w~x)|_{k+1} - (u~z w~x)|_{k} ] /dzc[k] }  (x-face i, z-faces k+1, k)
 *  with q~d the mean of the two values of q adjacent along d; H_v alike; H_w with the z
 *  difference of (w~z)^2 between cell centres k and k-1 divided by dzm[k].  A flux through a
 *  wall face is 0 (the normal velocity vanishes there).  Wall-face rows are left 0.
 * Pressure gradient: the projection's own G (fsei_oracle.c, a7).
 * Viscous term: lap q = (dxx q + dyy q) + dzz q with the flux-form second differences of
 *  visc_rows (reading V3-V6) written out as gradient differences.
 *  rhs_q = ((gdt H + rdt Hprev) - adt G p) + (2 beta) lap q      (each operation rounded)
 *  rhs_q = rhs_q + adt f_q                                        if a body force is given (Eq. 3: f outside the bracket)
 *  Hprev <- H.
 */
typedef struct {
    int nx, ny, nz, bc_x, bc_y;
    double rdx, rdy;
    const double *rdzc, *rdzm;
} sgrid;

static inline int wrapi(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

/* value of component q at (i,j,k) with the boundary conventions: periodic wrap; beyond a wall: */
/* normal component -> 0 (wall face n) ; tangential -> ghost = -(first interior) ; z likewise.  */
static inline double fetch(const sgrid *g, const double *q, int comp, int i, int j, int k)
{
    int nx = g->nx, ny = g->ny, nz = g->nz;
    double sign = 1.0;
    if (i < 0 || i >= nx) {
        if (g->bc_x == BC_P) i = wrapi(i, nx);
        else if (comp == COMP_U) return 0.0;
        else { i = i < 0 ? 0 : nx - 1; sign = -sign; }
    }
    if (j < 0 || j >= ny) {
        if (g->bc_y == BC_P) j = wrapi(j, ny);
        else if (comp == COMP_V) return 0.0;
        else { j = j < 0 ? 0 : ny - 1; sign = -sign; }
    }
    if (k < 0 || k >= nz) {
        if (comp == COMP_W) return 0.0;
        k = k < 0 ? 0 : nz - 1; sign = -sign;
    }
    double val = q[IDX(i, j, k)];
    return sign < 0 ? -val : val;
}

/* second differences in gradient form */
static inline double d2_uniform(const sgrid *g, const double *q, int comp, int dir, int i, int j, int k)
{
    int di = dir == DIR_X, dj = dir == DIR_Y;
    double r = dir == DIR_X ? g->rdx : g->rdy;
    double c0 = q[((size_t)k * g->ny + j) * g->nx + i];
    double qp = fetch(g, q, comp, i + di, j + dj, k), qm = fetch(g, q, comp, i - di, j - dj, k);
    double gp = (qp - c0) * r, gm = (c0 - qm) * r;
    return (gp - gm) * r;
}
static inline double d2_z(const sgrid *g, const double *q, int comp, int i, int j, int k)
{
    int nx = g->nx, ny = g->ny, nz = g->nz;
    double c0 = q[IDX(i, j, k)];
    if (comp != COMP_W) {
        double gp = (k + 1 < nz) ? (q[IDX(i, j, k + 1)] - c0) * g->rdzm[k + 1] : (0.0 - c0) * (2.0 * g->rdzc[k]);
        double gm = (k > 0) ? (c0 - q[IDX(i, j, k - 1)]) * g->rdzm[k] : (c0 - 0.0) * (2.0 * g->rdzc[k]);
        return (gp - gm) * g->rdzc[k];
    }
    double wp = (k + 1 < nz) ? q[IDX(i, j, k + 1)] : 0.0;
    double gp = (wp - c0) * g->rdzc[k], gm = (c0 - q[IDX(i, j, k - 1)]) * g->rdzc[k - 1];
    return (gp - gm) * g->rdzm[k];
}

static inline int wall_row(const sgrid *g, int comp, int i, int j, int k)
{
    return (comp == COMP_U && g->bc_x == BC_W && i == 0) || (comp == COMP_V && g->bc_y == BC_W && j == 0) ||
           (comp == COMP_W && k == 0);
}

/* lap q at the position of component comp (0 on wall rows) */
static inline double vel_lap(const sgrid *g, const double *q, int comp, int i, int j, int k)
{
    if (wall_row(g, comp, i, j, k)) return 0.0;
    return (d2_uniform(g, q, comp, DIR_X, i, j, k) + d2_uniform(g, q, comp, DIR_Y, i, j, k)) + d2_z(g, q, comp, i, j, k);
}

/* is the x-face `i` (0..nx) / y-face j / z-face k a wall face? */
static inline int xwall(const sgrid *g, int i) { return g->bc_x == BC_W && (i <= 0 || i >= g->nx); }
static inline int ywall(const sgrid *g, int j) { return g->bc_y == BC_W && (j <= 0 || j >= g->ny); }
static inline int zwall(const sgrid *g, int k) { return k <= 0 || k >= g->nz; }

static inline double conv_u(const sgrid *g, const double *u, const double *v, const double *w, int i, int j, int k)
{
    double c0 = fetch(g, u, COMP_U, i, j, k);
    double ucp = 0.5 * (c0 + fetch(g, u, COMP_U, i + 1, j, k));
    double ucm = 0.5 * (fetch(g, u, COMP_U, i - 1, j, k) + c0);
    double fx = (ucp * ucp - ucm * ucm) * g->rdx;
    double fa = ywall(g, j + 1) ? 0.0 : (0.5 * (c0 + fetch(g, u, COMP_U, i, j + 1, k))) *
                                        (0.5 * (fetch(g, v, COMP_V, i - 1, j + 1, k) + fetch(g, v, COMP_V, i, j + 1, k)));
    double fb = ywall(g, j) ? 0.0 : (0.5 * (fetch(g, u, COMP_U, i, j - 1, k) + c0)) *
                                    (0.5 * (fetch(g, v, COMP_V, i - 1, j, k) + fetch(g, v, COMP_V, i, j, k)));
    double fy = (fa - fb) * g->rdy;
    double ga = zwall(g, k + 1) ? 0.0 : (0.5 * (c0 + fetch(g, u, COMP_U, i, j, k + 1))) *
                                        (0.5 * (fetch(g, w, COMP_W, i - 1, j, k + 1) + fetch(g, w, COMP_W, i, j, k + 1)));
    double gb = zwall(g, k) ? 0.0 : (0.5 * (fetch(g, u, COMP_U, i, j, k - 1) + c0)) *
                                    (0.5 * (fetch(g, w, COMP_W, i - 1, j, k) + fetch(g, w, COMP_W, i, j, k)));
    double fz = (ga - gb) * g->rdzc[k];
    return -((fx + fy) + fz);
}
static inline double conv_v(const sgrid *g, const double *u, const double *v, const double *w, int i, int j, int k)
{
    double c0 = fetch(g, v, COMP_V, i, j, k);
    double fa = xwall(g, i + 1) ? 0.0 : (0.5 * (c0 + fetch(g, v, COMP_V, i + 1, j, k))) *
                                        (0.5 * (fetch(g, u, COMP_U, i + 1, j - 1, k) + fetch(g, u, COMP_U, i + 1, j, k)));
    double fb = xwall(g, i) ? 0.0 : (0.5 * (fetch(g, v, COMP_V, i - 1, j, k) + c0)) *
                                    (0.5 * (fetch(g, u, COMP_U, i, j - 1, k) + fetch(g, u, COMP_U, i, j, k)));
    double fx = (fa - fb) * g->rdx;
    double vcp = 0.5 * (c0 + fetch(g, v, COMP_V, i, j + 1, k));
    double vcm = 0.5 * (fetch(g, v, COMP_V, i, j - 1, k) + c0);
    double fy = (vcp * vcp - vcm * vcm) * g->rdy;
    double ga = zwall(g, k + 1) ? 0.0 : (0.5 * (c0 + fetch(g, v, COMP_V, i, j, k + 1))) *
                                        (0.5 * (fetch(g, w, COMP_W, i, j - 1, k + 1) + fetch(g, w, COMP_W, i, j, k + 1)));
    double gb = zwall(g, k) ? 0.0 : (0.5 * (fetch(g, v, COMP_V, i, j, k - 1) + c0)) *
                                    (0.5 * (fetch(g, w, COMP_W, i, j - 1, k) + fetch(g, w, COMP_W, i, j, k)));
    double fz = (ga - gb) * g->rdzc[k];
    return -((fx + fy) + fz);
}
static inline double conv_w(const sgrid *g, const double *u, const double *v, const double *w, int i, int j, int k)
{
    double c0 = fetch(g, w, COMP_W, i, j, k);
    double fa = xwall(g, i + 1) ? 0.0 : (0.5 * (c0 + fetch(g, w, COMP_W, i + 1, j, k))) *
                                        (0.5 * (fetch(g, u, COMP_U, i + 1, j, k - 1) + fetch(g, u, COMP_U, i + 1, j, k)));
    double fb = xwall(g, i) ? 0.0 : (0.5 * (fetch(g, w, COMP_W, i - 1, j, k) + c0)) *
                                    (0.5 * (fetch(g, u, COMP_U, i, j, k - 1) + fetch(g, u, COMP_U, i, j, k)));
    double fx = (fa - fb) * g->rdx;
    double ga = ywall(g, j + 1) ? 0.0 : (0.5 * (c0 + fetch(g, w, COMP_W, i, j + 1, k))) *
                                        (0.5 * (fetch(g, v, COMP_V, i, j + 1, k - 1) + fetch(g, v, COMP_V, i, j + 1, k)));
    double gb = ywall(g, j) ? 0.0 : (0.5 * (fetch(g, w, COMP_W, i, j - 1, k) + c0)) *
                                    (0.5 * (fetch(g, v, COMP_V, i, j, k - 1) + fetch(g, v, COMP_V, i, j, k)));
    double fy = (ga - gb) * g->rdy;
    double wcp = 0.5 * (c0 + fetch(g, w, COMP_W, i, j, k + 1));
    double wcm = 0.5 * (fetch(g, w, COMP_W, i, j, k - 1) + c0);
    double fz = (wcp * wcp - wcm * wcm) * g->rdzm[k];
    return -((fx + fy) + fz);
}

static int sgrid_init(sgrid *g, int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y)
{
    double *rc = malloc(sizeof(double) * nz), *rm = malloc(sizeof(double) * nz);
    if (!rc || !rm) return 4;
    zmetric_double(nz, zc, rc, rm);
    g->nx = nx; g->ny = ny; g->nz = nz; g->bc_x = bc_x; g->bc_y = bc_y;
    g->rdx = 1.0 / (Lx / (double)nx); g->rdy = 1.0 / (Ly / (double)ny);
    g->rdzc = rc; g->rdzm = rm;
    return 0;
}
static void sgrid_free(sgrid *g) { free((void *)g->rdzc); free((void *)g->rdzm); }

/* H = -div(u u): the three components at their own positions; wall rows 0. */
int oracle_convective(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                      const double *u, const double *v, const double *w, double *hu, double *hv, double *hw)
{
    sgrid g;
    if (sgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y)) return 4;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                size_t t = IDX(i, j, k);
                double a = wall_row(&g, COMP_U, i, j, k) ? 0.0 : conv_u(&g, u, v, w, i, j, k);
                double b = wall_row(&g, COMP_V, i, j, k) ? 0.0 : conv_v(&g, u, v, w, i, j, k);
                double c = wall_row(&g, COMP_W, i, j, k) ? 0.0 : conv_w(&g, u, v, w, i, j, k);
                hu[t] = a; hv[t] = b; hw[t] = c;
            }
    sgrid_free(&g);
    return 0;
}

/* out = lap q at the position of component comp (exported for the pins). */
int oracle_velocity_laplacian(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                              int comp, const double *q, double *out)
{
    sgrid g;
    if (sgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y)) return 4;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) out[IDX(i, j, k)] = vel_lap(&g, q, comp, i, j, k);
    sgrid_free(&g);
    return 0;
}

/* NEXT-2: rhs of the implicit step and the new H (stored over H^{n-1}).  u, v, w, p are read only. */
int oracle_explicit_terms(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                          const double *u, const double *v, const double *w, const double *p,
                          const double *fu, const double *fv, const double *fw,
                          double *hu, double *hv, double *hw, double *ru, double *rv, double *rw,
                          double gamma_dt, double rho_dt, double alpha_dt, double beta)
{
    sgrid g;
    if (sgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y)) return 4;
    size_t N = (size_t)nx * ny * nz;
    double *nu = malloc(sizeof(double) * N), *nv = malloc(sizeof(double) * N), *nw = malloc(sizeof(double) * N);
    if (!nu || !nv || !nw) return 4;
    int rc = oracle_convective(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, u, v, w, nu, nv, nw);
    if (rc) return rc;
    const double tb = 2.0 * beta;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                size_t t = IDX(i, j, k);
                double c0 = p[t];
                if (wall_row(&g, COMP_U, i, j, k)) ru[t] = 0.0;
                else {
                    double gp = (c0 - p[IDX(wrapi(i - 1, nx), j, k)]) * g.rdx;
                    ru[t] = ((gamma_dt * nu[t] + rho_dt * hu[t]) - alpha_dt * gp) + tb * vel_lap(&g, u, COMP_U, i, j, k);
                    if (fu) ru[t] = ru[t] + alpha_dt * fu[t];
                }
                if (wall_row(&g, COMP_V, i, j, k)) rv[t] = 0.0;
                else {
                    double gp = (c0 - p[IDX(i, wrapi(j - 1, ny), k)]) * g.rdy;
                    rv[t] = ((gamma_dt * nv[t] + rho_dt * hv[t]) - alpha_dt * gp) + tb * vel_lap(&g, v, COMP_V, i, j, k);
                    if (fv) rv[t] = rv[t] + alpha_dt * fv[t];
                }
                if (wall_row(&g, COMP_W, i, j, k)) rw[t] = 0.0;
                else {
                    double gp = (c0 - p[IDX(i, j, k - 1)]) * g.rdzm[k];
                    rw[t] = ((gamma_dt * nw[t] + rho_dt * hw[t]) - alpha_dt * gp) + tb * vel_lap(&g, w, COMP_W, i, j, k);
                    if (fw) rw[t] = rw[t] + alpha_dt * fw[t];
                }
            }
    memcpy(hu, nu, sizeof(double) * N); memcpy(hv, nv, sizeof(double) * N); memcpy(hw, nw, sizeof(double) * N);
    free(nu); free(nv); free(nw);
    sgrid_free(&g);
    return 0;
}
