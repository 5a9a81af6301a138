/*
 * fsei_ibm_oracle.c -- CPU ORACLE for the IB-MLS transfer operators.  TEST INFRASTRUCTURE
 * (same rules as fsei_oracle.c: loaded only by tests/, __graft_entry__.smoke() and bench.py's CPU legs; shares no code,
 * header, table or constant with paper_2103_15187_b200/).
 *
 * What it follows (P:Lnnn = /root/reference/PAPER.md line nnn):
 *   "the no-slip boundary condition is then imposed on some Lagrangian markers ... and then transferred to several
 *   Eulerian grid-points ...  A three-dimensional support domain consisting of N_e = n x n x n Eulerian nodes (n = 3 is
 *   typically used) is created around each Lagrangian marker, and the fluid velocity at the body position is computed
 *   interpolating the velocity of the N_e Eulerian grid-points in the support domain as
 *        u_i(x_b) = sum_{k=1..N_e} phi_i^k(x_b) u_i(x_k)                                   (Eq. 4)
 *   where the phi_i^k are the transfer operators ... a linear basis function is used, p^T(x) = [1, x, y, z], with an
 *   exponential weight function centered at the location of the Lagrangian marker [17].  The interpolated velocity (4)
 *   is used to compute the IB force at the exact location of the marker which is then transferred back to the Eulerian
 *   grid-points as a distributed forcing.  This procedure is applied to all Lagrangian markers for the three velocity
 *   components"                                                                         (Fig. 2, sec. 2.1)
 *   "the 4x4 system of equations that has to be solved for each Lagrangian marker to compute the phi_i^k weights"
 *                                                                                      (sec. 3.2)
 * The paper prints no formula for the weight, the force or the spreading; they are the moving-least-squares
 * construction of its refs [15]-[17], recorded as readings M1..M8 in DESIGN.md sec. 3:
 *   M1 support: the 3 x 3 x 3 nodes of the component's OWN staggered grid around the node nearest to the marker
 *      (periodic wrap in a periodic direction; in a wall direction the centre index is clamped to [1, n-2])
 *   M2 weight: W_k = exp(-(r_k/eps)^2), eps = 0.3, r_k^2 = sum_d ((x_k,d - x_b,d)/(1.5 h_d))^2, h_x = dx, h_y = dy,
 *      h_z = half the distance between the two outer z-nodes of the support (no cut-off: the 27 nodes all carry weight)
 *   M3 shape functions: phi^k = p^T(x_b) A^-1 W_k p(x_k),  A = sum_k W_k p(x_k) p^T(x_k)   (4 x 4, symmetric)
 *      evaluated with the basis written in marker-centred, spacing-scaled coordinates xi_d = (x_d - x_b,d)/h_d
 *      (span{1,x,y,z} is invariant under affine maps, so phi is the same; p(x_b) = e_0)
 *   M4 interpolation: U_c(l) = sum_k phi^k u_c(x_k)                                           (Eq. 4)
 *   M5 force at the marker: F_c(l) = (V_c(l) - U_c(l)) * inv_dt      (V = velocity of the body at the marker)
 *   M6 spreading: f_c(x_k) += c_l phi^k F_c(l),  c_l = dV_l / sum_k phi^k dV_k,  dV_l = A_l h_l,
 *      h_l = (dx + dy + dz_kc)/3, dV_k = dx dy dz_k the control volume of node k (dz_k = dzc[k] for u, v; dzm[k] for w):
 *      the total force is conserved, sum_k f_k dV_k = sum_l F_l dV_l
 *   M7 node positions: u at (i dx, (j+1/2) dy, zm[k]); v at ((i+1/2) dx, j dy, zm[k]); w at ((i+1/2) dx, (j+1/2) dy, zc[k])
 *   M8 a marker's position is taken modulo the period in a periodic direction.
 * Arithmetic in real_t (long double in the parity build).
 */
#include <math.h>
#include <stdlib.h>
#include <stddef.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real_t;
#define R_EXP expl
#define R_FLOOR floorl
#define R_FABS fabsl
#else
typedef double real_t;
#define R_EXP exp
#define R_FLOOR floor
#define R_FABS fabs
#endif

enum { BC_P = 0, BC_W = 1 };
#define MLS_EPS ((real_t)0.3)

typedef struct {
    int nx, ny, nz, bc_x, bc_y;
    real_t dx, dy, Lx, Ly;
    const double *zc;
} mgrid;

/* coordinate of node m of component comp along z (M7), and its control-volume height */
static real_t znode(const mgrid *g, int comp, int k) { return comp == 2 ? (real_t)g->zc[k] : ((real_t)g->zc[k] + (real_t)g->zc[k + 1]) / 2; }
static real_t zvol(const mgrid *g, int comp, int k)
{
    if (comp != 2) return (real_t)g->zc[k + 1] - (real_t)g->zc[k];
    if (k == 0) return 0;
    return ((real_t)g->zc[k] + (real_t)g->zc[k + 1]) / 2 - ((real_t)g->zc[k - 1] + (real_t)g->zc[k]) / 2;
}

/* nearest node along a uniform direction: nodes at (m + off) h; returns the centre index and the marker coordinate
   reduced to the period (M8) */
static int nearest_uniform(real_t x, real_t h, real_t off, int n, int periodic, real_t L, real_t *xred)
{
    if (periodic) x -= R_FLOOR(x / L) * L;
    *xred = x;
    int c = (int)R_FLOOR(x / h - off + (real_t)0.5);
    if (periodic) { if (c < 0) c += n; if (c >= n) c -= n; }
    else { if (c < 1) c = 1; if (c > n - 2) c = n - 2; }
    return c;
}

/* The 27 shape functions of marker (xb, yb, zb) for component comp: node linear indices idx[27] (x fastest within
   the support: s = (dk*3 + dj)*3 + di), phi[27], and the control volumes vol[27].  Returns h_l through *hl. */
static int mls_weights(const mgrid *g, int comp, real_t xb, real_t yb, real_t zb, size_t *idx, real_t *phi, real_t *vol, real_t *hl)
{
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    real_t xr, yr;
    int ic = nearest_uniform(xb, g->dx, comp == 0 ? 0 : (real_t)0.5, nx, g->bc_x == BC_P, g->Lx, &xr);
    int jc = nearest_uniform(yb, g->dy, comp == 1 ? 0 : (real_t)0.5, ny, g->bc_y == BC_P, g->Ly, &yr);
    int kc = 0;                                            /* nearest z node, clamped to [1, nz-2] */
    real_t best = -1;
    for (int k = 0; k < nz; k++) { real_t d = R_FABS(znode(g, comp, k) - zb); if (best < 0 || d < best) { best = d; kc = k; } }
    if (kc < 1) kc = 1;
    if (kc > nz - 2) kc = nz - 2;
    real_t hz = (znode(g, comp, kc + 1) - znode(g, comp, kc - 1)) / 2;
    real_t A[4][5] = {{0}}, W[27], P[27][4];
    for (int dk = -1; dk <= 1; dk++)
        for (int dj = -1; dj <= 1; dj++)
            for (int di = -1; di <= 1; di++) {
                int s = ((dk + 1) * 3 + (dj + 1)) * 3 + (di + 1);
                int i = ic + di, j = jc + dj, k = kc + dk;
                /* node coordinates, unwrapped so that the support is contiguous around the (reduced) marker */
                real_t xk = ((real_t)i + (comp == 0 ? 0 : (real_t)0.5)) * g->dx;
                real_t yk = ((real_t)j + (comp == 1 ? 0 : (real_t)0.5)) * g->dy;
                if (g->bc_x == BC_P) { if (xk - xr > g->Lx / 2) xk -= g->Lx; if (xr - xk > g->Lx / 2) xk += g->Lx; i = ((i % nx) + nx) % nx; }
                if (g->bc_y == BC_P) { if (yk - yr > g->Ly / 2) yk -= g->Ly; if (yr - yk > g->Ly / 2) yk += g->Ly; j = ((j % ny) + ny) % ny; }
                real_t zk = znode(g, comp, k);
                real_t xi = (xk - xr) / g->dx, et = (yk - yr) / g->dy, ze = (zk - zb) / hz;
                real_t r2 = (xi * xi + et * et + ze * ze) / ((real_t)1.5 * (real_t)1.5);
                W[s] = R_EXP(-r2 / (MLS_EPS * MLS_EPS));
                P[s][0] = 1; P[s][1] = xi; P[s][2] = et; P[s][3] = ze;
                for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) A[a][b] += W[s] * P[s][a] * P[s][b];
                idx[s] = ((size_t)k * ny + j) * nx + i;
                vol[s] = g->dx * g->dy * zvol(g, comp, k);
            }
    /* solve A lam = e_0 (M3: p(x_b) = e_0 in marker-centred coordinates), Gaussian elimination with partial pivoting */
    A[0][4] = 1; A[1][4] = 0; A[2][4] = 0; A[3][4] = 0;
    for (int c = 0; c < 4; c++) {
        int piv = c;
        for (int r = c + 1; r < 4; r++) if (R_FABS(A[r][c]) > R_FABS(A[piv][c])) piv = r;
        if (A[piv][c] == 0) return 1;
        if (piv != c) for (int b = 0; b < 5; b++) { real_t t = A[c][b]; A[c][b] = A[piv][b]; A[piv][b] = t; }
        for (int r = c + 1; r < 4; r++) {
            real_t m = A[r][c] / A[c][c];
            for (int b = c; b < 5; b++) A[r][b] -= m * A[c][b];
        }
    }
    real_t lam[4];
    for (int c = 3; c >= 0; c--) {
        real_t s = A[c][4];
        for (int b = c + 1; b < 4; b++) s -= A[c][b] * lam[b];
        lam[c] = s / A[c][c];
    }
    for (int s = 0; s < 27; s++) phi[s] = W[s] * (lam[0] * P[s][0] + lam[1] * P[s][1] + lam[2] * P[s][2] + lam[3] * P[s][3]);
    *hl = (g->dx + g->dy + zvol(g, comp == 2 ? 2 : 0, kc)) / 3;
    return 0;
}

static void mgrid_init(mgrid *g, int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y)
{
    g->nx = nx; g->ny = ny; g->nz = nz; g->bc_x = bc_x; g->bc_y = bc_y; g->Lx = Lx; g->Ly = Ly;
    g->dx = (real_t)Lx / nx; g->dy = (real_t)Ly / ny; g->zc = zc;
}

/* shape functions of one marker (exported for the pins) */
int oracle_mls_weights(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                       int comp, double xb, double yb, double zb, long *idx, double *phi)
{
    mgrid g; mgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y);
    size_t id[27]; real_t ph[27], vol[27], hl;
    if (nx < 3 || ny < 3 || nz < 3) return 2;
    int rc = mls_weights(&g, comp, xb, yb, zb, id, ph, vol, &hl);
    for (int s = 0; s < 27; s++) { idx[s] = (long)id[s]; phi[s] = (double)ph[s]; }
    return rc;
}

/* M4: ub[c][l] = sum_k phi^k q_c(x_k) for the three components (ub: 3 arrays of n) */
int oracle_mls_interpolate(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                           long n, const double *xm, const double *ym, const double *zm,
                           const double *u, const double *v, const double *w, double *ub, double *vb, double *wb)
{
    mgrid g; mgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y);
    const double *q[3] = {u, v, w};
    double *o[3] = {ub, vb, wb};
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (long l = 0; l < n; l++)
        for (int c = 0; c < 3; c++) {
            size_t id[27]; real_t ph[27], vol[27], hl, s = 0;
            bad |= mls_weights(&g, c, xm[l], ym[l], zm[l], id, ph, vol, &hl);
            for (int k = 0; k < 27; k++) s += ph[k] * (real_t)q[c][id[k]];
            o[c][l] = (double)s;
        }
    return bad;
}

/* M6: f_c(x_k) += c_l phi^k F_c(l) (serial over the markers: the oracle's sums have one fixed order) */
int oracle_mls_spread(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                      long n, const double *xm, const double *ym, const double *zm, const double *area,
                      const double *Fu, const double *Fv, const double *Fw, double *fu, double *fv, double *fw)
{
    mgrid g; mgrid_init(&g, nx, ny, nz, Lx, Ly, zc, bc_x, bc_y);
    const double *F[3] = {Fu, Fv, Fw};
    double *f[3] = {fu, fv, fw};
    size_t N = (size_t)nx * ny * nz;
    for (int c = 0; c < 3; c++) {
        real_t *acc = calloc(N, sizeof(real_t));
        if (!acc) return 4;
        for (long l = 0; l < n; l++) {
            size_t id[27]; real_t ph[27], vol[27], hl, den = 0;
            if (mls_weights(&g, c, xm[l], ym[l], zm[l], id, ph, vol, &hl)) { free(acc); return 1; }
            for (int k = 0; k < 27; k++) den += ph[k] * vol[k];
            real_t cl = (real_t)area[l] * hl / den;
            for (int k = 0; k < 27; k++) acc[id[k]] += cl * ph[k] * (real_t)F[c][l];
        }
        for (size_t t = 0; t < N; t++) f[c][t] = (double)((real_t)f[c][t] + acc[t]);
        free(acc);
    }
    return 0;
}

/* M4-M6 chained: interpolate, F = (V - U) inv_dt, spread.  Fb (3 arrays of n) receives the marker forces. */
int oracle_ibm_forcing(int nx, int ny, int nz, double Lx, double Ly, const double *zc, int bc_x, int bc_y,
                       long n, const double *xm, const double *ym, const double *zm, const double *area,
                       const double *Vu, const double *Vv, const double *Vw,
                       const double *u, const double *v, const double *w, double inv_dt,
                       double *Fu, double *Fv, double *Fw, double *fu, double *fv, double *fw)
{
    int rc = oracle_mls_interpolate(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, n, xm, ym, zm, u, v, w, Fu, Fv, Fw);
    if (rc) return rc;
    for (long l = 0; l < n; l++) {
        Fu[l] = (Vu[l] - Fu[l]) * inv_dt; Fv[l] = (Vv[l] - Fv[l]) * inv_dt; Fw[l] = (Vw[l] - Fw[l]) * inv_dt;
    }
    return oracle_mls_spread(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, n, xm, ym, zm, area, Fu, Fv, Fw, fu, fv, fw);
}
