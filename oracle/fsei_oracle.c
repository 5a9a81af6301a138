/*
 * fsei_oracle.c -- CPU ORACLE for the pressure projection.  TEST INFRASTRUCTURE.
 *
 * This file is the plain, slow, obviously-correct definition of what the hot
 * path computes.  It is test infrastructure: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  The product
 * (paper_2103_15187_b200/) never includes, links or calls anything in oracle/,
 * and this file shares no code, header, table or constant with the CUDA path.
 *
 * What it follows (P:Lnnn = /root/reference/PAPER.md line nnn):
 *   - central second-order finite differences on a staggered mesh      (sec. 2.1)
 *   - fractional-step method, pressure as Lagrange multiplier that
 *     enforces the solenoidal condition                                (sec. 2.1, Eq. 3)
 *   - periodic x,y, wall-normal z                                      (Fig. 4)
 *   - FFT as the external routine for the elliptic solve
 *   - Thomas' algorithm for tridiagonal systems                        (sec. 3.1)
 *   - the elliptic equation imposing mass conservation                 (sec. 4)
 * The paper prints no equation for the projection itself; every detail below is
 * the reading recorded in DESIGN.md section 3 (R1..R20).
 *
 * The method is DIRECT: it reaches, up to rounding and the gauge, the exact
 * solution of  D G phi = D u* / (alpha dt).  So the oracle is that definition
 * written out: full complex DFTs of every x-line and y-line (no half-spectrum
 * trick, no blocking, no fusion), one Thomas solve per wavenumber pair, inverse
 * DFTs.  real_t is `long double` (x87 80-bit) in the parity build and `double`
 * in the timed cpu_baseline build of the same source.
 *
 * Stencil steps (divergence, projection) are ALWAYS computed in IEEE double in
 * a fixed operation order with no FMA contraction (compile with
 * -ffp-contract=off): the paper's precision is double and the order is
 * reading R20, so a CUDA kernel that keeps the same order matches bit for bit.
 *
 * Pins (tests/test_oracle_*.py): discrete eigenfunctions with modified
 * wavenumbers, dense brute force D*G on 8x8x8, manufactured solutions,
 * post-projection divergence, gauge, FFT/DCT against O(n^2) definitions,
 * Thomas against dense solves.  Nothing here is "parity unpinned".
 *
 * Layout: all fields are C-order [nz][ny][nx], x fastest.
 */
#include <math.h>
#include <float.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real_t;
#define R_COS cosl
#define R_SIN sinl
#define R_PI 3.14159265358979323846264338327950288L
#else
typedef double real_t;
#define R_COS cos
#define R_SIN sin
#define R_PI 3.14159265358979323846264338327950288
#endif

enum { ORACLE_BC_PERIODIC = 0, ORACLE_BC_NEUMANN = 1 };

/* Mantissa bits of the arithmetic type of the solve (53 = double, 64 = x87). */
int oracle_real_mant_bits(void) { return (int)(sizeof(real_t) == sizeof(double) ? DBL_MANT_DIG : LDBL_MANT_DIG); }

#define IDX(i, j, k) (((size_t)(k) * (size_t)ny + (size_t)(j)) * (size_t)nx + (size_t)(i))

/* ------------------------------------------------------------------------- */
/* Discrete Fourier transform: recursive decimation in time, radix 2 and 3,   */
/* O(n^2) definition for any other length.  w[] is the table e^{s 2 pi i m/n0}*/
/* of the top-level length n0; a sub-transform of length n uses stride n0/n.  */
/* ------------------------------------------------------------------------- */
static void dft_rec(int n, const real_t *xr, const real_t *xi, int xs,
                    real_t *yr, real_t *yi, const real_t *wr, const real_t *wi, int ws)
{
    if (n == 1) { yr[0] = xr[0]; yi[0] = xi[0]; return; }
    if (n % 2 == 0) {
        int h = n / 2;
        dft_rec(h, xr, xi, 2 * xs, yr, yi, wr, wi, 2 * ws);                      /* even samples */
        dft_rec(h, xr + xs, xi + xs, 2 * xs, yr + h, yi + h, wr, wi, 2 * ws);    /* odd samples  */
        for (int k = 0; k < h; k++) {
            real_t er = yr[k], ei = yi[k], pr = yr[k + h], pi = yi[k + h];
            real_t tr = wr[k * ws] * pr - wi[k * ws] * pi;                       /* w^k * O[k]   */
            real_t ti = wr[k * ws] * pi + wi[k * ws] * pr;
            yr[k] = er + tr;     yi[k] = ei + ti;
            yr[k + h] = er - tr; yi[k + h] = ei - ti;
        }
        return;
    }
    if (n % 3 == 0) {
        int t = n / 3;
        for (int r = 0; r < 3; r++)
            dft_rec(t, xr + r * xs, xi + r * xs, 3 * xs, yr + r * t, yi + r * t, wr, wi, 3 * ws);
        for (int k = 0; k < t; k++) {
            real_t ar[3], ai[3];
            for (int r = 0; r < 3; r++) { ar[r] = yr[k + r * t]; ai[r] = yi[k + r * t]; }
            for (int q = 0; q < 3; q++) {                    /* output index k + q t */
                real_t sr = ar[0], si = ai[0];
                for (int r = 1; r < 3; r++) {
                    int m = (int)(((long)r * (long)(k + q * t)) % n);            /* w_n^{r (k+qt)} */
                    sr += wr[m * ws] * ar[r] - wi[m * ws] * ai[r];
                    si += wr[m * ws] * ai[r] + wi[m * ws] * ar[r];
                }
                yr[k + q * t] = sr; yi[k + q * t] = si;
            }
        }
        return;
    }
    for (int k = 0; k < n; k++) {                            /* definition */
        real_t sr = 0, si = 0;
        for (int j = 0; j < n; j++) {
            int m = (int)(((long)j * (long)k) % n);
            sr += wr[m * ws] * xr[j * xs] - wi[m * ws] * xi[j * xs];
            si += wr[m * ws] * xi[j * xs] + wi[m * ws] * xr[j * xs];
        }
        yr[k] = sr; yi[k] = si;
    }
}

typedef struct { int n; real_t *wf_r, *wf_i, *wb_r, *wb_i; } dft_table;

static void dft_table_init(dft_table *t, int n)
{
    t->n = n;
    t->wf_r = malloc(sizeof(real_t) * n); t->wf_i = malloc(sizeof(real_t) * n);
    t->wb_r = malloc(sizeof(real_t) * n); t->wb_i = malloc(sizeof(real_t) * n);
    for (int m = 0; m < n; m++) {
        real_t a = 2 * R_PI * (real_t)m / (real_t)n;
        t->wf_r[m] = R_COS(a); t->wf_i[m] = -R_SIN(a);       /* forward  e^{-2 pi i m/n} (R15) */
        t->wb_r[m] = R_COS(a); t->wb_i[m] = R_SIN(a);        /* backward e^{+2 pi i m/n}       */
    }
}
static void dft_table_free(dft_table *t) { free(t->wf_r); free(t->wf_i); free(t->wb_r); free(t->wb_i); }

/* y = DFT(x) (sign<0, unnormalised) or y = inverse DFT(x) incl. 1/n (sign>0). */
static void dft_apply(const dft_table *t, int sign, const real_t *xr, const real_t *xi,
                      real_t *yr, real_t *yi)
{
    int n = t->n;
    if (sign < 0) dft_rec(n, xr, xi, 1, yr, yi, t->wf_r, t->wf_i, 1);
    else {
        dft_rec(n, xr, xi, 1, yr, yi, t->wb_r, t->wb_i, 1);
        for (int k = 0; k < n; k++) { yr[k] /= (real_t)n; yi[k] /= (real_t)n; }
    }
}

/* ------------------------------------------------------------------------- */
/* Cosine transforms (reading R15):                                           */
/*   DCT-II   X_k = sum_j x_j cos(pi k (j+1/2)/n)                  unnormalised*/
/*   inverse  x_j = (X_0 + 2 sum_{k>=1} X_k cos(pi k (j+1/2)/n))/n             */
/* computed through the even extension y of length 2n (y_j = y_{2n-1-j} = x_j)*/
/* for which  Y_k = 2 e^{i pi k/(2n)} X_k.  t2 is the length-2n table.        */
/* ------------------------------------------------------------------------- */
static void dct2_apply(const dft_table *t2, const real_t *x, real_t *X, real_t *work /* 8n */)
{
    int n = t2->n / 2;
    real_t *yr = work, *yi = work + 2 * n, *Yr = work + 4 * n, *Yi = work + 6 * n;
    for (int j = 0; j < n; j++) { yr[j] = x[j]; yr[2 * n - 1 - j] = x[j]; }
    for (int j = 0; j < 2 * n; j++) yi[j] = 0;
    dft_apply(t2, -1, yr, yi, Yr, Yi);
    for (int k = 0; k < n; k++) {
        real_t a = R_PI * (real_t)k / (real_t)(2 * n);
        X[k] = (R_COS(a) * Yr[k] + R_SIN(a) * Yi[k]) / 2;     /* Re(e^{-ia} Y_k)/2 */
    }
}
static void dct3_apply(const dft_table *t2, const real_t *X, real_t *x, real_t *work /* 8n */)
{
    int n = t2->n / 2;
    real_t *Yr = work, *Yi = work + 2 * n, *yr = work + 4 * n, *yi = work + 6 * n;
    for (int k = 0; k < n; k++) {
        real_t a = R_PI * (real_t)k / (real_t)(2 * n);
        Yr[k] = 2 * R_COS(a) * X[k]; Yi[k] = 2 * R_SIN(a) * X[k];
    }
    Yr[n] = 0; Yi[n] = 0;
    for (int k = 1; k < n; k++) { Yr[2 * n - k] = Yr[k]; Yi[2 * n - k] = -Yi[k]; }
    dft_apply(t2, +1, Yr, Yi, yr, yi);
    for (int j = 0; j < n; j++) x[j] = yr[j];
}

/* ------------------------------------------------------------------------- */
/* Thomas' algorithm for  a_k x_{k-1} + b_k x_k + c_k x_{k+1} = d_k. */
/* a[0] and c[n-1] are not referenced.  cp is scratch of length n.            */
/* ------------------------------------------------------------------------- */
static void thomas(int n, const real_t *a, const real_t *b, const real_t *c,
                   const real_t *d, real_t *x, real_t *cp)
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

/* Wall-normal metric coefficients of L = D G (readings R2, R5, R20).          */
/* The metrics are fp64 DATA of the grid, evaluated once in double exactly as  */
/* the stencils a1 / a7 evaluate them (zmetric_double below):                  */
/*   dzc[k] = zc[k+1]-zc[k]                     cell heights,   k = 0..nz-1    */
/*   dzm[k] = (zc[k]+zc[k+1])/2 - (zc[k-1]+zc[k])/2  centre spacings, k >= 1   */
/*   rdzc = 1/dzc, rdzm = 1/dzm                 (each rounded to double)       */
/* and L = D G is the product of those very stencils (R5), so                  */
/*   a_k = rdzm[k] rdzc[k] (a_0 = 0),  c_k = rdzm[k+1] rdzc[k] (c_{nz-1} = 0)  */
/* with the products (and everything after) in real_t.  Evaluating the metrics */
/* in real_t instead would solve an operator that differs from the stencils'   */
/* by up to ulp(zc)/dz ~ 1e-12 near the upper wall and leave a post-projection */
/* divergence ~30x above the fp64 floor (R5).                        */
static void zcoef(int nz, const double *zc, real_t *dzc, real_t *dzm, real_t *a, real_t *c)
{
    double *rc = malloc(sizeof(double) * nz), *rm = malloc(sizeof(double) * nz);
    for (int k = 0; k < nz; k++) {
        double hc = zc[k + 1] - zc[k];
        dzc[k] = (real_t)hc;
        rc[k] = 1.0 / hc;
    }
    dzm[0] = 0; rm[0] = 0.0;
    for (int k = 1; k < nz; k++) {
        double hm = 0.5 * (zc[k] + zc[k + 1]) - 0.5 * (zc[k - 1] + zc[k]);
        dzm[k] = (real_t)hm;
        rm[k] = 1.0 / hm;
    }
    for (int k = 0; k < nz; k++) {
        a[k] = (k > 0) ? (real_t)rm[k] * (real_t)rc[k] : 0;
        c[k] = (k < nz - 1) ? (real_t)rm[k + 1] * (real_t)rc[k] : 0;
    }
    free(rc); free(rm);
}

/* Modified wavenumbers (reading R6; the periodic form is B:north_star's):    */
/*   periodic  (2 cos(2 pi m/n) - 2)/h^2,   Neumann  (2 cos(pi m/n) - 2)/h^2  */
static void modified_wavenumbers(int n, double L, int bc, real_t *lam)
{
    real_t h = (real_t)L / (real_t)n;
    for (int m = 0; m < n; m++) {
        real_t ang = (bc == ORACLE_BC_PERIODIC ? 2 : 1) * R_PI * (real_t)m / (real_t)n;
        lam[m] = (2 * R_COS(ang) - 2) / (h * h);
    }
}

/* The (kx,ky)=(0,0) column (readings R7, R8): the operator is singular there.*/
/* Flux form of the equation: with G_k the gradient at face k (G_0 = G_nz = 0)*/
/*   G_{k+1} - G_k = rhs_k dzc[k]   =>  F_k = F_{k-1} + rhs_{k-1} dzc[k-1]    */
/*   phi_k = phi_{k-1} + F_k dzm[k],  phi_0 = 0 (pinned),                     */
/* then shifted to the volume-weighted zero mean  sum_k phi_k dzc[k] = 0.     */
static void gauge_column(int nz, const real_t *dzc, const real_t *dzm, const real_t *d, real_t *x)
{
    real_t F = 0, vol = 0, acc = 0;
    x[0] = 0;
    for (int k = 1; k < nz; k++) {
        F += d[k - 1] * dzc[k - 1];
        x[k] = x[k - 1] + F * dzm[k];
    }
    for (int k = 0; k < nz; k++) { acc += x[k] * dzc[k]; vol += dzc[k]; }
    real_t mean = acc / vol;
    for (int k = 0; k < nz; k++) x[k] -= mean;
}

/* ------------------------------------------------------------------------- */
/* Step a1: rhs = D u* / (alpha dt)  (readings R4, R20).        */
/* Element [k][j][i] of u/v/w is the value on the LOW x/y/z face of cell      */
/* (i,j,k).  Periodic direction: face n == face 0.  Wall direction: the high  */
/* wall face is not stored and is 0; stored face 0 is the low wall.           */
/* Always IEEE double, fixed order:                                           */
/*   ((du*rdx + dv*rdy) + dw*rdzc[k]) * (1/alpha_dt)                          */
/* ------------------------------------------------------------------------- */
int oracle_divergence(int nx, int ny, int nz, double Lx, double Ly, const double *zc,
                      int bc_x, int bc_y, const double *u, const double *v, const double *w,
                      double alpha_dt, double *rhs)
{
    if (nx < 1 || ny < 1 || nz < 2 || alpha_dt == 0.0) return 1;
    const double rdx = 1.0 / (Lx / (double)nx), rdy = 1.0 / (Ly / (double)ny);
    const double inv_adt = 1.0 / alpha_dt;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++) {
        const double rdz = 1.0 / (zc[k + 1] - zc[k]);
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                double up = (i + 1 < nx) ? u[IDX(i + 1, j, k)] : (bc_x == ORACLE_BC_PERIODIC ? u[IDX(0, j, k)] : 0.0);
                double vp = (j + 1 < ny) ? v[IDX(i, j + 1, k)] : (bc_y == ORACLE_BC_PERIODIC ? v[IDX(i, 0, k)] : 0.0);
                double wp = (k + 1 < nz) ? w[IDX(i, j, k + 1)] : 0.0;
                double du = up - u[IDX(i, j, k)];
                double dv = vp - v[IDX(i, j, k)];
                double dw = wp - w[IDX(i, j, k)];
                rhs[IDX(i, j, k)] = ((du * rdx + dv * rdy) + dw * rdz) * inv_adt;
            }
    }
    return 0;
}

/* L phi = D G phi, the 7-point operator of a1 after a7 (reading R5), in double,*/
/* fixed order  ((gxp-gxm)*rdx + (gyp-gym)*rdy) + (gzp-gzm)*rdzc[k]           */
/* with face gradients g = (phi_hi - phi_lo)*r and 0 on wall faces.           */
static inline double lap_at(int nx, int ny, int nz, int bc_x, int bc_y, const double *phi,
                            double rdx, double rdy, const double *rdzc, const double *rdzm,
                            int i, int j, int k)
{
    double c0 = phi[IDX(i, j, k)];
    double gxm, gxp, gym, gyp, gzm, gzp;
    if (i > 0) gxm = (c0 - phi[IDX(i - 1, j, k)]) * rdx;
    else gxm = (bc_x == ORACLE_BC_PERIODIC) ? (c0 - phi[IDX(nx - 1, j, k)]) * rdx : 0.0;
    if (i + 1 < nx) gxp = (phi[IDX(i + 1, j, k)] - c0) * rdx;
    else gxp = (bc_x == ORACLE_BC_PERIODIC) ? (phi[IDX(0, j, k)] - c0) * rdx : 0.0;
    if (j > 0) gym = (c0 - phi[IDX(i, j - 1, k)]) * rdy;
    else gym = (bc_y == ORACLE_BC_PERIODIC) ? (c0 - phi[IDX(i, ny - 1, k)]) * rdy : 0.0;
    if (j + 1 < ny) gyp = (phi[IDX(i, j + 1, k)] - c0) * rdy;
    else gyp = (bc_y == ORACLE_BC_PERIODIC) ? (phi[IDX(i, 0, k)] - c0) * rdy : 0.0;
    gzm = (k > 0) ? (c0 - phi[IDX(i, j, k - 1)]) * rdzm[k] : 0.0;
    gzp = (k + 1 < nz) ? (phi[IDX(i, j, k + 1)] - c0) * rdzm[k + 1] : 0.0;
    return ((gxp - gxm) * rdx + (gyp - gym) * rdy) + (gzp - gzm) * rdzc[k];
}

static void zmetric_double(int nz, const double *zc, double *rdzc, double *rdzm)
{
    for (int k = 0; k < nz; k++) rdzc[k] = 1.0 / (zc[k + 1] - zc[k]);
    rdzm[0] = 0.0;
    for (int k = 1; k < nz; k++) rdzm[k] = 1.0 / (0.5 * (zc[k] + zc[k + 1]) - 0.5 * (zc[k - 1] + zc[k]));
}

/* out = L phi (exported so the tests can form manufactured right-hand sides). */
int oracle_laplacian(int nx, int ny, int nz, double Lx, double Ly, const double *zc,
                     int bc_x, int bc_y, const double *phi, double *out)
{
    const double rdx = 1.0 / (Lx / (double)nx), rdy = 1.0 / (Ly / (double)ny);
    double *rdzc = malloc(sizeof(double) * nz), *rdzm = malloc(sizeof(double) * nz);
    if (!rdzc || !rdzm) return 4;
    zmetric_double(nz, zc, rdzc, rdzm);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++)
                out[IDX(i, j, k)] = lap_at(nx, ny, nz, bc_x, bc_y, phi, rdx, rdy, rdzc, rdzm, i, j, k);
    free(rdzc); free(rdzm);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Step a7: velocity correction and pressure update (readings R4, R9). */
/*   u -= adt*((phi_i - phi_{i-1})*rdx)    (wall faces untouched)             */
/*   v -= adt*((phi_j - phi_{j-1})*rdy)                                       */
/*   w -= adt*((phi_k - phi_{k-1})*rdzm[k])   for k >= 1                      */
/*   p += phi                 if beta == 0                                    */
/*   p += phi - beta*(L phi)  otherwise, L phi from the stencil (not from rhs)*/
/* ------------------------------------------------------------------------- */
int oracle_project(int nx, int ny, int nz, double Lx, double Ly, const double *zc,
                   int bc_x, int bc_y, double *u, double *v, double *w, double *p,
                   const double *phi, double alpha_dt, double beta)
{
    const double rdx = 1.0 / (Lx / (double)nx), rdy = 1.0 / (Ly / (double)ny);
    double *rdzc = malloc(sizeof(double) * nz), *rdzm = malloc(sizeof(double) * nz);
    if (!rdzc || !rdzm) return 4;
    zmetric_double(nz, zc, rdzc, rdzm);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                double c0 = phi[IDX(i, j, k)];
                if (i > 0) u[IDX(i, j, k)] = u[IDX(i, j, k)] - alpha_dt * ((c0 - phi[IDX(i - 1, j, k)]) * rdx);
                else if (bc_x == ORACLE_BC_PERIODIC)
                    u[IDX(i, j, k)] = u[IDX(i, j, k)] - alpha_dt * ((c0 - phi[IDX(nx - 1, j, k)]) * rdx);
                if (j > 0) v[IDX(i, j, k)] = v[IDX(i, j, k)] - alpha_dt * ((c0 - phi[IDX(i, j - 1, k)]) * rdy);
                else if (bc_y == ORACLE_BC_PERIODIC)
                    v[IDX(i, j, k)] = v[IDX(i, j, k)] - alpha_dt * ((c0 - phi[IDX(i, ny - 1, k)]) * rdy);
                if (k > 0) w[IDX(i, j, k)] = w[IDX(i, j, k)] - alpha_dt * ((c0 - phi[IDX(i, j, k - 1)]) * rdzm[k]);
                if (beta == 0.0) p[IDX(i, j, k)] = p[IDX(i, j, k)] + c0;
                else {
                    double l = lap_at(nx, ny, nz, bc_x, bc_y, phi, rdx, rdy, rdzc, rdzm, i, j, k);
                    p[IDX(i, j, k)] = p[IDX(i, j, k)] + (c0 - beta * l);
                }
            }
    free(rdzc); free(rdzm);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Steps a2..a6: phi = solution of L phi = rhs with the gauge of R7.          */
/* Forward transform in x then y, one tridiagonal solve per (kx,ky), inverse  */
/* transform in y then x.  Full complex spectrum in   */
/* real_t; nothing is blocked or fused.                                       */
/* ------------------------------------------------------------------------- */
int oracle_poisson_solve(int nx, int ny, int nz, double Lx, double Ly, const double *zc,
                         int bc_x, int bc_y, const double *rhs, double *phi)
{
    if (nx < 1 || ny < 1 || nz < 2) return 1;
    size_t N = (size_t)nx * ny * nz;
    real_t *sr = malloc(sizeof(real_t) * N), *si = malloc(sizeof(real_t) * N);
    real_t *dzc = malloc(sizeof(real_t) * nz), *dzm = malloc(sizeof(real_t) * nz);
    real_t *za = malloc(sizeof(real_t) * nz), *zcc = malloc(sizeof(real_t) * nz);
    real_t *lamx = malloc(sizeof(real_t) * nx), *lamy = malloc(sizeof(real_t) * ny);
    if (!sr || !si || !dzc || !dzm || !za || !zcc || !lamx || !lamy) return 4;
    zcoef(nz, zc, dzc, dzm, za, zcc);
    modified_wavenumbers(nx, Lx, bc_x, lamx);
    modified_wavenumbers(ny, Ly, bc_y, lamy);

    dft_table tx, ty;       /* periodic: length n; Neumann: length 2n (even extension) */
    dft_table_init(&tx, bc_x == ORACLE_BC_PERIODIC ? nx : 2 * nx);
    dft_table_init(&ty, bc_y == ORACLE_BC_PERIODIC ? ny : 2 * ny);
    int nmax = nx > ny ? nx : ny; if (nz > nmax) nmax = nz;

#pragma omp parallel
    {
        real_t *lr = malloc(sizeof(real_t) * nmax), *li = malloc(sizeof(real_t) * nmax);
        real_t *or_ = malloc(sizeof(real_t) * nmax), *oi = malloc(sizeof(real_t) * nmax);
        real_t *wk = malloc(sizeof(real_t) * 8 * nmax);
        real_t *bd = malloc(sizeof(real_t) * nmax), *cp = malloc(sizeof(real_t) * nmax);

        /* a2: x-forward on every x-line */
#pragma omp for schedule(static)
        for (long row = 0; row < (long)ny * nz; row++) {
            size_t base = (size_t)row * nx;
            for (int i = 0; i < nx; i++) { lr[i] = (real_t)rhs[base + i]; li[i] = 0; }
            if (bc_x == ORACLE_BC_PERIODIC) dft_apply(&tx, -1, lr, li, or_, oi);
            else { dct2_apply(&tx, lr, or_, wk); for (int i = 0; i < nx; i++) oi[i] = 0; }
            for (int i = 0; i < nx; i++) { sr[base + i] = or_[i]; si[base + i] = oi[i]; }
        }
        /* a3: y-forward on every y-line */
#pragma omp for schedule(static)
        for (long col = 0; col < (long)nx * nz; col++) {
            int k = (int)(col / nx), i = (int)(col % nx);
            for (int j = 0; j < ny; j++) { lr[j] = sr[IDX(i, j, k)]; li[j] = si[IDX(i, j, k)]; }
            if (bc_y == ORACLE_BC_PERIODIC) dft_apply(&ty, -1, lr, li, or_, oi);
            else { dct2_apply(&ty, lr, or_, wk); dct2_apply(&ty, li, oi, wk); }
            for (int j = 0; j < ny; j++) { sr[IDX(i, j, k)] = or_[j]; si[IDX(i, j, k)] = oi[j]; }
        }
        /* a4: one tridiagonal system per wavenumber pair, Re and Im as two right-hand sides */
#pragma omp for schedule(static)
        for (long col = 0; col < (long)nx * ny; col++) {
            int j = (int)(col / nx), i = (int)(col % nx);
            for (int k = 0; k < nz; k++) { lr[k] = sr[IDX(i, j, k)]; li[k] = si[IDX(i, j, k)]; }
            if (i == 0 && j == 0) {                       /* lambda_x + lambda_y = 0: singular, gauge column */
                gauge_column(nz, dzc, dzm, lr, or_);
                gauge_column(nz, dzc, dzm, li, oi);
            } else {
                for (int k = 0; k < nz; k++) bd[k] = -(za[k] + zcc[k]) + lamx[i] + lamy[j];
                thomas(nz, za, bd, zcc, lr, or_, cp);
                thomas(nz, za, bd, zcc, li, oi, cp);
            }
            for (int k = 0; k < nz; k++) { sr[IDX(i, j, k)] = or_[k]; si[IDX(i, j, k)] = oi[k]; }
        }
        /* a5: y-inverse */
#pragma omp for schedule(static)
        for (long col = 0; col < (long)nx * nz; col++) {
            int k = (int)(col / nx), i = (int)(col % nx);
            for (int j = 0; j < ny; j++) { lr[j] = sr[IDX(i, j, k)]; li[j] = si[IDX(i, j, k)]; }
            if (bc_y == ORACLE_BC_PERIODIC) dft_apply(&ty, +1, lr, li, or_, oi);
            else { dct3_apply(&ty, lr, or_, wk); dct3_apply(&ty, li, oi, wk); }
            for (int j = 0; j < ny; j++) { sr[IDX(i, j, k)] = or_[j]; si[IDX(i, j, k)] = oi[j]; }
        }
        /* a6: x-inverse; phi is the real part */
#pragma omp for schedule(static)
        for (long row = 0; row < (long)ny * nz; row++) {
            size_t base = (size_t)row * nx;
            for (int i = 0; i < nx; i++) { lr[i] = sr[base + i]; li[i] = si[base + i]; }
            if (bc_x == ORACLE_BC_PERIODIC) dft_apply(&tx, +1, lr, li, or_, oi);
            else dct3_apply(&tx, lr, or_, wk);
            for (int i = 0; i < nx; i++) phi[base + i] = (double)or_[i];
        }
        free(lr); free(li); free(or_); free(oi); free(wk); free(bd); free(cp);
    }
    dft_table_free(&tx); dft_table_free(&ty);
    free(sr); free(si); free(dzc); free(dzm); free(za); free(zcc); free(lamx); free(lamy);
    return 0;
}

/* One whole projection: a1, a2..a6, a7.  phi is returned for inspection. */
int oracle_pressure_projection(int nx, int ny, int nz, double Lx, double Ly, const double *zc,
                               int bc_x, int bc_y, double *u, double *v, double *w, double *p,
                               double *phi, double alpha_dt, double beta)
{
    int rc = oracle_divergence(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, u, v, w, alpha_dt, phi);
    if (rc) return rc;
    rc = oracle_poisson_solve(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, phi, phi);
    if (rc) return rc;
    return oracle_project(nx, ny, nz, Lx, Ly, zc, bc_x, bc_y, u, v, w, p, phi, alpha_dt, beta);
}

/* ------------------------------------------------------------------------- */
/* Building blocks exported on double arrays so the tests can pin each one.   */
/* ------------------------------------------------------------------------- */
int oracle_dft(int n, int sign, const double *xr, const double *xi, double *yr, double *yi)
{
    if (n < 1) return 1;
    dft_table t; dft_table_init(&t, n);
    real_t *b = calloc((size_t)4 * n, sizeof(real_t));
    for (int j = 0; j < n; j++) { b[j] = xr[j]; b[n + j] = xi[j]; }
    dft_apply(&t, sign, b, b + n, b + 2 * n, b + 3 * n);
    for (int j = 0; j < n; j++) { yr[j] = (double)b[2 * n + j]; yi[j] = (double)b[3 * n + j]; }
    free(b); dft_table_free(&t);
    return 0;
}
int oracle_dct(int n, int inverse, const double *x, double *y)
{
    dft_table t; dft_table_init(&t, 2 * n);
    real_t *b = malloc(sizeof(real_t) * 10 * n);
    for (int j = 0; j < n; j++) b[j] = x[j];
    if (!inverse) dct2_apply(&t, b, b + n, b + 2 * n); else dct3_apply(&t, b, b + n, b + 2 * n);
    for (int j = 0; j < n; j++) y[j] = (double)b[n + j];
    free(b); dft_table_free(&t);
    return 0;
}
int oracle_thomas(int n, const double *a, const double *b, const double *c, const double *d, double *x)
{
    real_t *m = malloc(sizeof(real_t) * 6 * n);
    for (int k = 0; k < n; k++) { m[k] = a[k]; m[n + k] = b[k]; m[2 * n + k] = c[k]; m[3 * n + k] = d[k]; }
    thomas(n, m, m + n, m + 2 * n, m + 3 * n, m + 4 * n, m + 5 * n);
    for (int k = 0; k < n; k++) x[k] = (double)m[4 * n + k];
    free(m);
    return 0;
}
/* z-operator coefficients and the gauge column, as the solve uses them. */
int oracle_zcoef(int nz, const double *zc, double *dzc, double *dzm, double *a, double *c)
{
    real_t *m = malloc(sizeof(real_t) * 4 * nz);
    zcoef(nz, zc, m, m + nz, m + 2 * nz, m + 3 * nz);
    for (int k = 0; k < nz; k++) { dzc[k] = (double)m[k]; dzm[k] = (double)m[nz + k]; a[k] = (double)m[2 * nz + k]; c[k] = (double)m[3 * nz + k]; }
    free(m);
    return 0;
}
int oracle_gauge_column(int nz, const double *zc, const double *d, double *x)
{
    real_t *m = malloc(sizeof(real_t) * 6 * nz);
    zcoef(nz, zc, m, m + nz, m + 2 * nz, m + 3 * nz);
    for (int k = 0; k < nz; k++) m[4 * nz + k] = d[k];
    gauge_column(nz, m, m + nz, m + 4 * nz, m + 5 * nz);
    for (int k = 0; k < nz; k++) x[k] = (double)m[5 * nz + k];
    free(m);
    return 0;
}
int oracle_modified_wavenumbers(int n, double L, int bc, double *lam)
{
    real_t *m = malloc(sizeof(real_t) * n);
    modified_wavenumbers(n, L, bc, m);
    for (int k = 0; k < n; k++) lam[k] = (double)m[k];
    free(m);
    return 0;
}
