// ibm.cuh -- IB-MLS transfer operators (Eq. 4, Fig. 2):
//   u_c(x_b) = sum_{k=1..27} phi^k(x_b) u_c(x_k)        interpolation of each velocity component to a marker
//   F_c = (V_c - u_c(x_b)) / dt                          IB force at the marker
//   f_c(x_k) += c_l phi^k F_c                            distributed forcing on the Eulerian nodes
// with phi^k the moving-least-squares shape functions of a linear basis [1, x, y, z] and an exponential weight on the
// 3 x 3 x 3 support of the component's own staggered grid (readings M1..M8 of DESIGN.md sec. 3).
//
// The paper's CUDA Fortran subroutine gives 16 threads to the 4 x 4 system of a marker (V100/A100).  Here one
// thread owns one (marker, component): the 27 weights, the symmetric 4 x 4 moment matrix (10 sums), its Cholesky
// solve and the 27 shape functions all stay in registers, nothing is exchanged between threads, and neighbouring
// threads (the three components of a marker, then the next marker) touch neighbouring cache lines.  The gathers are
// L2 hits for any cloud that is denser than the grid; the scatter uses fp64 red.global.add (order-free sum).
#pragma once
#include "kernel_env.cuh"
#include "plan_types.cuh"

namespace fsei {

struct MlsGrid {
    int nx, ny, nz, bcx, bcy;
    double dx, dy, Lx, Ly;
    const double* zc;      // [nz + 1] z-face coordinates (device)
};

struct MlsStencil {
    size_t base[27];       // linear node indices
    double phi[27];
    double cl_den;         // sum_k phi^k dV_k
    double hl;             // local grid size (dx + dy + dz_kc)/3
};

FSEI_DEV double mls_znode(const MlsGrid& G, int comp, int k) { return comp == 2 ? G.zc[k] : 0.5 * (G.zc[k] + G.zc[k + 1]); }
FSEI_DEV double mls_zvol(const MlsGrid& G, int comp, int k)
{
    if (comp != 2) return G.zc[k + 1] - G.zc[k];
    return k == 0 ? 0.0 : 0.5 * (G.zc[k] + G.zc[k + 1]) - 0.5 * (G.zc[k - 1] + G.zc[k]);
}

// centre index along a uniform direction and the coordinate reduced to the period
FSEI_DEV int mls_nearest(double x, double h, double off, int n, bool periodic, double L, double& xred)
{
    if (periodic) x -= floor(x / L) * L;
    xred = x;
    int c = (int)floor(x / h - off + 0.5);
    if (periodic) { if (c < 0) c += n; if (c >= n) c -= n; }
    else { c = c < 1 ? 1 : (c > n - 2 ? n - 2 : c); }
    return c;
}

// centre node (ic, jc, kc) of the 3 x 3 x 3 support of one (marker, component); xr, yr: coordinates reduced to the period
FSEI_DEV void mls_centre(const MlsGrid& G, int comp, double xb, double yb, double zb, int& ic, int& jc, int& kc, double& xr, double& yr)
{
    ic = mls_nearest(xb, G.dx, comp == 0 ? 0.0 : 0.5, G.nx, G.bcx == BC_PERIODIC, G.Lx, xr);
    jc = mls_nearest(yb, G.dy, comp == 1 ? 0.0 : 0.5, G.ny, G.bcy == BC_PERIODIC, G.Ly, yr);
    // nearest z node: bisection for the last node <= zb, then the closer of it and the next (ties: the lower one)
    int lo = 0, hi = G.nz - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (mls_znode(G, comp, mid) <= zb) lo = mid; else hi = mid - 1; }
    kc = lo;
    if (kc + 1 < G.nz && fabs(mls_znode(G, comp, kc + 1) - zb) < fabs(mls_znode(G, comp, kc) - zb)) kc++;
    kc = kc < 1 ? 1 : (kc > G.nz - 2 ? G.nz - 2 : kc);
}

// the 27 shape functions of one (marker, component)
FSEI_DEV void mls_stencil(const MlsGrid& G, int comp, double xb, double yb, double zb, MlsStencil& M)
{
    double xr, yr;
    int ic, jc, kc;
    mls_centre(G, comp, xb, yb, zb, ic, jc, kc, xr, yr);
    const double zk[3] = {mls_znode(G, comp, kc - 1), mls_znode(G, comp, kc), mls_znode(G, comp, kc + 1)};
    const double rhz = 2.0 / (zk[2] - zk[0]);
    // per-direction scaled offsets of the three nodes and their node indices
    double xi[3], et[3], ze[3]; int ii[3], jj[3];
#pragma unroll
    for (int d = 0; d < 3; d++) {
        int i = ic + d - 1, j = jc + d - 1;
        double xk = ((double)i + (comp == 0 ? 0.0 : 0.5)) * G.dx, yk = ((double)j + (comp == 1 ? 0.0 : 0.5)) * G.dy;
        if (G.bcx == BC_PERIODIC) { if (xk - xr > 0.5 * G.Lx) xk -= G.Lx; if (xr - xk > 0.5 * G.Lx) xk += G.Lx; i = i < 0 ? i + G.nx : (i >= G.nx ? i - G.nx : i); }
        if (G.bcy == BC_PERIODIC) { if (yk - yr > 0.5 * G.Ly) yk -= G.Ly; if (yr - yk > 0.5 * G.Ly) yk += G.Ly; j = j < 0 ? j + G.ny : (j >= G.ny ? j - G.ny : j); }
        xi[d] = (xk - xr) / G.dx; et[d] = (yk - yr) / G.dy; ze[d] = (zk[d] - zb) * rhz;
        ii[d] = i; jj[d] = j;
    }
    // weights and the moment matrix A = sum W p p^T (symmetric, p = [1, xi, eta, zeta])
    // the weight exp(-(xi^2 + eta^2 + zeta^2) / (1.5 eps)^2) is a product of three one-dimensional factors: 9 exponentials per
    // (marker, component) instead of 27 (the product differs from the exponential of the sum by rounding only: ~2 ulp)
    const double inv = 1.0 / (1.5 * 1.5 * 0.3 * 0.3);
    double wx[3], wy[3], wz[3];
#pragma unroll
    for (int d = 0; d < 3; d++) { wx[d] = exp(-(xi[d] * xi[d]) * inv); wy[d] = exp(-(et[d] * et[d]) * inv); wz[d] = exp(-(ze[d] * ze[d]) * inv); }
    double a00 = 0, a01 = 0, a02 = 0, a03 = 0, a11 = 0, a12 = 0, a13 = 0, a22 = 0, a23 = 0, a33 = 0;
#pragma unroll
    for (int dk = 0; dk < 3; dk++)
#pragma unroll
        for (int dj = 0; dj < 3; dj++)
#pragma unroll
            for (int di = 0; di < 3; di++) {
                const int s = (dk * 3 + dj) * 3 + di;
                const double W = wx[di] * (wy[dj] * wz[dk]);
                M.phi[s] = W;
                a00 += W; a01 += W * xi[di]; a02 += W * et[dj]; a03 += W * ze[dk];
                a11 += W * xi[di] * xi[di]; a12 += W * xi[di] * et[dj]; a13 += W * xi[di] * ze[dk];
                a22 += W * et[dj] * et[dj]; a23 += W * et[dj] * ze[dk]; a33 += W * ze[dk] * ze[dk];
                M.base[s] = ((size_t)(kc + dk - 1) * G.ny + jj[dj]) * G.nx + ii[di];
            }
    // A lam = e_0 by Cholesky A = L L^T (A is symmetric positive definite: 27 nodes in general position)
    const double l00 = sqrt(a00), l10 = a01 / l00, l20 = a02 / l00, l30 = a03 / l00;
    const double l11 = sqrt(a11 - l10 * l10), l21 = (a12 - l20 * l10) / l11, l31 = (a13 - l30 * l10) / l11;
    const double l22 = sqrt(a22 - l20 * l20 - l21 * l21), l32 = (a23 - l30 * l20 - l31 * l21) / l22;
    const double l33 = sqrt(a33 - l30 * l30 - l31 * l31 - l32 * l32);
    const double y0 = 1.0 / l00, y1 = -l10 * y0 / l11, y2 = -(l20 * y0 + l21 * y1) / l22, y3 = -(l30 * y0 + l31 * y1 + l32 * y2) / l33;
    const double m3 = y3 / l33, m2 = (y2 - l32 * m3) / l22, m1 = (y1 - l21 * m2 - l31 * m3) / l11, m0 = (y0 - l10 * m1 - l20 * m2 - l30 * m3) / l00;
    double den = 0.0;
    const double dxdy = G.dx * G.dy;
#pragma unroll
    for (int dk = 0; dk < 3; dk++) {
        const double vol = dxdy * mls_zvol(G, comp, kc + dk - 1);
#pragma unroll
        for (int dj = 0; dj < 3; dj++)
#pragma unroll
            for (int di = 0; di < 3; di++) {
                const int s = (dk * 3 + dj) * 3 + di;
                const double ph = M.phi[s] * (m0 + m1 * xi[di] + m2 * et[dj] + m3 * ze[dk]);
                M.phi[s] = ph;
                den += ph * vol;
            }
    }
    M.cl_den = den;
    M.hl = (G.dx + G.dy + mls_zvol(G, comp, kc)) / 3.0;
}

struct MlsArgs {
    MlsGrid G;
    long n;
    const double *xm, *ym, *zm, *area;      // markers (device); area may be null for interpolation
    const double* q[3];                     // u, v, w (interpolation input)
    const double* V[3];                     // body velocity at the markers (forcing)
    double* Fb[3];                          // marker values: interpolated velocity (MODE 0) or force (MODE 1 out, MODE 2 in)
    double* f[3];                           // Eulerian forcing fields (accumulated)
    double inv_dt;
};

// MODE 0: interpolate (Fb = U);  1: forcing (Fb = (V - U) inv_dt, f += spread);  2: spread (f += spread of Fb)
// one thread per (marker, component): t = 3 l + c
template <int MODE>
FSEI_GLOBAL(128, 1) k_mls(const FSEI_GRID_CONSTANT MlsArgs A)
{
    const long t = (long)blockIdx.x * 128 + threadIdx.x;
    if (t >= 3 * A.n) return;
    const long l = t / 3; const int c = (int)(t - 3 * l);
    MlsStencil M;
    mls_stencil(A.G, c, A.xm[l], A.ym[l], A.zm[l], M);
    double F;
    if (MODE != 2) {
        const double* __restrict__ q = A.q[c];
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < 27; k++) s += M.phi[k] * q[M.base[k]];
        if (MODE == 0) { A.Fb[c][l] = s; return; }
        F = (A.V[c][l] - s) * A.inv_dt;
        A.Fb[c][l] = F;
    } else F = A.Fb[c][l];
    const double cl = A.area[l] * M.hl / M.cl_den * F;
    double* __restrict__ f = A.f[c];
#pragma unroll
    for (int k = 0; k < 27; k++) atomicAdd(f + M.base[k], cl * M.phi[k]);
}

// The forcing fields are zero except on the supports of the markers, so the substep need not stream them: after the explicit
// terms (evaluated without a body force) this kernel visits the support nodes again and forms rhs += alpha_dt f there -- the
// same two operations, in the same order, as the dense path of k_explicit_terms.  A node shared by several supports is taken
// by whichever thread swaps its accumulated sum out of f first (the others read back 0 and leave); f is all-zero again
// afterwards.  Wall-face rows (u at i = 0 / v at j = 0 on a wall-bounded box, w at k = 0) keep rhs = 0 (V7).
struct MlsApplyArgs {
    MlsGrid G;
    long n;
    const double *xm, *ym, *zm;
    double* f[3];
    double* r[3];
    double adt;
};

FSEI_GLOBAL(128, 1) k_mls_apply(const FSEI_GRID_CONSTANT MlsApplyArgs A)
{
    const long t = (long)blockIdx.x * 128 + threadIdx.x;
    if (t >= 3 * A.n) return;
    const long l = t / 3; const int c = (int)(t - 3 * l);
    const MlsGrid& G = A.G;
    double xr, yr;
    int ic, jc, kc;
    mls_centre(G, c, A.xm[l], A.ym[l], A.zm[l], ic, jc, kc, xr, yr);
    double* __restrict__ f = A.f[c];
    double* __restrict__ r = A.r[c];
#pragma unroll
    for (int dk = -1; dk <= 1; dk++)
#pragma unroll
        for (int dj = -1; dj <= 1; dj++)
#pragma unroll
            for (int di = -1; di <= 1; di++) {
                int i = ic + di, j = jc + dj;
                const int k = kc + dk;
                if (G.bcx == BC_PERIODIC) i = i < 0 ? i + G.nx : (i >= G.nx ? i - G.nx : i);
                if (G.bcy == BC_PERIODIC) j = j < 0 ? j + G.ny : (j >= G.ny ? j - G.ny : j);
                const size_t b = ((size_t)k * G.ny + j) * G.nx + i;
                const double val = __longlong_as_double((long long)atomicExch(reinterpret_cast<unsigned long long*>(f + b), 0ull));
                const bool wall_row = (c == 0 && i == 0 && G.bcx != BC_PERIODIC) || (c == 1 && j == 0 && G.bcy != BC_PERIODIC) || (c == 2 && k == 0);
                if (val != 0.0 && !wall_row) r[b] = __dadd_rn(r[b], __dmul_rn(A.adt, val));
            }
}

}  // namespace fsei
