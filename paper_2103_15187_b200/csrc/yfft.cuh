// yfft.cuh -- per-thread phases of the y-direction transforms on a shared-memory tile
// [ny rows][C columns] of complex values (column = one x-slot, c fastest: the tile is a
// straight copy of C adjacent slots of every row of one z-plane).  Steps a3 / a5.
#pragma once
#include "plan_types.cuh"

namespace fsei {

template <bool NEUMANN> struct YAddr {
    int c, C, N;
    FSEI_HD int operator()(int n) const { return (NEUMANN ? dct_perm(n, N) : n) * C + c; }
};

template <int R, bool INV, bool NEUMANN>
FSEI_HD void y_pass(const YParams& P, cplx* sm, int C, int Ns, int tid, int nt)
{
    const int M = Ns / R, per = P.N / R, tmul = P.N / Ns;
    for (int w = tid; w < C * per; w += nt) {
        int b = w / C, c = w - b * C;
        int blk = b / M, n2 = b - blk * M;
        YAddr<NEUMANN> A; A.c = c; A.C = C; A.N = P.N;
        fft_butterfly<R, INV>(sm, A, blk, n2, Ns, M, tmul, P.tw);
    }
}

template <bool INV, bool NEUMANN>
FSEI_HD void y_pass_dispatch(const YParams& P, cplx* sm, int C, int R, int Ns, int tid, int nt)
{
    switch (R) {
        case 16: y_pass<16, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
        case 8:  y_pass<8, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
        case 5:  y_pass<5, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
        case 4:  y_pass<4, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
        case 3:  y_pass<3, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
        default: y_pass<2, INV, NEUMANN>(P, sm, C, Ns, tid, nt); break;
    }
}

// Neumann only.  After the forward passes V = FFT(reordered column) sits at physical row
// perm(pos[k]); the column is two packed real sequences a + i b.  Pair k with N-k:
//   Va = (Vk + conj Vm)/2, Vb = (Vk - conj Vm)/(2i), ta = w_k Va, tb = w_k Vb
//   row(k) <- (Re ta, Re tb),  row(N-k) <- (-Im ta, -Im tb)
FSEI_HD void y_post_forward_dct(const YParams& P, cplx* sm, int C, int tid, int nt)
{
    const int N = P.N, half = N >> 1;
    for (int w = tid; w < C * half; w += nt) {
        int kk = w / C, c = w - kk * C;
        int k = kk + 1;                                   // k = 1 .. N/2 ; k = 0 needs nothing (X_0 = V_0)
        int r1 = dct_perm(P.pos[k], N) * C + c, r2 = dct_perm(P.pos[N - k], N) * C + c;
        cplx vk = sm[r1], vm = sm[r2];
        cplx wk = P.tw_dct[k];
        cplx Va = cmake(0.5 * (vk.re + vm.re), 0.5 * (vk.im - vm.im));
        cplx D = cmake(vk.re - vm.re, vk.im + vm.im);
        cplx Vb = cmake(0.5 * D.im, -0.5 * D.re);
        cplx ta = cmul(Va, wk), tb = cmul(Vb, wk);
        sm[r1] = cmake(ta.re, tb.re);
        if (k != N - k) sm[r2] = cmake(-ta.im, -tb.im);
    }
}
FSEI_HD void y_pre_inverse_dct(const YParams& P, cplx* sm, int C, int tid, int nt)
{
    const int N = P.N, half = N >> 1;
    for (int w = tid; w < C * half; w += nt) {
        int kk = w / C, c = w - kk * C;
        int k = kk + 1;
        int r1 = dct_perm(P.pos[k], N) * C + c, r2 = dct_perm(P.pos[N - k], N) * C + c;
        cplx xk = sm[r1], xm = sm[r2];
        cplx wk = P.tw_dct[k];
        if (k == N - k) {                                 // X = cos(pi/4) V for both parts, V real
            sm[r1] = cmake(xk.re * 1.41421356237309504880168872420969808, xk.im * 1.41421356237309504880168872420969808);
        } else {
            cplx ta = cmulc(cmake(xk.re, -xm.re), wk);    // V^a_k
            cplx tb = cmulc(cmake(xk.im, -xm.im), wk);    // V^b_k
            sm[r1] = cmake(ta.re - tb.im, ta.im + tb.re);             // ta + i tb
            sm[r2] = cmake(ta.re + tb.im, -ta.im + tb.re);            // conj(ta) + i conj(tb)
        }
    }
}

// global <-> tile: g points at element (row 0, first slot of the tile) of the plane; rows are
// `gpitch` complex apart.
FSEI_HD void y_load(cplx* sm, const cplx* g, size_t gpitch, int N, int C, int tid, int nt)
{
    for (int w = tid; w < N * C; w += nt) {
        int r = w / C, c = w - r * C;
        sm[w] = g[(size_t)r * gpitch + c];
    }
}
FSEI_HD void y_store(const cplx* sm, cplx* g, size_t gpitch, int N, int C, int tid, int nt)
{
    for (int w = tid; w < N * C; w += nt) {
        int r = w / C, c = w - r * C;
        g[(size_t)r * gpitch + c] = sm[w];
    }
}

}  // namespace fsei
