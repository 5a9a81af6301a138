// xfft.cuh -- per-thread phases of the x-direction transforms on a shared-memory tile of
// `lines` lines (each N = nx/2 complex values at pitch P.pitch, index n stored at padx(n)).
// Steps a2 / a6 of the path (include/fsei.h; R15).
#pragma once
#include "plan_types.cuh"

namespace fsei {

struct XAddr {
    int base;
    FSEI_HD int operator()(int n) const { return base + padx(n); }
};

// (a, b) = (x[2t], x[2t+1]) of one real line -> the complex work sequence in shared memory
FSEI_HD void x_put_pair(const XParams& P, cplx* line, int t, double a, double b)
{
    if (P.bc == BC_PERIODIC) {
        line[padx(t)] = cmake(a, b);
    } else {                                   // Makhoul reorder: v[t] = x[2t], v[n-1-t] = x[2t+1]; z_m = v[2m] + i v[2m+1]
        int q0 = t, q1 = P.n - 1 - t;
        reinterpret_cast<double*>(&line[padx(q0 >> 1)])[q0 & 1] = a;
        reinterpret_cast<double*>(&line[padx(q1 >> 1)])[q1 & 1] = b;
    }
}
FSEI_HD void x_get_pair(const XParams& P, const cplx* line, int t, double& a, double& b)
{
    if (P.bc == BC_PERIODIC) {
        cplx z = line[padx(t)]; a = z.re; b = z.im;
    } else {
        int q0 = t, q1 = P.n - 1 - t;
        a = reinterpret_cast<const double*>(&line[padx(q0 >> 1)])[q0 & 1];
        b = reinterpret_cast<const double*>(&line[padx(q1 >> 1)])[q1 & 1];
    }
}

// one pass over the tile
template <int R, bool INV>
FSEI_HD void x_pass(const XParams& P, cplx* sm, int lines, int Ns, int tid, int nt)
{
    const int M = Ns / R, per = P.N / R, tmul = P.N / Ns;
    for (int w = tid; w < lines * per; w += nt) {
        int line = w / per, b = w - line * per;
        int blk = b / M, n2 = b - blk * M;
        XAddr A; A.base = line * P.pitch;
        fft_butterfly<R, INV>(sm, A, blk, n2, Ns, M, tmul, P.tw);
    }
}

template <bool INV>
FSEI_HD void x_pass_dispatch(const XParams& P, cplx* sm, int lines, int R, int Ns, int tid, int nt)
{
    switch (R) {
        case 16: x_pass<16, INV>(P, sm, lines, Ns, tid, nt); break;
        case 8:  x_pass<8, INV>(P, sm, lines, Ns, tid, nt); break;
        case 5:  x_pass<5, INV>(P, sm, lines, Ns, tid, nt); break;
        case 4:  x_pass<4, INV>(P, sm, lines, Ns, tid, nt); break;
        case 3:  x_pass<3, INV>(P, sm, lines, Ns, tid, nt); break;
        default: x_pass<2, INV>(P, sm, lines, Ns, tid, nt); break;
    }
}

// quarter-wave twiddle of the DCT: V_k -> (X_k, X_{n-k}) = (Re(w_k V_k), -Im(w_k V_k)) and back
FSEI_HD cplx dct_tw_fwd(cplx V, cplx w) { cplx t = cmul(V, w); return cmake(t.re, -t.im); }
FSEI_HD cplx dct_tw_inv(cplx S, cplx w) { return cmulc(cmake(S.re, -S.im), w); }

// after the forward passes: Z (FFT of the packed sequence) -> half spectrum of the real line
FSEI_HD void x_post_forward(const XParams& P, cplx* sm, int lines, int tid, int nt)
{
    const int N = P.N, half = N >> 1, per = half + 1;
    for (int w = tid; w < lines * per; w += nt) {
        int line = w / per, k = w - line * per;
        cplx* L = sm + line * P.pitch;
        if (k == 0) {
            cplx z = L[0];
            double x0 = z.re + z.im, xn = z.re - z.im;
            if (P.bc == BC_NEUMANN) xn *= FSEI_SQRT1_2;                    // X_{n/2} = V_{n/2} cos(pi/4)
            L[0] = cmake(x0, xn);
        } else {
            int p1 = padx(P.pos[k]), p2 = padx(P.pos[N - k]);
            cplx zk = L[p1], zm = L[p2];
            cplx E = cmake(0.5 * (zk.re + zm.re), 0.5 * (zk.im - zm.im));   // (Zk + conj Zm)/2
            cplx D = cmake(zk.re - zm.re, zk.im + zm.im);                   // Zk - conj Zm
            cplx O = cmake(0.5 * D.im, -0.5 * D.re);                        // D / (2i)
            cplx T = cmul(O, P.tw_r2c[k]);
            cplx xk = cadd(E, T), xm = cconj(csub(E, T));
            if (P.bc == BC_NEUMANN) { xk = dct_tw_fwd(xk, P.tw_dct[k]); xm = dct_tw_fwd(xm, P.tw_dct[N - k]); }
            L[p1] = xk;
            if (k != N - k) L[p2] = xm;
        }
    }
}

// before the inverse passes: half spectrum -> Z
FSEI_HD void x_pre_inverse(const XParams& P, cplx* sm, int lines, int tid, int nt)
{
    const int N = P.N, half = N >> 1, per = half + 1;
    for (int w = tid; w < lines * per; w += nt) {
        int line = w / per, k = w - line * per;
        cplx* L = sm + line * P.pitch;
        if (k == 0) {
            cplx s = L[0];
            double x0 = s.re, xn = s.im;
            if (P.bc == BC_NEUMANN) xn *= 1.41421356237309504880168872420969808;
            L[0] = cmake(0.5 * (x0 + xn), 0.5 * (x0 - xn));
        } else {
            int p1 = padx(P.pos[k]), p2 = padx(P.pos[N - k]);
            cplx xk = L[p1], xm = L[p2];
            if (P.bc == BC_NEUMANN) { xk = dct_tw_inv(xk, P.tw_dct[k]); xm = dct_tw_inv(xm, P.tw_dct[N - k]); }
            cplx E = cmake(0.5 * (xk.re + xm.re), 0.5 * (xk.im - xm.im));   // (Xk + conj Xm)/2
            cplx T = cmake(0.5 * (xk.re - xm.re), 0.5 * (xk.im + xm.im));   // (Xk - conj Xm)/2
            cplx O = cmulc(T, P.tw_r2c[k]);
            cplx zk = cmake(E.re - O.im, E.im + O.re);                       // E + i O
            cplx zm = cmake(E.re + O.im, -(E.im - O.re));                    // conj(E - i O)
            L[p1] = zk;
            if (k != N - k) L[p2] = zm;
        }
    }
}

// global <-> tile.  g points at the first real (resp. complex) element of the tile's first line.
FSEI_HD void x_load_real(const XParams& P, cplx* sm, const double* g, int lines, int tid, int nt)
{
    for (int w = tid; w < lines * P.N; w += nt) {
        int line = w / P.N, t = w - line * P.N;
        const double* s = g + (size_t)line * P.n + 2 * t;
        x_put_pair(P, sm + line * P.pitch, t, s[0], s[1]);
    }
}
FSEI_HD void x_store_real(const XParams& P, const cplx* sm, double* g, int lines, int tid, int nt)
{
    for (int w = tid; w < lines * P.N; w += nt) {
        int line = w / P.N, t = w - line * P.N;
        double a, b;
        x_get_pair(P, sm + line * P.pitch, t, a, b);
        double* d = g + (size_t)line * P.n + 2 * t;
        d[0] = a * P.scale; d[1] = b * P.scale;
    }
}
FSEI_HD void x_load_spec(const XParams& P, cplx* sm, const cplx* g, int lines, int tid, int nt)
{
    for (int w = tid; w < lines * P.N; w += nt) {
        int line = w / P.N, t = w - line * P.N;
        sm[line * P.pitch + padx(t)] = g[(size_t)line * P.N + t];
    }
}
FSEI_HD void x_store_spec(const XParams& P, const cplx* sm, cplx* g, int lines, int tid, int nt)
{
    for (int w = tid; w < lines * P.N; w += nt) {
        int line = w / P.N, t = w - line * P.N;
        g[(size_t)line * P.N + t] = sm[line * P.pitch + padx(t)];
    }
}

}  // namespace fsei
