// yzfused.cuh -- steps a3+a4 (first half) and a4 (second half)+a5 as TWO z-marching kernels on the blocked
// spectrum layout (xfast.cuh: [nxc / CB][nz][ny][CB]); include/fsei.h, P:L208 (Thomas); DESIGN.md sec. 6.
//
// Thomas' algorithm along z is a forward elimination that needs plane k-1 only and a back substitution that
// needs plane k+1 only.  So the elimination rides on the y-forward transform and the substitution on the
// y-inverse transform, if those kernels march along z:
//
//   k_yz_forward : a CTA owns one x-slot tile (CB slots x all ny rows) and visits k = 0 .. nz-1.  Per plane: the
//                  tile (contiguous in the blocked layout) arrives by cp.async.bulk while the previous plane is
//                  transformed; register-resident Stockham FFT (or DCT-II) along y; then
//                  d'_k = (d_k - a_k d'_{k-1}) / piv_k with d'_{k-1} carried in registers, either on the last pass'
//                  outputs (single-spectrum tiles) or in one pass over the row pairs (kk, ny-kk) that also splits
//                  the two Hermitian y-spectra of a column that carries two real x-sequences; d'_k is stored.
//   k_yz_backward: same tiles, k = nz-1 .. 0: x_k = d'_k - (c_k / piv_k) x_{k+1} (x_{k+1} in registers), the
//                  special columns are replaced by their separately solved values, merge + inverse transform,
//                  store.
// The spectrum therefore makes two round trips through HBM for a3+a4+a5 instead of four (y, two Thomas sweeps, y).
// The arithmetic per element is exactly that of yfast.cuh / zfast.cuh (same operations in the same order).
#pragma once
#include "yfast.cuh"

namespace fsei {

struct YZFused {
    int nxc, ny, nz;
    int untangle;               // periodic y: columns [0, untangle) are split / merged (0, 1 or nxc)
    int pp;                     // bc = (P,P): special columns (row 0, slot 0) AND (row ny/2, slot 0), both parts;
                                // otherwise only the Re part of (row 0, slot 0)
    const cplx* tw;             // e^{-2 pi i j / ny}
    const cplx* tw_dct;         // e^{-i pi k / (2 ny)}   (Neumann y only)
    const double* za;           // a_k
    const double* zcc;          // c_k
    const double* ip;           // reciprocal pivots, blocked [nxc / CB][nz][ny][CB][NCOMP]
    cplx* special_in;           // [2][nz] right-hand sides of the special columns (written by k_yz_forward)
    const cplx* special;        // [2][nz] their solutions (k_z_special)
    int ktw;                    // twist plane (zfast.cuh): nz = plain Thomas, one CTA per tile (grid.y = 1); < nz = twisted
                                // factorisation, planes [0, ktw) and [ktw, nz) swept towards each other by two CTAs
                                // per tile (grid.y = 2) -- for grids with fewer tiles than SMs
    cplx* mid;                  // twisted only: [ntiles][2][ny CB] copies of d'_{ktw-1} and e'_{ktw}, the two planes both
                                // back-substitution CTAs of a tile start from (each overwrites one of them in place)
    int tile_shift[2];          // tile = (blockIdx.x + tile_shift[blockIdx.y]) % ntiles: puts the one tile that carries
                                // the split / merge work (tile 0 on (P,P)) on a CTA that is likely alone on its SM
};

template <class C, int CB, bool NEU, int NCOMP> struct YZSmem {
    static constexpr int TILE = C::N * CB;                      // complex per plane tile
    static constexpr int IPT = C::N * CB * NCOMP;               // doubles per pivot tile
    static constexpr int BUF = C::PITCH * CB;
    static constexpr int DCT = NEU ? C::N / 2 + 1 : 0;
    static constexpr size_t COMMON = 128 + sizeof(cplx) * (TILE + BUF + C::TW + DCT);
    static constexpr size_t FWD = COMMON;                                  // pivots read from global memory (L2-prefetched)
    static constexpr size_t BWD = COMMON + sizeof(double) * IPT;          // pivots land beside the tile
};

// grid nxc / CB, block T*CB, dynamic shared memory YZSmem::FWD.  spec: blocked spectrum after the x-forward step.
template <class C, int CB, bool NEU, int NCOMP>
FSEI_GLOBAL(C::T * CB, 1) k_yz_forward(YZFused P, cplx* spec)
{
    using L = YZSmem<C, CB, NEU, NCOMP>;
    constexpr int N = C::N, T = C::T, R0 = C::R0, NT = T * CB;
    constexpr int NB0 = N / R0, PER0 = PassShape<N, R0, 1, T>::PER;
    static_assert(NB0 % T == 0, "first pass must tile the column exactly");
    FSEI_DYN_SMEM(smraw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    cplx* land = reinterpret_cast<cplx*>(smraw + 128);           // [N][CB] dense
    cplx* buf = land + L::TILE;
    cplx* tws = buf + L::BUF;
    cplx* tdct = tws + C::TW;
    const int tid = threadIdx.x;
    const int tl = tid / CB, c = tid - tl * CB;
    const int tile = (int)((blockIdx.x + (blockIdx.y ? P.tile_shift[1] : P.tile_shift[0])) % gridDim.x), c0 = tile * CB, col = c0 + c;
    const int nz = P.nz;
    // this CTA's sweep: planes [0, ktw) upwards with the coupling a_k to the plane below (blockIdx.y = 0), or planes
    // [ktw, nz) downwards with the coupling c_k to the plane above (blockIdx.y = 1, twisted factorisation only)
    const bool up = blockIdx.y == 0;
    const int kfirst = up ? 0 : nz - 1, kstep = up ? 1 : -1, kcount = up ? P.ktw : nz - P.ktw;
    const double* coef = up ? P.za : P.zcc;
    const bool pairing = NEU || (c0 < P.untangle);             // CTA-uniform
    const bool mine = NEU || (col < P.untangle);
    cplx* tile0 = spec + (size_t)tile * nz * L::TILE;            // plane k of this tile at tile0 + k TILE
    const double* ip0 = P.ip + (size_t)tile * nz * L::IPT;

    // plane k: the tile lands in shared memory; the tile of plane k+1 and the pivots of plane k are pulled into L2
    // (the bulk load one plane later and the pivot loads at the end of this plane then complete at L2 latency)
    auto issue = [&](int k, bool more) {
        abar_expect(bar, (unsigned)(L::TILE * sizeof(cplx)));
        bulk_g2s(land, tile0 + (size_t)k * L::TILE, (unsigned)(L::TILE * sizeof(cplx)), bar);
        if (more) bulk_prefetch_l2(tile0 + (size_t)(k + kstep) * L::TILE, (unsigned)(L::TILE * sizeof(cplx)));
        bulk_prefetch_l2(ip0 + (size_t)k * L::IPT, (unsigned)(L::IPT * sizeof(double)));
    };
    if (tid == 0) abar_init(bar);
    fft_fill_twiddles<C>(tws, P.tw, tid, NT);
    if (NEU) for (int i = tid; i < L::DCT; i += NT) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();
    if (tid == 0 && kcount > 0) issue(kfirst, kcount > 1);
    unsigned parity = 0;

    constexpr int RL = (C::NP == 3) ? C::R2 : C::R1, NSL = N / RL;   // last pass: output slot i RL + q = row tl + i T + q NSL
    constexpr int NSLOT = PassShape<N, RL, NSL, T>::PER * RL;
    constexpr int ITP = N / (2 * T) + 1;                             // two-spectra tiles: row pairs (kk, N-kk), kk = tl + i T
    constexpr int NCARRY = (NSLOT > 2 * ITP) ? NSLOT : 2 * ITP;
    cplx carry[NCARRY];                                          // d'_{k-1} of this thread's elements
#pragma unroll
    for (int m = 0; m < NCARRY; m++) carry[m] = cmake(0.0, 0.0);
    double a_k = kcount > 0 ? coef[kfirst] : 0.0;

    for (int it = 0; it < kcount; it++) {
        const int k = kfirst + it * kstep;
        const bool more = it + 1 < kcount;
        abar_wait(bar, parity); parity ^= 1;
        auto next = [&]() { if (tid == 0 && more) issue(k + kstep, it + 2 < kcount); };
        auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
            for (int i = 0; i < PER0; i++) {
#pragma unroll
                for (int q = 0; q < R0; q++) {
                    const int n = tl + i * T + q * NB0;
                    v0[i][q] = land[(NEU ? dct_perm(n, N) : n) * CB + c];
                }
            }
        };
        // last plane of a twisted sweep: also kept aside for the back substitution's start
        cplx* gm = (P.ktw < nz && !more) ? P.mid + ((size_t)tile * 2 + (up ? 0 : 1)) * L::TILE : nullptr;
        if (!pairing) {
            // Columns with a single spectrum: the elimination runs on the last pass' outputs while they are still in
            // registers (output slot s of this thread is row RB(s) every plane, so d'_{k-1} is carried per slot).
            const double a = a_k;
            a_k = more ? coef[k + kstep] : 0.0;
            const double* ipk = ip0 + (size_t)k * L::IPT;
            cplx* gk = tile0 + (size_t)k * L::TILE;
            double ipv[NSLOT][NCOMP];
            auto pivots = [&]() {
#pragma unroll
                for (int s = 0; s < NSLOT; s++) {
                    const int b = tl + (s / RL) * T, n = b + (s % RL) * NSL;
                    if (b < NSL) {
#pragma unroll
                        for (int q = 0; q < NCOMP; q++) ipv[s][q] = ld_stream(ipk + (size_t)(n * CB + c) * NCOMP + q);
                    }
                }
            };
            auto elim = [&](int n, cplx d, int s) {
                carry[s] = cmake((d.re - a * carry[s].re) * ipv[s][0], (d.im - a * carry[s].im) * ipv[s][NCOMP - 1]);
                gk[n * CB + c] = carry[s];
                if (gm) gm[n * CB + c] = carry[s];
            };
            fft_column<C, CB, false, false, false>(tl, c, true, buf, tws, load0, elim, next, pivots);
            FSEI_SYNC();
            continue;
        }
        // Tiles whose columns carry two spectra: transform into the staging buffer, then ONE pass per thread over its row
        // pairs (kk, N-kk): split (+ quarter-wave twiddle), elimination with d'_{k-1} carried per pair slot, stores.
        fft_column<C, CB, false, false, true>(tl, c, true, buf, tws, load0, YOut<C, CB>{buf, c}, next);
        double ipv[2 * ITP][NCOMP];                              // reciprocal pivots (L2 hits), in flight across the barrier
        {
            const double* ipk = ip0 + (size_t)k * L::IPT;
#pragma unroll
            for (int i2 = 0; i2 < ITP; i2++) {
                const int kk = tl + i2 * T;
                if (kk <= N / 2) {
#pragma unroll
                    for (int q = 0; q < NCOMP; q++) {
                        ipv[2 * i2][q] = ld_stream(ipk + (size_t)(kk * CB + c) * NCOMP + q);
                        ipv[2 * i2 + 1][q] = ld_stream(ipk + (size_t)((kk ? N - kk : 0) * CB + c) * NCOMP + q);
                    }
                }
            }
        }
        FSEI_SYNC();
        {
            const double a = a_k;
            a_k = more ? coef[k + kstep] : 0.0;             // next plane's coefficient: latency hidden by this plane
            cplx* gk = tile0 + (size_t)k * L::TILE;
            cplx r1[ITP], r2[ITP];                               // rows kk and N-kk after the split
#pragma unroll
            for (int i2 = 0; i2 < ITP; i2++) {
                const int kk = tl + i2 * T;
                if (kk > N / 2) continue;
                const cplx p1 = buf[C::pad(kk) * CB + c], p2 = buf[C::pad(kk ? N - kk : 0) * CB + c];
                if (kk == 0 || (!NEU && (2 * kk == N || !mine))) { r1[i2] = p1; r2[i2] = p2; continue; }
                cplx A = cmake(0.5 * (p1.re + p2.re), 0.5 * (p1.im - p2.im));       // (P1 + conj P2)/2
                cplx D = cmake(p1.re - p2.re, p1.im + p2.im);
                cplx B = cmake(0.5 * D.im, -0.5 * D.re);                            // (P1 - conj P2)/(2i)
                if (NEU) {
                    const cplx wk = tdct[kk];
                    const cplx ta = cmul(A, wk), tb = cmul(B, wk);
                    r1[i2] = cmake(ta.re, tb.re); r2[i2] = cmake(-ta.im, -tb.im);
                } else { r1[i2] = A; r2[i2] = B; }
            }
#pragma unroll
            for (int i2 = 0; i2 < ITP; i2++) {
                const int kk = tl + i2 * T;
                if (kk > N / 2) continue;
                const bool two = kk != 0 && 2 * kk != N;        // row N-kk is a different row
                if (tile == 0 && c == 0) {                      // right-hand sides of the special columns
                    if (kk == 0) P.special_in[k] = r1[i2];
                    else if (P.pp && 2 * kk == N) P.special_in[nz + k] = r1[i2];
                }
                cplx& c1 = carry[2 * i2];
                c1 = cmake((r1[i2].re - a * c1.re) * ipv[2 * i2][0], (r1[i2].im - a * c1.im) * ipv[2 * i2][NCOMP - 1]);
                gk[kk * CB + c] = c1;
                if (gm) gm[kk * CB + c] = c1;
                if (two) {
                    cplx& c2 = carry[2 * i2 + 1];
                    c2 = cmake((r2[i2].re - a * c2.re) * ipv[2 * i2 + 1][0], (r2[i2].im - a * c2.im) * ipv[2 * i2 + 1][NCOMP - 1]);
                    gk[(N - kk) * CB + c] = c2;
                    if (gm) gm[(N - kk) * CB + c] = c2;
                }
            }
        }
        FSEI_SYNC();
    }
}

// grid nxc / CB, block T*CB, dynamic shared memory YZSmem::BWD.  spec: d' from k_yz_forward; P.special solved.
template <class C, int CB, bool NEU, int NCOMP>
FSEI_GLOBAL(C::T * CB, 1) k_yz_backward(YZFused P, cplx* spec)
{
    using L = YZSmem<C, CB, NEU, NCOMP>;
    constexpr int N = C::N, T = C::T, R0 = C::R0, NT = T * CB;
    constexpr int EPT = (N * CB) / NT;
    FSEI_DYN_SMEM(smraw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    cplx* land = reinterpret_cast<cplx*>(smraw + 128);
    cplx* buf = land + L::TILE;
    cplx* tws = buf + L::BUF;
    cplx* tdct = tws + C::TW;
    double* ipb = reinterpret_cast<double*>(tdct + L::DCT);      // [IPT]
    const int tid = threadIdx.x;
    const int tl = tid / CB, c = tid - tl * CB;
    const int tile = (int)((blockIdx.x + (blockIdx.y ? P.tile_shift[1] : P.tile_shift[0])) % gridDim.x), c0 = tile * CB, col = c0 + c;
    const int nz = P.nz;
    // this CTA's sweep: planes [0, ktw) downwards from ktw-1 (blockIdx.y = 0; the whole column when ktw = nz), or planes
    // [ktw, nz) upwards from ktw (blockIdx.y = 1, twisted factorisation only)
    const bool down = blockIdx.y == 0;
    const int kfirst = down ? P.ktw - 1 : P.ktw, kstep = down ? -1 : 1, kcount = down ? P.ktw : nz - P.ktw;
    const double* coef = down ? P.zcc : P.za;
    const bool pairing = NEU || (c0 < P.untangle);
    const bool mine = NEU || (col < P.untangle);
    const double SQ2 = 1.41421356237309504880168872420969808;
    cplx* tile0 = spec + (size_t)tile * nz * L::TILE;
    const double* ip0 = P.ip + (size_t)tile * nz * L::IPT;

    auto issue = [&](int k, bool more) {
        abar_expect(bar, (unsigned)(L::TILE * sizeof(cplx) + L::IPT * sizeof(double)));
        bulk_g2s(land, tile0 + (size_t)k * L::TILE, (unsigned)(L::TILE * sizeof(cplx)), bar);
        bulk_g2s(ipb, ip0 + (size_t)k * L::IPT, (unsigned)(L::IPT * sizeof(double)), bar);
        if (more) {                                              // next plane's bytes: DRAM -> L2 now
            bulk_prefetch_l2(tile0 + (size_t)(k + kstep) * L::TILE, (unsigned)(L::TILE * sizeof(cplx)));
            bulk_prefetch_l2(ip0 + (size_t)(k + kstep) * L::IPT, (unsigned)(L::IPT * sizeof(double)));
        }
    };
    if (tid == 0) abar_init(bar);
    fft_fill_twiddles<C>(tws, P.tw, tid, NT);
    if (NEU) for (int i = tid; i < L::DCT; i += NT) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();
    if (tid == 0 && kcount > 0) issue(kfirst, kcount > 1);
    unsigned parity = 0;

    constexpr int ITP = N / (2 * T) + 1;                             // two-spectra tiles: row pairs (kk, N-kk), kk = tl + i T
    constexpr int NCARRY = (EPT > 2 * ITP) ? EPT : 2 * ITP;
    cplx carry[NCARRY];                                          // x of the plane just left, per element of this thread
#pragma unroll
    for (int m = 0; m < NCARRY; m++) carry[m] = cmake(0.0, 0.0);
    if (P.ktw < nz) {
        // Twisted factorisation: the two eliminations met between planes m-1 and m,
        //   x_{m-1} + cp x_m = d'_{m-1},   ap x_{m-1} + x_m = e'_m      (cp = c_{m-1} / piv_{m-1}, ap = a_m / piv_m)
        // so x_m = (e'_m - ap d'_{m-1}) / (1 - ap cp) and x_{m-1} = d'_{m-1} - cp x_m.  The downward sweep starts from x_m,
        // the upward one from x_{m-1}; each CTA works them out for its own elements (slot order of its substitution).
        const int m = P.ktw;
        const double cm1 = P.zcc[m - 1], am = P.za[m];
        const cplx* dm1 = P.mid + (size_t)tile * 2 * L::TILE;      // copies left by k_yz_forward
        const cplx* em = dm1 + L::TILE;
        const double* ipm1 = ip0 + (size_t)(m - 1) * L::IPT;
        const double* iqm = ip0 + (size_t)m * L::IPT;
#pragma unroll
        for (int s = 0; s < NCARRY; s++) {
            // element of carry slot s: pair slots (row kk or N-kk) on two-spectra tiles, first-pass input slots otherwise
            const int kk = tl + (s >> 1) * T;
            const bool ok = pairing ? (kk <= N / 2 && (!(s & 1) || (kk != 0 && 2 * kk != N))) : (s < EPT);
            if (!ok) continue;
            const int e = pairing ? ((s & 1) ? N - kk : kk) * CB + c : (tl + (s / R0) * T + (s % R0) * (N / R0)) * CB + c;
            const cplx d1 = dm1[e], e0 = em[e];
            double x[2];
#pragma unroll
            for (int q = 0; q < 2; q++) {
                const int qc = q ? NCOMP - 1 : 0;
                const double cp = cm1 * ipm1[e * NCOMP + qc], ap = am * iqm[e * NCOMP + qc];
                const double dv = q ? d1.im : d1.re, ev = q ? e0.im : e0.re;
                const double xm = (ev - ap * dv) / (1.0 - ap * cp);
                x[q] = down ? xm : dv - cp * xm;
            }
            carry[s] = cmake(x[0], x[1]);
        }
    }
    double c_k = kcount > 0 ? coef[kfirst] : 0.0;

    for (int it = 0; it < kcount; it++) {
        const int k = kfirst + it * kstep;
        const bool more = it + 1 < kcount;
        abar_wait(bar, parity); parity ^= 1;
        if (!pairing) {
            // Columns with a single spectrum (no special column among them): the substitution feeds the first pass
            // of the inverse transform directly; x_{k+1} is carried per input slot of that pass.
            constexpr int NB0 = N / R0, PER0 = PassShape<N, R0, 1, T>::PER;
            static_assert(NB0 % T == 0 && PER0 * R0 == EPT, "first pass must tile the column exactly");
            const double cz = c_k;
            c_k = more ? coef[k + kstep] : 0.0;
            cplx* gk = tile0 + (size_t)k * L::TILE;
            auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
                for (int i = 0; i < PER0; i++) {
#pragma unroll
                    for (int q = 0; q < R0; q++) {
                        const int e = (tl + i * T + q * NB0) * CB + c, s = i * R0 + q;
                        const cplx dp = land[e];
                        const double ipr = ipb[e * NCOMP], ipi = ipb[e * NCOMP + (NCOMP - 1)];
                        carry[s] = cmake(dp.re - (cz * ipr) * carry[s].re, dp.im - (cz * ipi) * carry[s].im);
                        v0[i][q] = carry[s];
                    }
                }
            };
            auto next = [&]() { if (tid == 0 && more) issue(k + kstep, it + 2 < kcount); };
            auto out = [&](int n, cplx z, int) { gk[n * CB + c] = z; };
            fft_column<C, CB, true, false, false>(tl, c, true, buf, tws, load0, out, next);
            FSEI_SYNC();
            continue;
        }
        // Tiles whose columns carry two spectra: ONE pass per thread over its row pairs (kk, N-kk): substitution with
        // x_{k+1} carried per pair slot, special columns, merge (+ quarter-wave twiddle) into the staging buffer.
        {
            const double cz = c_k;
            c_k = more ? coef[k + kstep] : 0.0;
            cplx dp1[ITP], dp2[ITP];
            double ip1[ITP][NCOMP], ip2[ITP][NCOMP];
#pragma unroll
            for (int i2 = 0; i2 < ITP; i2++) {
                const int kk = tl + i2 * T;
                if (kk > N / 2) continue;
                const int e1 = kk * CB + c, e2 = (kk ? N - kk : 0) * CB + c;
                dp1[i2] = land[e1]; dp2[i2] = land[e2];
#pragma unroll
                for (int q = 0; q < NCOMP; q++) { ip1[i2][q] = ipb[e1 * NCOMP + q]; ip2[i2][q] = ipb[e2 * NCOMP + q]; }
            }
#pragma unroll
            for (int i2 = 0; i2 < ITP; i2++) {
                const int kk = tl + i2 * T;
                if (kk > N / 2) continue;
                const bool two = kk != 0 && 2 * kk != N;
                cplx& c1 = carry[2 * i2];
                c1 = cmake(dp1[i2].re - (cz * ip1[i2][0]) * c1.re, dp1[i2].im - (cz * ip1[i2][NCOMP - 1]) * c1.im);
                cplx a = c1, b = cmake(0.0, 0.0);
                if (two) {
                    cplx& c2 = carry[2 * i2 + 1];
                    c2 = cmake(dp2[i2].re - (cz * ip2[i2][0]) * c2.re, dp2[i2].im - (cz * ip2[i2][NCOMP - 1]) * c2.im);
                    b = c2;
                }
                if (tile == 0 && c == 0) {                      // separately solved columns
                    if (kk == 0) { const cplx sv = P.special[k]; a.re = sv.re; if (P.pp) a.im = sv.im; }
                    else if (P.pp && 2 * kk == N) a = P.special[nz + k];
                }
                if (kk == 0 || (!NEU && (2 * kk == N || !mine))) {
                    buf[C::pad(kk) * CB + c] = a;
                    if (two) buf[C::pad(N - kk) * CB + c] = b;
                    continue;
                }
                if (NEU && 2 * kk == N) { buf[C::pad(kk) * CB + c] = cmake(a.re * SQ2, a.im * SQ2); continue; }
                if (NEU) {
                    const cplx wk = tdct[kk];
                    const cplx ta = cmulc(cmake(a.re, -b.re), wk);     // V^a_k
                    const cplx tb = cmulc(cmake(a.im, -b.im), wk);     // V^b_k
                    a = ta; b = tb;
                }
                buf[C::pad(kk) * CB + c] = cmake(a.re - b.im, a.im + b.re);          // A + i B
                buf[C::pad(N - kk) * CB + c] = cmake(a.re + b.im, -a.im + b.re);     // conj A + i conj B
            }
        }
        FSEI_SYNC();
        if (tid == 0 && more) issue(k + kstep, it + 2 < kcount); // landing tiles consumed: prefetch the next plane
        cplx* gk = tile0 + (size_t)k * L::TILE;
        auto out = [&](int n, cplx z, int) { gk[(NEU ? dct_perm(n, N) : n) * CB + c] = z; };
        auto load0 = [&](cplx (*v0)[R0]) { fft_pass_load<N, R0, 1, T>(tl, YIn<C, CB>{buf, c}, v0); };
        fft_column<C, CB, true, true, false>(tl, c, true, buf, tws, load0, out, NoHook{});
        FSEI_SYNC();
    }
}

}  // namespace fsei
