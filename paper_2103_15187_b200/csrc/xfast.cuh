// xfast.cuh -- fast-path kernels of steps a1+a2 (divergence fused into the x-forward transform) and a6
// (x-inverse transform), for line lengths nx = 2 N with N = 2^a or 3 2^a (include/fsei.h; P:L30, P:L87,
// P:L91; R15, sec. 6).
//
// A CTA of T*LPB threads owns LPB adjacent x-lines (rows j) and marches along z over `kchunk` planes:
// T threads per line, each holding the line's butterflies of one Stockham pass in registers
// (fast_fft.cuh).  The lines of plane k+1 are fetched by the TMA engine (cp.async.bulk into a shared-memory
// landing tile, completion on an mbarrier) while the CTA transforms plane k, so no thread ever waits on a
// global load.  Real lines are transformed as N complex values z_t = x[2t] + i x[2t+1] followed
// (forward) or preceded (inverse) by the Hermitian pair step; Neumann lines go through Makhoul's
// even/odd reorder (staged in shared memory) and the quarter-wave twiddle (DCT-II / DCT-III).
//
// Spectrum layout (natural order, in place in the phi buffer): line (j,k) holds N complex slots;
//   periodic: slot 0 = (X_0, X_N) (both real), slot s = X_s for s = 1..N-1
//   Neumann : slot 0 = (X_0, X_N),             slot s = (X_s, X_{nx-s})
// Marching along z gives the fused divergence its reuse: the w(k+1) lines a CTA reads for plane k are the
// w(k) lines it reads one iteration later, so u, v, w each come from DRAM once.
#pragma once
#include "kernel_env.cuh"
#include "fast_fft.cuh"
#include "plan_types.cuh"
#include "stencil.cuh"
#include "xfft.cuh"
#include <type_traits>

namespace fsei {

struct XFast {
    int nx, ny, nz, N;          // N = nx / 2
    int kchunk;                 // planes per CTA
    const cplx* tw;             // e^{-2 pi i j / N},  j in [0, N)
    const cplx* tw_r2c;         // e^{-2 pi i k / nx}, k in [0, N/2]
    const cplx* tw_dct;         // e^{-i pi k / (2 nx)}, k in [0, N]   (Neumann only)
    double scale;               // 1 / (N ny), applied by the inverse store
};

template <class C> struct SmIn {
    const cplx* s;
    FSEI_HD cplx operator()(int n) const { return s[C::pad(n)]; }
};
template <class C> struct SmOut {
    cplx* s;
    FSEI_HD void operator()(int n, cplx v, int = 0) const { s[C::pad(n)] = v; }
};

// staging tile of a real line (Neumann): one pad double every 4 keeps the stride-4 reads of the reorder
// conflict-free
FSEI_HD int xs_pad(int s) { return s + (s >> 2); }
FSEI_HD int xs_pitch(int n) { return n + (n >> 2) + 2; }
// Makhoul: index of the natural line element that sits at position s of the reordered sequence v
FSEI_HD int makhoul(int s, int n) { return (s < (n >> 1)) ? 2 * s : 2 * (n - 1 - s) + 1; }

// lines per CTA and shared-memory carve-up of the x kernels.
//   [mbarrier | landing tile (TMA destination) | line buffers | twiddles | r2c twiddles | dct twiddles | staging]
// landing tile: forward: u lines [LPB], v lines [LPB+1] (row j+1 of the last line), w lines of planes k and k+1
// [2][LPB] (doubles, n per line); inverse / non-fused forward: LPB lines of n doubles.
template <class C, bool NEU> struct XShape {
    static constexpr int N = C::N;
    static constexpr size_t tables = sizeof(cplx) * (C::TW + N / 2 + 1 + (NEU ? N + 1 : 0));
    static constexpr size_t bytes(int L) {
        return 128 + sizeof(double) * (size_t)(4 * L + 1) * 2 * N + sizeof(cplx) * (size_t)L * (C::PITCH + 8) + tables +
               (NEU ? sizeof(double) * (size_t)L * (2 * N + (2 * N >> 2) + 2) : 0);
    }
    static constexpr int fit(int L) { return (L <= 1 || bytes(L) <= 200 * 1024) ? L : fit(L - 1); }
    static constexpr int pow2_floor(int v) { return v <= 1 ? 1 : 2 * pow2_floor(v / 2); }
    // about 256 threads, <= 200 KB, a power of two: the blocked layout's segments (16 LPB CB bytes) stay 128-byte
    // aligned and LPB divides the usual ny
    static constexpr int LPB = fit(pow2_floor((256 / C::T) > 0 ? (256 / C::T) : 1));
};

// LL = lines of n doubles in the landing tile: 4 LPB + 1 (fused forward) or LPB
template <class C, int LPB, bool NEU, int LL> struct XSmemLayout {
    static constexpr int N = C::N;
    static constexpr int LAND = LL * 2 * N;                     // doubles
    static constexpr int BUF = LPB * (C::PITCH + 8);            // complex (slack: the blocked x-inverse pads its line pitch to 2 mod 8)
    static constexpr int TWS = C::TW;
    static constexpr int R2C = N / 2 + 1;
    static constexpr int DCT = NEU ? N + 1 : 0;
    static constexpr int XS = NEU ? LPB * (2 * N + (2 * N >> 2) + 2) : 0;     // doubles
    static constexpr size_t BYTES = 128 + sizeof(double) * LAND + sizeof(cplx) * (BUF + TWS + R2C + DCT) + sizeof(double) * XS;
};


// Whole line transform for the threads of one line.  load0(v) fills the first pass' registers (from the landing
// tile / staging; IN_BUF: from the line buffer itself, then a barrier separates its reads from the writes);
// `out` receives the natural-order result (OUT_BUF: it writes the line buffer, so a barrier precedes it).
// hook() runs on every thread right after the first barrier, i.e. once every thread has consumed its first-pass
// input (that is where the next tile's asynchronous load is issued).  Must be reached by every thread of the CTA;
// `act` false = this thread's line does not exist.
struct NoHook { FSEI_HD void operator()() const {} };

// gid >= 0: the line's T threads are whole warps (T % 32 == 0) and synchronise among themselves through named barrier
// gid + 1, so that the lines of a CTA drift apart instead of meeting at every pass; the barrier that precedes a real
// hook stays CTA-wide (the hook is where the landing tile, read by every line, is refilled).
template <class C, bool INV, bool IN_BUF, bool OUT_BUF, class Load0, class Out, class Hook>
FSEI_DEV void fft_line(int tl, bool act, cplx* buf, const cplx* tws, Load0 load0, Out out, Hook hook, int gid = -1)
{
    constexpr int N = C::N, T = C::T;
    constexpr bool HOOKED = !std::is_same<Hook, NoHook>::value;
    static_assert(C::NP >= 2, "pipelined kernels need at least two passes");
    SmIn<C> bin{buf}; SmOut<C> bout{buf};
    auto lsync = [&]() { if (T % 32 == 0 && gid >= 0) { FSEI_GROUP_SYNC(gid + 1, T); } else { FSEI_SYNC(); } };
    {
        cplx v[PassShape<N, C::R0, 1, T>::PER][C::R0];
        if (act) load0(v);
        if (IN_BUF) { if (HOOKED) { FSEI_SYNC(); } else lsync(); hook(); }
        if (act) fft_pass_compute<N, C::R0, 1, T, INV>(tl, tws, v, bout);
    }
    if (!IN_BUF && HOOKED) { FSEI_SYNC(); } else lsync();
    if (!IN_BUF) hook();
    {
        cplx v[PassShape<N, C::R1, C::R0, T>::PER][C::R1];
        if (act) fft_pass_load<N, C::R1, C::R0, T>(tl, bin, v);
        if constexpr (C::NP == 2) {
            if (OUT_BUF) lsync();
            if (act) fft_pass_compute<N, C::R1, C::R0, T, INV>(tl, tws, v, out);
            return;
        } else {
            lsync();
            if (act) fft_pass_compute<N, C::R1, C::R0, T, INV>(tl, tws, v, bout);
        }
    }
    lsync();
    if constexpr (C::NP >= 3) {
        cplx v[PassShape<N, C::R2, C::R0 * C::R1, T>::PER][C::R2];
        if (act) fft_pass_load<N, C::R2, C::R0 * C::R1, T>(tl, bin, v);
        if (OUT_BUF) lsync();
        if (act) fft_pass_compute<N, C::R2, C::R0 * C::R1, T, INV>(tl, tws + C::TW1, v, out);
    }
}

FSEI_HD cplx ld2(const double* p) { return *reinterpret_cast<const cplx*>(p); }
FSEI_HD void st2(double* p, cplx v) { *reinterpret_cast<cplx*>(p) = v; }

// Spectrum layouts.  CB = 0: natural, line (j,k) holds its N slots contiguously at (k ny + j) N.
// CB > 0: blocked by x-slot tiles of CB slots, [N / CB][nz][ny][CB] -- the (ny x CB) tile of one plane is contiguous,
// which is what the z-marching y kernels (yzfused.cuh) stream; slot p of line (j,k) sits at
// ((p / CB) nz + k) ny + j) CB + p % CB.
template <int CB> FSEI_HD size_t spec_index(int N, int ny, int nz, int k, int j, int p)
{
    if (CB == 0) return ((size_t)k * ny + j) * N + p;
    return (((size_t)(p / (CB ? CB : 1)) * nz + k) * ny + j) * CB + p % (CB ? CB : 1);
}
template <int CB> struct SpecLine {
    cplx* base; size_t tstride;
    FSEI_HD SpecLine(cplx* spec, int N, int ny, int nz, int k, int j)
        : base(spec + ((size_t)k * ny + j) * (CB ? CB : N)), tstride((size_t)nz * ny * CB) {}
    FSEI_HD cplx& operator[](int p) const { return CB ? base[(size_t)(p / (CB ? CB : 1)) * tstride + p % (CB ? CB : 1)] : base[p]; }
};
// rows (x-slot tiles) per TMA box of the blocked x-inverse load: the largest divisor of nxt that is <= 256
FSEI_HD constexpr int xi_box_tiles(int nxt) { int b = nxt < 256 ? nxt : 256; while (nxt % b) b--; return b; }

// ---------------------------------------------------------------------------------------------------
// a1 + a2: spec(line) = R2C / DCT-II of  rhs(line),  rhs = D(u,v,w)/(alpha dt) (FUSED) or read from `u`
// grid (ceil(ny / LPB), ceil(nz / kchunk)), block T*LPB, dynamic shared memory XSmemLayout::BYTES
// ---------------------------------------------------------------------------------------------------
template <class C, int LPB, bool NEU, bool FUSED, int CB = 0>
FSEI_GLOBAL(C::T * LPB, 1) k_xf_fast(XFast P, SParams S, const double* u, const double* v, const double* w,
                                     double inv_adt, cplx* spec)
{
    using L = XSmemLayout<C, LPB, NEU, (FUSED ? 4 * LPB + 1 : LPB)>;
    constexpr int N = C::N, T = C::T, R0 = C::R0;
    constexpr int NB0 = N / R0, PER0 = PassShape<N, R0, 1, T>::PER;
    static_assert(NB0 % T == 0, "first pass must tile the line exactly");
    constexpr int NPAIR = N / T;                                  // real pairs per thread
    constexpr int n = 2 * N;
    FSEI_DYN_SMEM(smraw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    double* land = reinterpret_cast<double*>(smraw + 128);
    cplx* buf = reinterpret_cast<cplx*>(land + L::LAND);
    cplx* tws = buf + L::BUF;
    cplx* tr2c = tws + L::TWS;
    cplx* tdct = tr2c + L::R2C;
    double* xs = reinterpret_cast<double*>(tdct + L::DCT);
    double* LU = land;                                            // [LPB][n]
    double* LV = LU + LPB * n;                                    // [LPB + 1][n]
    double* LW = LV + (LPB + 1) * n;                              // [2][LPB][n], plane k in slot k & 1
    const int tid = threadIdx.x, nt = T * LPB;
    const int li = tid / T, tl = tid - li * T;
    const int ny = P.ny, nz = P.nz;
    const int j0 = blockIdx.x * LPB, j = j0 + li;
    const int nl = (ny - j0 < LPB) ? ny - j0 : LPB;               // lines of this CTA that exist
    const bool act = j < ny;
    const int k0 = blockIdx.y * P.kchunk, k1 = (k0 + P.kchunk < nz) ? k0 + P.kchunk : nz;
    const size_t plane = (size_t)ny * n;
    const int nzw = nz + (S.halo_hi ? 1 : 0);                     // planes of w there are: a z-slab is followed by its neighbour's first plane
    const bool yper = S.bcy == BC_PERIODIC, xper = S.bcx == BC_PERIODIC;
    const bool wrap = (j0 + nl == ny);                            // row j+1 of the last line wraps (or is a wall)
    const bool has_jp = (j + 1 < ny) || yper;

    // asynchronous load of the tile of plane k (one thread)
    auto issue = [&](int k) {
        const unsigned lb = n * sizeof(double);
        const size_t g0 = ((size_t)k * ny + j0) * n;
        if (!FUSED) {
            abar_expect(bar, nl * lb);
            bulk_g2s(LU, u + g0, nl * lb, bar);
            if (k + 1 < k1) bulk_prefetch_l2(u + g0 + plane, nl * lb);
            return;
        }
        const int nv = wrap ? nl : nl + 1;
        const bool first = (k == k0), up = (k + 1 < nzw);
        unsigned total = nl * lb + nv * lb + ((wrap && yper) ? lb : 0) + (first ? nl * lb : 0) + (up ? nl * lb : 0);
        abar_expect(bar, total);
        bulk_g2s(LU, u + g0, nl * lb, bar);
        bulk_g2s(LV, v + g0, nv * lb, bar);
        if (wrap && yper) bulk_g2s(LV + nl * n, v + (size_t)k * plane, lb, bar);
        if (first) bulk_g2s(LW + (size_t)(k & 1) * LPB * n, w + g0, nl * lb, bar);
        if (up) bulk_g2s(LW + (size_t)((k + 1) & 1) * LPB * n, w + g0 + plane, nl * lb, bar);
        if (k + 1 < k1) {                                          // the plane after: DRAM -> L2 now
            bulk_prefetch_l2(u + g0 + plane, nl * lb);
            bulk_prefetch_l2(v + g0 + plane, nv * lb);
            if (k + 2 < nzw) bulk_prefetch_l2(w + g0 + 2 * plane, nl * lb);
        }
    };

    if (tid == 0) abar_init(bar);
    fft_fill_twiddles<C>(tws, P.tw, tid, nt);
    for (int i = tid; i < L::R2C; i += nt) tr2c[i] = P.tw_r2c[i];
    if (NEU) for (int i = tid; i < L::DCT; i += nt) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();
    if (tid == 0 && k0 < k1) issue(k0);
    unsigned parity = 0;

    cplx* lbuf = buf + li * C::PITCH;
    double* lxs = xs + (NEU ? li * xs_pitch(n) : 0);
    const double* lu = LU + li * n;
    const double* lv = LV + li * n;

    double rdz_next = (FUSED && k0 < k1) ? S.rdzc[k0 + S.kofs] : 0.0;      // (a z-slab: the metric tables are global)
    for (int k = k0; k < k1; k++) {
        const double rdz_k = rdz_next;                             // metric of this plane, loaded one plane ahead
        if (FUSED && k + 1 < k1) rdz_next = S.rdzc[k + 1 + S.kofs];
        abar_wait(bar, parity); parity ^= 1;
        // (rhs[2t], rhs[2t+1]) of line (j,k) from the landing tile
        auto rhs_pair = [&](int t) -> cplx {
            if (!FUSED) return ld2(lu + 2 * t);
            const double* lwk = LW + ((size_t)(k & 1) * LPB + li) * n;
            const double* lwp = LW + ((size_t)((k + 1) & 1) * LPB + li) * n;
            cplx uu = ld2(lu + 2 * t);
            double un = (2 * t + 2 < n) ? lu[2 * t + 2] : (xper ? lu[0] : 0.0);
            cplx vv = ld2(lv + 2 * t);
            cplx vp = has_jp ? ld2(lv + n + 2 * t) : cmake(0.0, 0.0);
            cplx wk = ld2(lwk + 2 * t);
            cplx wp = (k + 1 < nzw) ? ld2(lwp + 2 * t) : cmake(0.0, 0.0);
            const double rdz = rdz_k;
            return cmake(div_cell(uu.re, uu.im, vv.re, vp.re, wk.re, wp.re, S.rdx, S.rdy, rdz, inv_adt),
                         div_cell(uu.im, un, vv.im, vp.im, wk.im, wp.im, S.rdx, S.rdy, rdz, inv_adt));
        };
        auto next = [&]() { if (tid == 0 && k + 1 < k1) issue(k + 1); };
        if (NEU) {
            // stage the real line, then the first pass reads it through Makhoul's reorder
            if (act) {
#pragma unroll
                for (int e = 0; e < NPAIR; e++) {
                    int t = tl + e * T;
                    cplx r = rhs_pair(t);
                    lxs[xs_pad(2 * t)] = r.re; lxs[xs_pad(2 * t + 1)] = r.im;
                }
            }
            FSEI_SYNC();
            next();
        }
        auto load0 = [&](cplx (*v0)[R0]) {
#pragma unroll
            for (int i = 0; i < PER0; i++) {
#pragma unroll
                for (int q = 0; q < R0; q++) {
                    const int t = tl + i * T + q * NB0;
                    if (NEU) v0[i][q] = cmake(lxs[xs_pad(makhoul(2 * t, n))], lxs[xs_pad(makhoul(2 * t + 1, n))]);
                    else v0[i][q] = rhs_pair(t);
                }
            }
        };
        if (NEU) fft_line<C, false, false, true>(tl, act, lbuf, tws, load0, SmOut<C>{lbuf}, NoHook{}, li);
        else fft_line<C, false, false, true>(tl, act, lbuf, tws, load0, SmOut<C>{lbuf}, next, li);
        FSEI_SYNC();
        // Hermitian pair step (+ quarter-wave twiddle): Z -> packed half spectrum, written to global memory
        auto pair_store = [&](const cplx* lb, const SpecLine<CB>& g, int p) {
            if (p == 0) {
                cplx z = lb[0];
                double x0 = z.re + z.im, xn = z.re - z.im;
                if (NEU) xn *= FSEI_SQRT1_2;                               // X_{n/2} = V_{n/2} cos(pi/4)
                g[0] = cmake(x0, xn);
            } else {
                cplx zk = lb[C::pad(p)], zm = lb[C::pad(N - p)];
                cplx E = cmake(0.5 * (zk.re + zm.re), 0.5 * (zk.im - zm.im));   // (Zk + conj Zm)/2
                cplx D = cmake(zk.re - zm.re, zk.im + zm.im);                   // Zk - conj Zm
                cplx O = cmake(0.5 * D.im, -0.5 * D.re);                        // D / (2i)
                cplx Tt = cmul(O, tr2c[p]);
                cplx xk = cadd(E, Tt), xm = cconj(csub(E, Tt));
                if (NEU) { xk = dct_tw_fwd(xk, tdct[p]); xm = dct_tw_fwd(xm, tdct[N - p]); }
                g[p] = xk;
                if (p != N - p) g[N - p] = xm;
            }
        };
        if (CB == 0) {
            if (act) {
                const SpecLine<CB> g(spec, N, ny, nz, k, j);
                for (int p = tl; p <= N / 2; p += T) pair_store(lbuf, g, p);
            }
        } else {
            // blocked layout: adjacent threads take (slot within tile, line, tile) in that order, so that a warp
            // writes whole 16 LPB CB-byte segments of the [tile][k][j][CB] array
            constexpr int CBq = CB ? CB : 1, HP = N / 2 / CBq + 1;
            for (int wi = tid; wi < HP * LPB * CBq; wi += nt) {
                const int cc = wi % CBq, l2 = (wi / CBq) % LPB, p = (wi / (CBq * LPB)) * CBq + cc;
                if (p > N / 2 || l2 >= nl) continue;
                pair_store(buf + l2 * C::PITCH, SpecLine<CB>(spec, N, ny, nz, k, j0 + l2), p);
            }
        }
        FSEI_SYNC();
    }
}

// ---------------------------------------------------------------------------------------------------
// a6: phi(line) = scale * C2R / DCT-III of spec(line), in place
// ---------------------------------------------------------------------------------------------------
// CB > 0: the spectrum is in the blocked layout and the landing tile is fetched through `map`, a 3-D view
// (2 ny CB doubles, nz, N / CB) of it with boxes (2 LPB CB, 1, xi_box_tiles(N / CB)): landing tile [N / CB][LPB][CB].
// CB = 0 (natural layout): the landing tile is line-major [LPB][N], and the Hermitian pair step (half spectrum -> Z) is
// FOLDED into the first pass' loads: a thread forms its R0 inputs Z(m) straight from X(m), X(N-m) of the landing tile
// (unit stride across the threads of a line in both directions: no bank conflicts), so the line skips the separate pair
// phase with its shared-memory round trip and CTA barrier; each pair is then evaluated by both of its owners -- a few more
// flops on an fp64 pipe that is a third busy (configs[1]: 0.066 -> 0.058 ms).  On the blocked layout a line-major landing
// tile would need one TMA box per line with a 32-byte inner dimension, which the TMA engine serves at a third of the
// speed of the 128-byte boxes (measured: x_inverse 2.65 -> 8.7 ms at configs[3]).  There the fold is done on the
// [tile][line][CB] tile as it lands, with the THREADS remapped instead: eight consecutive threads are (slot-in-tile 0..1) x
// (line 0..3) of one tile, so a quarter-warp reads 128 contiguous bytes of the landing tile for X(m) and -- the mirror
// tiles of the two slots being neighbours -- a permutation of 128 contiguous bytes for X(N-m); the line buffers get a
// pitch of 2 (mod 8) elements so that the same eight threads (two neighbouring butterflies of four lines) stay
// conflict-free in every pass.  A warp then holds all four lines, so the passes meet at CTA barriers.
template <class C, int LPB, bool NEU, int CB = 0>
FSEI_GLOBAL(C::T * LPB, (XSmemLayout<C, LPB, NEU, LPB>::BYTES <= 112 * 1024 ? 2 : 1)) k_xi_fast(XFast P, const FSEI_GRID_CONSTANT TmaMap3D map, const cplx* spec, double* phi)
{
    using L = XSmemLayout<C, LPB, NEU, LPB>;
    constexpr int N = C::N, T = C::T, R0 = C::R0;
    constexpr int NPAIR = N / T;
    constexpr int n = 2 * N;
    FSEI_DYN_SMEM(smraw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smraw);
    cplx* land = reinterpret_cast<cplx*>(smraw + 128);             // [LPB][N] packed spectrum lines
    cplx* buf = reinterpret_cast<cplx*>(reinterpret_cast<double*>(smraw + 128) + L::LAND);
    cplx* tws = buf + L::BUF;
    cplx* tr2c = tws + L::TWS;
    cplx* tdct = tr2c + L::R2C;
    double* xs = reinterpret_cast<double*>(tdct + L::DCT);
    const int tid = threadIdx.x, nt = T * LPB;
    constexpr int CBm = CB ? CB : 1;
    // natural layout: thread = (line, butterfly) line-major.  Blocked layout: (slot in tile, line, tile) fastest-first
    const int li = CB ? (tid / CBm) % LPB : tid / T;
    const int tl = CB ? (tid / (CBm * LPB)) * CBm + tid % CBm : tid - li * T;
    constexpr int XP = CB ? C::PITCH + ((10 - C::PITCH % 8) % 8) : C::PITCH;      // line-buffer pitch (blocked: 2 mod 8)
    static_assert(CB == 0 || (T % CBm == 0 && XP <= C::PITCH + 8), "blocked x-inverse thread mapping");
    const int ny = P.ny, nz = P.nz;
    const int j0 = blockIdx.x * LPB, j = j0 + li;
    const int nl = (ny - j0 < LPB) ? ny - j0 : LPB;
    const bool act = j < ny;
    const int k0 = blockIdx.y * P.kchunk, k1 = (k0 + P.kchunk < nz) ? k0 + P.kchunk : nz;
    auto issue = [&](int k) {
        if (CB == 0) {
            const unsigned bytes = (unsigned)(nl * N * sizeof(cplx));
            abar_expect(bar, bytes);
            bulk_g2s(land, spec + ((size_t)k * ny + j0) * N, bytes, bar);
        } else {                                                   // whole boxes: rows past ny arrive as zeros
            constexpr int NXT = N / (CB ? CB : 1), BT = xi_box_tiles(NXT);
            abar_expect(bar, (unsigned)(LPB * N * sizeof(cplx)));
#pragma unroll
            for (int b = 0; b < NXT / BT; b++) tma_load_3d(land + (size_t)b * BT * LPB * CB, &map, 2 * j0 * CB, k, b * BT, bar);
            if (k + 1 < k1) {                                      // the plane after: DRAM -> L2 now
#pragma unroll
                for (int b = 0; b < NXT / BT; b++) tma_prefetch_3d(&map, 2 * j0 * CB, k + 1, b * BT);
            }
        }
    };
    if (tid == 0) abar_init(bar);
    fft_fill_twiddles<C>(tws, P.tw, tid, nt);
    for (int i = tid; i < L::R2C; i += nt) tr2c[i] = P.tw_r2c[i];
    if (NEU) for (int i = tid; i < L::DCT; i += nt) tdct[i] = P.tw_dct[i];
    FSEI_SYNC();
    if (tid == 0 && k0 < k1) issue(k0);
    unsigned parity = 0;

    cplx* lbuf = buf + li * XP;
    double* lxs = xs + (NEU ? li * xs_pitch(n) : 0);
    const double scale = P.scale;

    // Z(m), m in [0, N), of this thread's line from the landing tile (line-major, or [tile][line][CB] on the blocked
    // layout): element m and element N - m come from the same pair (X_p, X_{N-p}), p = min(m, N - m)
    const cplx* FSEI_RESTRICT land_r = land;
    const cplx* FSEI_RESTRICT tr2c_r = tr2c;
    const cplx* FSEI_RESTRICT tdct_r = tdct;
    auto xat = [&](int q) -> cplx { return CB ? land_r[((q / CBm) * LPB + li) * CBm + q % CBm] : land_r[li * N + q]; };
    auto zin = [&](int m) -> cplx {
        if (m == 0) {
            const cplx s = xat(0);
            double x0 = s.re, xn = s.im;
            if (NEU) xn *= 1.41421356237309504880168872420969808;
            return cmake(0.5 * (x0 + xn), 0.5 * (x0 - xn));
        }
        const bool lo = 2 * m <= N;
        const int p = lo ? m : N - m;
        cplx xk = xat(p), xm = xat(N - p);
        if (NEU) { xk = dct_tw_inv(xk, tdct_r[p]); xm = dct_tw_inv(xm, tdct_r[N - p]); }
        const cplx E = cmake(0.5 * (xk.re + xm.re), 0.5 * (xk.im - xm.im));    // (Xk + conj Xm)/2
        const cplx Tt = cmake(0.5 * (xk.re - xm.re), 0.5 * (xk.im + xm.im));   // (Xk - conj Xm)/2
        const cplx O = cmulc(Tt, tr2c_r[p]);
        return lo ? cmake(E.re - O.im, E.im + O.re)                            // E + i O
                  : cmake(E.re + O.im, -(E.im - O.re));                        // conj(E - i O)
    };
    const int gid = CB ? -1 : li;          // blocked layout: a warp holds all the lines of the CTA -> CTA barriers

    for (int k = k0; k < k1; k++) {
        abar_wait(bar, parity); parity ^= 1;
        auto next = [&]() { if (tid == 0 && k + 1 < k1) issue(k + 1); };          // landing tile consumed: fetch the next plane
        double* gl = phi + ((size_t)k * ny + j) * n;
        auto load0 = [&](cplx (*v0)[R0]) { fft_pass_load<N, R0, 1, T>(tl, zin, v0); };
        if (!NEU) {
            auto out = [&](int t, cplx z, int) { st2(gl + 2 * t, cmake(z.re * scale, z.im * scale)); };
            fft_line<C, true, false, false>(tl, act, lbuf, tws, load0, out, next, gid);
        } else {
            auto out = [&](int t, cplx z, int) {
                lxs[xs_pad(makhoul(2 * t, n))] = z.re * scale; lxs[xs_pad(makhoul(2 * t + 1, n))] = z.im * scale;
            };
            fft_line<C, true, false, false>(tl, act, lbuf, tws, load0, out, next, gid);
            FSEI_SYNC();
            if (act) {
#pragma unroll
                for (int e = 0; e < NPAIR; e++) {
                    int t = tl + e * T;
                    st2(gl + 2 * t, cmake(lxs[xs_pad(2 * t)], lxs[xs_pad(2 * t + 1)]));
                }
            }
        }
        FSEI_SYNC();
    }
}

}  // namespace fsei
