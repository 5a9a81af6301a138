/*
 * fsei.h -- C ABI of libfsei: the fp64 pressure projection of the fractional-step
 * Navier-Stokes scheme on a staggered grid, hand-written for NVIDIA B200 (sm_100a).
 *
 * What the calls compute (P:Lnnn = line nnn of the paper text, arXiv 2103.15187):
 *   - "central second-order finite-differences discretized on a staggered mesh"   P:L87  (sec. 2.1)
 *   - "a fractional-step method is used"; the pressure "acts only as a Lagrangian
 *     multiplier assuring the solenoidal condition"                               P:L91  (sec. 2.1, Eq. 3)
 *   - periodic x,y, wall-normal z                                                 P:L240 (Fig. 4), P:L260-262 (sec. 5)
 *   - FFT as the routine of the elliptic solve, Thomas' algorithm for tridiagonals P:L30, P:L208 (sec. 3.1)
 *   - "the elliptic equation to impose mass conservation"                         P:L248 (sec. 4)
 * The paper prints no formula for the projection; the exact discrete operators are the
 * readings R1..R20 of DESIGN.md sec. 3 (standard second-order staggered projection).
 *
 * Data layout.  A field is nx*ny*nz contiguous doubles in C order [nz][ny][nx], x fastest:
 * element (i,j,k) at linear index (k*ny + j)*nx + i.  phi and p live at cell centres;
 * u[k][j][i], v[k][j][i], w[k][j][i] live on the LOW x-, y-, z-face of cell (i,j,k).
 * Periodic direction: face n is face 0.  Wall direction (z always; x or y when the bc is
 * FSEI_BC_NEUMANN): stored face 0 IS the low wall and the caller keeps it 0 (no
 * penetration); the high wall face is not stored and is 0.
 *
 * Pointers.  `zc` is a HOST pointer (copied at plan creation).  Every field pointer
 * (u, v, w, p, rhs, phi) is a DEVICE pointer to nx*ny*nz doubles, 16-byte aligned, owned
 * by the caller.  `cuda_stream` is a cudaStream_t cast to void* (NULL = default stream).
 *
 * Execution.  Calls enqueue kernels on `cuda_stream` and return; they never synchronise
 * the device and never allocate after plan creation (two documented exceptions, neither on the
 * compute path: fsei_pressure_projection_host allocates its staging fields on first use unless
 * the plan was created with FSEI_PLAN_HOST_FIELDS, and synchronises the stream before it returns;
 * fsei_plan_profile(plan, 1) creates its CUDA events when it is switched on).  A field pointer that
 * is not 16-byte aligned is rejected with FSEI_ERR_ARG.  Calls on different plans may run
 * concurrently; calls on ONE plan must be issued from one thread at a time and on one
 * stream at a time (the plan owns the factorisation tables, the scratch of the gauge
 * column and, on large grids, one workspace field that holds the spectrum in a blocked
 * layout; on small grids the transforms run in place in the caller's phi buffer).
 *
 * Errors.  Functions returning int return FSEI_OK or an FSEI_ERR_* code; nothing throws
 * across this boundary; fsei_last_error() gives a thread-local message for the last
 * failing call.  There is no CPU fallback: without a CUDA device fsei_plan_create fails
 * with FSEI_ERR_CUDA.
 */
#ifndef FSEI_H
#define FSEI_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fsei_plan fsei_plan;          /* opaque; owns device tables (wavenumbers, twiddles, z-factorisation) */

enum { FSEI_BC_PERIODIC = 0, FSEI_BC_NEUMANN = 1 };      /* bc_x, bc_y; z is always Neumann-phi / no-penetration */
enum { FSEI_OK = 0, FSEI_ERR_ARG = 1, FSEI_ERR_SIZE = 2, FSEI_ERR_GRID = 3, FSEI_ERR_ALLOC = 4, FSEI_ERR_CUDA = 5 };

/*
 * Plan for an nx x ny x nz grid (cells), uniform in x,y with extents Lx, Ly, wall-normal
 * z with face coordinates zc[0..nz] (strictly increasing; zc[0], zc[nz] are the walls;
 * cell centres are the midpoints).  DESIGN.md R2, R3, R5, R6.
 *   nx, ny : of the form 2^a 3^b 5^c in [4, 8192], nx a multiple of 4, ny even;
 *            2 <= nz <= 8192                                                    else FSEI_ERR_SIZE
 *   Lx, Ly > 0, zc finite and strictly increasing                              else FSEI_ERR_GRID
 *   bc_x, bc_y in {PERIODIC, NEUMANN}, zc != NULL                              else FSEI_ERR_ARG
 * Returns NULL on error (see fsei_last_error / fsei_last_error_code).
 */
fsei_plan*  fsei_plan_create(int nx, int ny, int nz, double Lx, double Ly,
                             const double* zc /* HOST, nz+1 */, int bc_x, int bc_y);
/*
 * Same, with per-plan options (no process-global state steers a plan):
 *   FSEI_PLAN_PATH_GENERIC | _FAST | _FUSED : force the kernel family instead of the plan's own choice (
 *       a family that has no instantiation for the size falls back to the next simpler one; FUSED with a line length
 *       whose landing tile exceeds the TMA box limit fails with FSEI_ERR_CUDA)
 *   FSEI_PLAN_TWIST_OFF / FSEI_PLAN_TWIST_ON : the twisted factorisation of the fused family
 *   FSEI_PLAN_VISC_GENERIC : fsei_viscous_step uses its generic kernels even where the fast family applies
 *   FSEI_PLAN_HOST_FIELDS : allocate, now, the five device fields fsei_pressure_projection_host stages through
 * Unknown flag bits -> FSEI_ERR_ARG.  fsei_plan_create(...) == fsei_plan_create_ex(..., 0).
 */
enum { FSEI_PLAN_PATH_GENERIC = 1, FSEI_PLAN_PATH_FAST = 2, FSEI_PLAN_PATH_FUSED = 3, FSEI_PLAN_PATH_MASK = 3,
       FSEI_PLAN_TWIST_OFF = 4, FSEI_PLAN_TWIST_ON = 8, FSEI_PLAN_HOST_FIELDS = 16, FSEI_PLAN_VISC_GENERIC = 32 };
fsei_plan*  fsei_plan_create_ex(int nx, int ny, int nz, double Lx, double Ly, const double* zc /* HOST, nz+1 */,
                                int bc_x, int bc_y, unsigned flags);
/* Kernel family the plan chose: 0 generic, 1 fast, 2 fused; +4 when the twisted factorisation is on; < 0: -FSEI_ERR_ARG. */
int         fsei_plan_kernel_family(const fsei_plan* plan);
void        fsei_plan_destroy(fsei_plan* plan);
const char* fsei_last_error(void);
int         fsei_last_error_code(void);
/* Device bytes the plan owns (tables + z-factorisation + scratch +, on large grids, one spectrum field). */
size_t      fsei_plan_workspace_bytes(const fsei_plan* plan);

/*
 * Step a1 (R4, R20):
 *   rhs = [ (u[i+1]-u[i])/dx + (v[j+1]-v[j])/dy + (w[k+1]-w[k])/dzc[k] ] / alpha_dt
 * with wrap-around in periodic directions and the missing high-wall face = 0, evaluated in
 * IEEE double in the fixed order ((du*rdx + dv*rdy) + dw*rdzc[k]) * (1/alpha_dt), no FMA.
 * rhs must not alias u, v, w.   alpha_dt == 0 or NULL pointer -> FSEI_ERR_ARG.
 */
int fsei_divergence(fsei_plan* plan, const double* u, const double* v, const double* w,
                    double alpha_dt, double* rhs, void* cuda_stream);

/*
 * Steps a2..a6 (R5-R8, R15): phi = solution of L phi = rhs,
 * L = D G the 7-point operator (periodic or homogeneous Neumann in x,y; homogeneous Neumann
 * in z), made unique by the volume-weighted zero mean  sum phi*dzc = 0.  Direct method:
 * transforms along x and y (real-to-complex FFT, or DCT-II for Neumann), one tridiagonal
 * solve per wavenumber pair along z, the (0,0) column by two prefix sums, inverse transforms.
 * phi may alias rhs (the solve runs in place in phi).
 */
int fsei_poisson_solve(fsei_plan* plan, const double* rhs, double* phi, void* cuda_stream);

/*
 * Step a7 (R4, R9), in place:
 *   u -= alpha_dt*(phi[i]-phi[i-1])/dx,  v -= alpha_dt*(phi[j]-phi[j-1])/dy,
 *   w[k] -= alpha_dt*(phi[k]-phi[k-1])/dzm[k] (k >= 1);  wall faces untouched;
 *   p += phi - beta*(L phi)   (beta = alpha_dt/(2 Re); beta == 0 -> p += phi).
 * phi must not alias u, v, w, p.
 */
int fsei_project(fsei_plan* plan, double* u, double* v, double* w, double* p, const double* phi,
                 double alpha_dt, double beta, void* cuda_stream);

/*
 * One whole projection a1..a7 enqueued back to back (the divergence is fused into the
 * x-forward transform and never written out).  phi is caller scratch of one field that
 * holds the pressure increment on return.  Same results as the three calls above.
 */
int fsei_pressure_projection(fsei_plan* plan, double* u, double* v, double* w, double* p, double* phi,
                             double alpha_dt, double beta, void* cuda_stream);

/*
 * Host-buffer convenience used for end-to-end timing: u,v,w,p are HOST pointers (pinned for
 * full speed and for the overlap below); copies them to plan-owned device fields, runs the projection,
 * copies u,v,w,p back and synchronises the stream.  The link is full duplex and p is not needed before the
 * correction a7, so u,v,w go up first, a1-a6 run, and a7 runs in up to 8 z chunks: chunk c of p goes up on a
 * plan-owned copy stream while the corrected chunks before it come down on another (same kernels, same results
 * as fsei_pressure_projection).  The 5 staging fields are allocated at plan creation when the plan was made with
 * FSEI_PLAN_HOST_FIELDS, else on first use; the two copy streams on first use; all freed with the plan.
 */
int fsei_pressure_projection_host(fsei_plan* plan, double* u, double* v, double* w, double* p,
                                  double alpha_dt, double beta, void* cuda_stream);

/*
 * ---- The two steps that precede the projection in one fluid substep ----------
 * Eq. 3:  (u^{n+1}-u^n)/dt + [gamma div(uu)^n + rho div(uu)^{n-1}] = -grad p + (1/(2Re)) lap(u^{n+1}+u^n) + f,
 * "explicit Adams-Bashforth ... for the nonlinear convective term and an implicit Crank-Nicolson method for the
 * viscous terms", gamma = 3/2, rho = -1/2, or the weights of a three-stage Runge-Kutta scheme; the
 * substep l has alpha_l = gamma_l + rho_l and beta = alpha_l dt/(2 Re).  Discrete operators: DESIGN.md V1..V12.
 *
 * fsei_explicit_terms (NEXT-2): second-order central, divergence-form convective term on the staggered mesh
 *   H_q   = -div(u q)                        at the position of each component q = u, v, w
 *   rhs_q = ((gamma_dt*H_q + rho_dt*Hprev_q) - alpha_dt*(G p)_q) + (2 beta)*(lap q)   [+ alpha_dt*f_q if a force is given:
 *           in Eq. 3 the force f stands outside the [gamma .. rho ..] bracket, so it carries the substep's weight alpha_dt]
 *   Hprev_q <- H_q
 * evaluated in IEEE double in that fixed order, no FMA: bit-identical to the definition.
 *   u, v, w, p     : in (read only).  fu, fv, fw: body force (e.g. the IB forcing), each may be NULL.
 *   hu, hv, hw     : in: H of the previous substep (zeros on the first); out: H of this substep.
 *   ru, rv, rw     : out.  No output may alias an input or another output           else FSEI_ERR_ARG
 *   Wall-face rows (w at k = 0; u at i = 0 / v at j = 0 on a wall-bounded box) get H = rhs = 0.
 *   On a slab plan (fsei_slab_plan_create) all fields are the rank's planes [k0, k1); u, v, w, p must be preceded in memory
 *   by plane k0-1 unless k0 == 0 and followed by plane k1 unless k1 == nz (one halo layer).
 */
int fsei_explicit_terms(fsei_plan* plan, const double* u, const double* v, const double* w, const double* p,
                        const double* fu, const double* fv, const double* fw, double* hu, double* hv, double* hw,
                        double* ru, double* rv, double* rw, double gamma_dt, double rho_dt, double alpha_dt,
                        double beta, void* cuda_stream);

/*
 * fsei_viscous_step (NEXT-1; sec. 3.1, Eq. 3): the implicit viscous step by approximate factorisation,
 *   q += [(1 - beta dxx)(1 - beta dyy)(1 - beta dzz)]^-1 rhs_q          for q = u, v, w, in place,
 * one tridiagonal system per grid line and direction (Thomas), cyclic in a periodic direction (the paper: Sherman-
 * Morrison; here the equivalent bordered elimination).  dxx, dyy, dzz are the second differences at
 * the staggered position of each component with no-slip walls (V3-V6); wall faces are never modified.
 *   ru, rv, rw : in: right-hand sides; DESTROYED (used as scratch).  beta >= 0 finite    else FSEI_ERR_ARG
 *   No field may alias another.  Any nx, ny, nz the plan accepts; both boundary types.
 * The factorisation tables for `beta` are built on first use (one extra small launch, plus a few microseconds of host
 * work) and kept for the last four values of beta used on this plan (a three-stage Runge-Kutta scheme cycles through
 * three); under stream capture they are rebuilt inside the graph, so a replay never depends on cached state.  Two kernel families: periodic x
 * and y with nx/32 in {2,4,8,12,16,24,32} and ny/32 in {2,3,4,6,8,12,16,24,32} run two fused launches for the three
 * components (40 B/cell each); any other grid runs the generic sweeps (nine launches).
 */
int fsei_viscous_step(fsei_plan* plan, double* u, double* v, double* w, double* ru, double* rv, double* rw,
                      double beta, void* cuda_stream);

/*
 * One whole fluid substep on a box without immersed bodies: fsei_explicit_terms -> fsei_viscous_step ->
 * fsei_pressure_projection (with the same alpha_dt, beta), enqueued back to back.  ru, rv, rw, phi are scratch fields.
 */
int fsei_fluid_substep(fsei_plan* plan, double* u, double* v, double* w, double* p, const double* fu, const double* fv,
                       const double* fw, double* hu, double* hv, double* hw, double* ru, double* rv, double* rw,
                       double* phi, double gamma_dt, double rho_dt, double alpha_dt, double beta, void* cuda_stream);

/*
 * fsei_viscous_step for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same operation (Eq. 3; the three tridiagonal sweeps of P:L208 per component),
 * computed by the generic kernel family with its factorisation tables in a file-scope `static __device__` array of libfsei
 * instead of plan-owned memory.  The call itself performs no cudaMalloc, cudaFree or allocating library call (the plan was
 * created earlier, at set-up; the array's device address is resolved then, once per device, by cudaGetSymbolAddress).
 *   Limit : nx, ny and nz each <= 1024 (the array holds 9 x (5 x 1024 + 8) doubles = 369 216 bytes, resident on every GPU
 *           that loads the library until the process exits)                                           else FSEI_ERR_SIZE
 *   Device: the current device must be the one the plan was created on                                else FSEI_ERR_ARG
 *   Result: bit-identical to fsei_viscous_step on a plan made with FSEI_PLAN_VISC_GENERIC; equal to rounding to the fast
 *           family's.  10 launches, always (no per-beta table cache: the array is shared).
 *   Sharing: every call on a device uses the same array and it keeps the last call's contents; each call rewrites all the
 *           entries it reads before it reads them (nothing needs clearing).  Calls that OVERLAP on the GPU -- other streams,
 *           other plans, other threads -- race on it: the caller serialises them.
 */
int fsei_viscous_step_noalloc(fsei_plan* plan, double* u, double* v, double* w, double* ru, double* rv, double* rw,
                              double beta, void* cuda_stream);

/*
 * ---- IB-MLS transfer operators (Eq. 4, Fig. 2; sec. 3.2) -----------------
 * "A three-dimensional support domain consisting of N_e = n x n x n Eulerian nodes (n = 3 ...) is created around each
 * Lagrangian marker, and the fluid velocity at the body position is computed interpolating ...
 *      u_i(x_b) = sum_{k=1..N_e} phi_i^k(x_b) u_i(x_k)                                              (Eq. 4)
 * ... a linear basis function is used, p^T(x) = [1, x, y, z], with an exponential weight function centered at the
 * location of the Lagrangian marker.  The interpolated velocity is used to compute the IB force at the exact location
 * of the marker which is then transferred back to the Eulerian grid-points as a distributed forcing ... for the three
 * velocity components."  Support, weight, force and spreading scale: readings M1..M8 of DESIGN.md sec. 3.
 *
 * Markers: n >= 0 markers as DEVICE arrays xm, ym, zm (coordinates; taken modulo the period in a periodic direction;
 * in a wall direction the support is clamped inside the box), area (the surface area each marker stands for).
 * Marker values (ub.., Fu.., Vu..) are DEVICE arrays of n doubles per component.  nz >= 3            else FSEI_ERR_SIZE
 *
 *   fsei_mls_interpolate : ub[l] = sum_k phi^k u(x_k) on u's staggered nodes; vb, wb alike.               (Eq. 4)
 *   fsei_mls_spread      : fu(x_k) += c_l phi^k Fu[l], c_l = area[l] h_l / sum_k phi^k dV_k (total force conserved);
 *                          fv, fw alike.  fp64 atomic adds: the sum over markers has no fixed order.
 *   fsei_ibm_forcing     : Fu[l] = (Vu[l] - ub[l]) * inv_dt (out), then the spreading of Fu into fu (+=); v, w alike:
 *                          the IB forcing f of Eq. 3 that fsei_explicit_terms takes as fu, fv, fw.  One kernel.
 *   fsei_ibm_apply_forcing: the forcing fields are zero except on the supports of the markers, so a substep need not stream
 *                          them: call fsei_explicit_terms WITHOUT a body force, then this -- it visits the support nodes of the
 *                          same markers and forms rhs += alpha_dt * f there (the two operations of the dense path, in its
 *                          order: same result), each node once, and leaves fu, fv, fw all-zero for the next substep.
 *                          Requires fu, fv, fw to be zero outside those supports (zero-fill them once, at allocation).
 * The forcing fields must not alias the velocity fields                                              else FSEI_ERR_ARG
 */
int fsei_mls_interpolate(fsei_plan* plan, long n, const double* xm, const double* ym, const double* zm,
                         const double* u, const double* v, const double* w, double* ub, double* vb, double* wb,
                         void* cuda_stream);
int fsei_mls_spread(fsei_plan* plan, long n, const double* xm, const double* ym, const double* zm, const double* area,
                    const double* Fu, const double* Fv, const double* Fw, double* fu, double* fv, double* fw,
                    void* cuda_stream);
int fsei_ibm_forcing(fsei_plan* plan, long n, const double* xm, const double* ym, const double* zm, const double* area,
                     const double* Vu, const double* Vv, const double* Vw, const double* u, const double* v, const double* w,
                     double inv_dt, double* Fu, double* Fv, double* Fw, double* fu, double* fv, double* fw,
                     void* cuda_stream);
int fsei_ibm_apply_forcing(fsei_plan* plan, long n, const double* xm, const double* ym, const double* zm, double* fu, double* fv,
                           double* fw, double* ru, double* rv, double* rw, double alpha_dt, void* cuda_stream);

/*
 * ---- Multi-GPU slab decomposition of the projection: per-rank stages -------------------------
 * "the Cartesian domain is split into slabs ... at most one halo layer is required on each side of a slab";
 * "all-to-all communications ... needed to solve both the equation for the provisional velocity and for the elliptic
 * equation".  One process per GPU.  A rank owns
 *   planes [k0, k1) of u, v, w, p, phi (a z-slab)            for a1-a3 and a5-a7, and
 *   x-slots [s0, s1) of the nx/2 packed wavenumber slots, for every row and EVERY plane (full z columns), for a4.
 * Between fsei_slab_forward and fsei_pencil_solve, and between fsei_pencil_solve and fsei_slab_backward, the spectrum
 * changes hands by an all-to-all (paper_2103_15187_b200/slab.py, torch.distributed).
 * Periodic x and y only; nx/2 and ny in the fast family's lengths                          else FSEI_ERR_ARG / _SIZE
 *
 * Layouts (DEVICE pointers, 16-byte aligned).  nzl = k1 - k0, nsl = s1 - s0.
 *   slab field   : [nzl][ny][nx] doubles.  w must be followed in memory by plane k1 (the neighbour's first plane) unless
 *                  k1 == nz; phi passed to fsei_slab_project must be preceded by plane k0-1 unless k0 == 0, and, when
 *                  beta != 0, followed by plane k1 unless k1 == nz.  (The pointer is the address of local plane 0.)
 *   slab spectrum: [nzl][ny][nx/2] complex (re, im), the packed natural-order layout of DESIGN.md sec. 2.
 *   pencil       : [nz][ny][nsl] complex: element (k, row, s0 + s) of the spectrum.
 */
fsei_plan* fsei_slab_plan_create(int nx, int ny, int nz, double Lx, double Ly, const double* zc /* HOST, nz+1, GLOBAL */,
                                 int bc_x, int bc_y, int k0, int k1, int s0, int s1);
/*
 * Peer-store exchange (the all-to-all folded into the kernels' epilogues).  Gives the plan the
 * pencil and the slab-spectrum buffer of EVERY rank (device pointers; on a multi-GPU node the peers' buffers mapped into
 * this process, e.g. torch symmetric memory) with the plane ranges k0s[0..nranks] and slot ranges s0s[0..nranks]
 * (nranks <= 8).  From then on fsei_slab_forward stores its result straight into the owners' pencils (its `spec`
 * argument is scratch) and fsei_pencil_solve stores its result straight into the owners' slab spectra (its `pencil`
 * keeps the forward-eliminated column); the caller orders the ranks (all forwards before any solve, all solves before
 * any backward).  nranks = 0 switches back to local results + explicit exchange.
 */
int fsei_slab_set_peers(fsei_plan* plan, int nranks, void* const* pencils, void* const* specs, const int* k0s, const int* s0s);
/* a1-a3 on the slab: spec = y-transform of x-transform of D(u,v,w)/alpha_dt.  spec must not alias u, v, w. */
int fsei_slab_forward(fsei_plan* plan, const double* u, const double* v, const double* w, double alpha_dt,
                      double* spec, void* cuda_stream);
/* a4 on the pencil, in place (the rank with s0 == 0 also solves the gauge column). */
int fsei_pencil_solve(fsei_plan* plan, double* pencil, void* cuda_stream);
/* a5, a6 on the slab: phi = inverse transforms of spec (phi may alias spec). */
int fsei_slab_backward(fsei_plan* plan, double* spec, double* phi, void* cuda_stream);
/* a7 on the slab (halo planes of phi as described above). */
int fsei_slab_project(fsei_plan* plan, double* u, double* v, double* w, double* p, const double* phi,
                      double alpha_dt, double beta, void* cuda_stream);

/*
 * The implicit viscous step on slabs (the all-to-all also serves "the equation for the provisional velocity").
 * fsei_slab_viscous_xy : the x and y sweeps of (I - beta dxx)(I - beta dyy) dq = r on the rank's planes, in place in ru, rv, rw.
 * fsei_pencil_viscous_z: the z sweep (I - beta dzz) of component comp (0 u, 1 v, 2 w) on full z columns, in place.  The real
 *                        slab field [nzl][ny][nx] is read as [nzl][ny][nx/2] pairs, so the pencil [nz][ny][2 nsl] doubles holds
 *                        columns x in [2 s0, 2 s1) and the spectrum's exchange lists serve unchanged.
 * fsei_slab_field_add  : q += r on the rank's planes (the provisional velocity q^ = q + dq).
 * The three together give the same result as fsei_viscous_step on the whole grid (same sweeps, same order).
 */
int fsei_slab_viscous_xy(fsei_plan* plan, double* ru, double* rv, double* rw, double beta, void* cuda_stream);
int fsei_pencil_viscous_z(fsei_plan* plan, double* pencil, int comp, double beta, void* cuda_stream);
int fsei_slab_field_add(fsei_plan* plan, double* q, const double* r, void* cuda_stream);

/*
 * Kernel-level timing aid for bench.py: number of kernels enqueued by the last
 * fsei_pressure_projection / fsei_poisson_solve call on this plan.
 */
int fsei_plan_last_launch_count(const fsei_plan* plan);

/*
 * Per-kernel device timing for the roofline report: while enabled, every launch the calls
 * above enqueue is bracketed by a pair of CUDA events on the caller's stream.
 * fsei_plan_profile_read waits for the recorded events, returns how many kernel kinds there are
 * (<= max_kernels; a NEGATIVE value -FSEI_ERR_* on failure) and fills, per kind, the summed
 * milliseconds and launch count since the last read (and, if names != NULL, static name strings);
 * it resets the sums.  fsei_plan_profile(plan, 1) creates the event pool (2048 launches between reads).
 */
int fsei_plan_profile(fsei_plan* plan, int enable);
int fsei_plan_profile_read(fsei_plan* plan, int max_kernels, double* ms_sum, long* count, const char** names);

#ifdef __cplusplus
}
#endif
#endif /* FSEI_H */
