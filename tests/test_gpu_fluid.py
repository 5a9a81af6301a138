"""GPU parity of the fluid-substep steps that precede the projection against the oracle,
through the C ABI (include/fsei.h: fsei_explicit_terms, fsei_viscous_step, fsei_fluid_substep).

Gates:
  explicit terms : BIT-EXACT (np.array_equal) -- stencils in a fixed IEEE-double order on both sides;
  viscous step   : max|q_gpu - q_oracle| <= 1e-12 * max|dq| + 2 ulp(max|q|) against the long-double oracle (the second
                   term is the rounding of the final q + dq in double on one side and long double on the other).
                   Derivation: each factor
                   (1 - beta d2) is an M-matrix with condition number <= 1 + 4 beta / h_min^2 (~2.5e3 for the wall cells
                   of configs[3] at Re = 3000, dt = 1e-3); the bordered / plain Thomas elimination is backward stable on
                   it, so the fp64 error is ~ eps * cond ~ 3e-13 relative to |dq|.
"""
import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

pytestmark = pytest.mark.gpu
P, W = 0, 1
EPS = 2.0 ** -52
ALL_BC = [(P, P), (W, W), (P, W), (W, P)]
SHAPES = [(32, 32, 32), (48, 24, 20), (36, 16, 33), (64, 12, 7), (40, 20, 12)]
# + grids with tiles whose halo lies inside the grid (they take TMA boxes; the rim keeps per-thread copies), ragged tiles on
# both axes and several z chunks per column of tiles
EXPL_SHAPES = SHAPES + [(96, 36, 9), (192, 54, 70), (144, 24, 5)]


def _case(shape, bc, seed=40, s=2.5, n=10):
    nx, ny, nz = shape
    g = (nx, ny, nz, 1.0, 1.5, inputs.tanh_grid(nz, s), bc[0], bc[1])
    f = [inputs.normal_field(seed, i, (nz, ny, nx)) for i in range(n)]
    u, v, w = f[:3]
    w[0] = 0
    if bc[0] == W: u[:, :, 0] = 0
    if bc[1] == W: v[:, 0, :] = 0
    return g, f


def _dev(arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in arrs]


def _plan(g):
    from paper_2103_15187_b200.binding import Plan
    return Plan.from_grid(g)


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("shape", EXPL_SHAPES)
@pytest.mark.parametrize("force", [False, True])
def test_explicit_terms_bit_exact(oracle_ld, shape, bc, force):
    import torch
    g, f = _case(shape, bc)
    u, v, w, p, h0, h1, h2, f0, f1, f2 = f
    gdt, rdt, adt, beta = 1.5e-3, -0.5e-3, 1e-3, 1e-3 / (2 * 300.0)
    ff = (f0, f1, f2) if force else (None, None, None)
    ho = [h0.copy(), h1.copy(), h2.copy()]
    ro = oracle_ld.explicit_terms(g, u, v, w, p, *ho, gdt, rdt, adt, beta, f=ff)
    plan = _plan(g)
    du, dv, dw, dp, dh0, dh1, dh2 = _dev([u, v, w, p, h0, h1, h2])
    dr = [torch.empty_like(du) for _ in range(3)]
    df = _dev(ff) if force else (None, None, None)
    plan.explicit_terms(du, dv, dw, dp, dh0, dh1, dh2, *dr, gdt, rdt, adt, beta, f=df)
    torch.cuda.synchronize()
    for c in range(3):
        assert np.array_equal(dr[c].cpu().numpy(), ro[c]), ("rhs", c)
        assert np.array_equal((dh0, dh1, dh2)[c].cpu().numpy(), ho[c]), ("H", c)
    assert np.array_equal(du.cpu().numpy(), u) and np.array_equal(dp.cpu().numpy(), p)      # inputs untouched
    plan.destroy()


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("beta", [1e-3 / 6000.0, 2e-3, 0.5])
def test_viscous_step_vs_oracle(oracle_ld, shape, bc, beta):
    import torch
    g, f = _case(shape, bc, seed=41)
    u, v, w, ru, rv, rw = f[:6]
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, ru, rv, rw, beta)
    plan = _plan(g)
    d = _dev([u, v, w, ru, rv, rw])
    plan.viscous_step(*d, beta)
    torch.cuda.synchronize()
    for c, (q0, qo) in enumerate(((u, uo), (v, vo), (w, wo))):
        got = d[c].cpu().numpy()
        scale = np.abs(qo - q0).max()
        assert np.abs(got - qo).max() <= 1e-12 * scale + 2 * EPS * np.abs(qo).max(), (c, np.abs(got - qo).max() / scale)
    # wall faces never move
    assert np.array_equal(d[2].cpu().numpy()[0], w[0])
    if bc[0] == W: assert np.array_equal(d[0].cpu().numpy()[:, :, 0], u[:, :, 0])
    if bc[1] == W: assert np.array_equal(d[1].cpu().numpy()[:, 0, :], v[:, 0, :])
    # a second call with another beta rebuilds the tables
    d2 = _dev([u, v, w, ru, rv, rw])
    plan.viscous_step(*d2, beta * 3)
    torch.cuda.synchronize()
    uo2, vo2, wo2 = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo2, vo2, wo2, ru, rv, rw, beta * 3)
    assert np.abs(d2[0].cpu().numpy() - uo2).max() <= 1e-12 * np.abs(uo2 - u).max() + 2 * EPS * np.abs(uo2).max()
    plan.destroy()


def test_viscous_step_config_grid_wall_cells(oracle_ld):
    """configs[3]'s z-grid (clustering 3.5, nz = 768) at reduced x,y and a physiological beta: the wall cells have
    beta/dz^2 ~ 3e2 ... the stiffest factor of the headline workload."""
    import torch
    g = inputs.make_grid(4, shape=(64, 32, 768))
    f = [inputs.normal_field(42, i, (768, 32, 64)) for i in range(6)]
    u, v, w, ru, rv, rw = f
    w[0] = 0
    beta = 1e-3 / (2 * 3000.0)
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, ru, rv, rw, beta)
    plan = _plan(g)
    d = _dev(f)
    plan.viscous_step(*d, beta)
    torch.cuda.synchronize()
    for c, (q0, qo) in enumerate(((u, uo), (v, vo), (w, wo))):
        assert np.abs(d[c].cpu().numpy() - qo).max() <= 1e-12 * np.abs(qo - q0).max() + 2 * EPS * np.abs(qo).max(), c
    plan.destroy()


@pytest.mark.parametrize("bc", [(P, P), (W, W)])
def test_fluid_substep_chain_vs_oracle(oracle_ld, bc):
    """Three RK3 substeps (explicit terms -> viscous step -> projection) enqueued with no host sync."""
    import torch
    shape = (48, 24, 20)
    g, f = _case(shape, bc, seed=43)
    u, v, w = [0.1 * t for t in f[:3]]
    p = np.zeros_like(u)
    h = [np.zeros_like(u) for _ in range(3)]
    dt, Re = 2e-3, 200.0
    gam, rho = (8 / 15, 5 / 12, 3 / 4), (0.0, -17 / 60, -5 / 12)
    plan = _plan(g)
    d = _dev([u, v, w, p] + h)
    scratch = [torch.empty_like(d[0]) for _ in range(4)]
    uo, vo, wo, po = u.copy(), v.copy(), w.copy(), p.copy()
    ho = [t.copy() for t in h]
    for l in range(3):
        al = gam[l] + rho[l]
        beta = al * dt / (2 * Re)
        plan.fluid_substep(*d[:4], *d[4:], *scratch, gam[l] * dt, rho[l] * dt, al * dt, beta)
        r = oracle_ld.explicit_terms(g, uo, vo, wo, po, *ho, gam[l] * dt, rho[l] * dt, al * dt, beta)
        oracle_ld.viscous_step(g, uo, vo, wo, *r, beta)
        oracle_ld.pressure_projection(g, uo, vo, wo, po, al * dt, beta)
    torch.cuda.synchronize()
    for c, ref in enumerate((uo, vo, wo, po)):
        got = d[c].cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max()), (c, np.abs(got - ref).max())
    div = np.abs(oracle_ld.divergence(g, *[d[c].cpu().numpy() for c in range(3)], 1.0)).max()
    assert div <= 1e-10, div
    plan.destroy()


def test_fluid_error_codes():
    import torch
    from paper_2103_15187_b200.binding import FseiError, ERR_ARG
    g, f = _case((32, 32, 32), (P, P))
    plan = _plan(g)
    d = _dev(f[:7])
    r = [torch.empty_like(d[0]) for _ in range(3)]
    with pytest.raises(FseiError) as e:
        plan.viscous_step(d[0], d[1], d[2], d[0], r[1], r[2], 1e-3)             # rhs aliases u
    assert e.value.code == ERR_ARG
    with pytest.raises(FseiError) as e:
        plan.viscous_step(d[0], d[1], d[2], *r, -1.0)                            # beta < 0
    assert e.value.code == ERR_ARG
    with pytest.raises(FseiError) as e:
        plan.explicit_terms(*d[:4], d[4], d[5], d[6], d[0], r[1], r[2], 1e-3, 0.0, 1e-3, 0.0)   # output aliases input
    assert e.value.code == ERR_ARG
    plan.destroy()


# ---------------------------------------------------------------------------------------------
# fast family of the viscous step (periodic x, y; partition solves in registers; two fused launches)
# ---------------------------------------------------------------------------------------------
FAST_SHAPES = [(64, 64, 9), (128, 96, 12), (256, 192, 7), (384, 256, 5), (512, 384, 5), (768, 512, 4), (1024, 768, 3),
               (1024, 1024, 2), (64, 1024, 40), (1024, 64, 33), (320, 160, 6), (640, 640, 4), (640, 320, 3), (576, 576, 4), (960, 576, 3), (576, 960, 3)]


@pytest.mark.parametrize("shape", FAST_SHAPES)
@pytest.mark.parametrize("beta", [1e-3 / 6000.0, 3e-4])
def test_viscous_fast_family_vs_oracle(oracle_ld, shape, beta):
    """beta/dx^2 spans 0.0007 (decoupled chunks) .. 300 (every unknown of a line coupled to every other)."""
    import torch
    from paper_2103_15187_b200 import binding
    g, f = _case(shape, (P, P), seed=44, n=6)
    u, v, w, ru, rv, rw = f
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, ru, rv, rw, beta)
    plan = _plan(g)
    d = _dev(f)
    plan.viscous_step(*d, beta)
    torch.cuda.synchronize()
    assert plan.last_launch_count == 3                              # factorisation tables + two fused passes
    for c, (q0, qo) in enumerate(((u, uo), (v, vo), (w, wo))):
        got = d[c].cpu().numpy()
        scale = np.abs(qo - q0).max()
        assert np.abs(got - qo).max() <= 1e-12 * scale + 2 * EPS * np.abs(qo).max(), (c, np.abs(got - qo).max() / scale)
    assert np.array_equal(d[2].cpu().numpy()[0], w[0])
    plan.viscous_step(*d, beta)                                      # same beta again: the tables are kept
    assert plan.last_launch_count == 2
    plan.destroy()
    # the generic family on the same grid (forced per plan) agrees to rounding
    pg = binding.Plan.from_grid(g, binding.VISC_GENERIC)
    dg = _dev(f)
    pg.viscous_step(*dg, beta)
    torch.cuda.synchronize()
    assert pg.last_launch_count == 10
    for c, qo in enumerate((uo, vo, wo)):
        assert np.abs(dg[c].cpu().numpy() - qo).max() <= 1e-12 * np.abs(qo - f[c]).max() + 2 * EPS * np.abs(qo).max()
    pg.destroy()


def test_viscous_beta_cache_and_graph_capture(oracle_ld):
    """The factorisation tables are kept for the last four betas (RK3 cycles through three); a whole fluid substep can be
    captured in a CUDA graph (no call synchronises or allocates) and replays correctly after other betas have been used."""
    import torch
    shape = (64, 64, 16)
    g, f = _case(shape, (P, P), seed=45, n=7)
    u, v, w, p, ru, rv, rw = f
    plan = _plan(g)
    betas = [1e-4, 2e-4, 3e-4]
    d = _dev([u, v, w, ru, rv, rw])
    for b in betas:
        plan.viscous_step(*d, b)
        assert plan.last_launch_count == 3                          # first use: tables built
    for b in betas:
        plan.viscous_step(*d, b)
        assert plan.last_launch_count == 2                          # cached
    # --- graph capture of one fluid substep
    dt, Re = 2e-3, 300.0
    beta = dt / (2 * Re)
    u0, v0, w0 = [0.1 * t for t in (u, v, w)]
    fld = _dev([u0, v0, w0, np.zeros_like(u)] + [np.zeros_like(u) for _ in range(7)])
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        plan.fluid_substep(*fld, 1.5 * dt, -0.5 * dt, dt, beta)
    torch.cuda.synchronize()
    for b in (5e-4, 6e-4, 7e-4, 8e-4, 9e-4):                        # evict every slot
        plan.viscous_step(*_dev([u, v, w, ru, rv, rw]), b)
    for t, a in zip(fld, [u0, v0, w0, np.zeros_like(u)] + [np.zeros_like(u) for _ in range(7)]):
        t.copy_(torch.from_numpy(a))
    graph.replay()
    torch.cuda.synchronize()
    uo, vo, wo, po = u0.copy(), v0.copy(), w0.copy(), np.zeros_like(u)
    ho = [np.zeros_like(u) for _ in range(3)]
    r = oracle_ld.explicit_terms(g, uo, vo, wo, po, *ho, 1.5 * dt, -0.5 * dt, dt, beta)
    oracle_ld.viscous_step(g, uo, vo, wo, *r, beta)
    oracle_ld.pressure_projection(g, uo, vo, wo, po, dt, beta)
    for c, ref in enumerate((uo, vo, wo, po)):
        assert np.abs(fld[c].cpu().numpy() - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max()), c
    plan.destroy()


# ---------------------------------------------------------------------------------------------
# configs[3] at FULL size (1024 x 1024 x 768), the launch configuration bench.py's fluid leg times: IB forcing of 1.19 M
# markers, explicit terms from TMA tiles in 64-plane marches, forcing applied on the markers' supports, fast viscous family
# ---------------------------------------------------------------------------------------------
def test_config4_full_size_fluid_rows(oracle_ld):
    """IB forcing: marker forces and the whole forcing fields against the oracle.  Explicit terms (+ apply): bit-exact on
    sampled groups of planes the oracle computes from sub-grids (a local stencil: the interior planes of a sub-grid of 8
    planes see the same inputs and metrics as in the whole grid) -- bottom wall, a 64-plane march boundary, the planes through
    the immersed body, top wall.  Viscous step: every output against the long-double oracle run on the whole grid."""
    import torch
    from paper_2103_15187_b200.binding import Plan
    if torch.cuda.get_device_properties(0).total_memory < 100e9:
        pytest.skip("needs a GPU with >= 100 GB")
    avail = 0.0
    with open("/proc/meminfo") as fh:
        for line in fh:
            if line.startswith("MemAvailable"):
                avail = int(line.split()[1]) / 1e6
    if avail < 120:
        pytest.skip(f"full-size oracle needs about 90 GB of host memory, {avail:.0f} GB available")
    case = inputs.make_case(4)
    g, nx, ny, nz = case.grid, case.nx, case.ny, case.nz
    zc = np.asarray(g[5])
    hu = [case.u, case.v, case.w]
    for a in hu:
        a *= 0.05
    hu[2][0] = 0
    dt, Re = case.alpha_dt, 3000.0
    gdt, rdt, adt, beta = 1.5 * dt, -0.5 * dt, dt, dt / (2 * Re)
    plan = Plan.from_grid(g)
    u, v, w = (torch.from_numpy(a).cuda() for a in hu)
    z = lambda: torch.zeros_like(u)
    p, h, r, f = z(), [z(), z(), z()], [z(), z(), z()], [z(), z(), z()]
    # ---- IB forcing (the marker cloud of bench.py)
    n = int(4 * 3.14159 * 0.3 ** 2 * nx * ny / (case.Lx * case.Ly))
    xm, ym, zm, area, V = inputs.sphere_markers(n, (0.5 * case.Lx, 0.5 * case.Ly, 0.5), 0.3, seed=7)
    dm = _dev([xm, ym, zm, area, *V])
    F = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.ibm_forcing(n, *dm[:4], *dm[4:], u, v, w, 1.0 / dt, *F, *f)
    torch.cuda.synchronize()
    fo = [np.zeros((nz, ny, nx)) for _ in range(3)]
    Fo = oracle_ld.ibm_forcing(g, xm, ym, zm, area, V, *hu, 1.0 / dt, fo)
    groups = [(0, 8, 0, 6), (60, 68, 2, 6), (380, 388, 2, 6), (nz - 8, nz, 2, 8)]        # sub-grid [a, b), compared sub-planes [lo, hi)
    fsub = [[None] * 3 for _ in groups]
    for c in range(3):
        assert np.abs(F[c].cpu().numpy() - Fo[c]).max() <= 1e-12 * np.abs(Fo[c]).max(), c
        got = f[c].cpu().numpy()
        assert np.count_nonzero(got) > n                                                   # the supports are there
        assert np.abs(got - fo[c]).max() <= 1e-12 * np.abs(fo[c]).max(), c
        for gi, (a, b, _, _) in enumerate(groups):
            fsub[gi][c] = got[a:b].copy()
        fo[c] = None
        del got
    del fo
    # ---- explicit terms without a dense force, then the forcing on the supports
    plan.explicit_terms(u, v, w, p, *h, *r, gdt, rdt, adt, beta)
    assert plan.last_launch_count == 1
    plan.ibm_apply_forcing(n, *dm[:3], *f, *r, adt)
    torch.cuda.synchronize()
    for c in range(3):
        assert not bool(f[c].any()), c                                                     # cleared for the next substep
    del f
    for gi, (a, b, lo, hi) in enumerate(groups):
        gs = (nx, ny, b - a, g[3], g[4], zc[a:b + 1].copy(), g[6], g[7])
        sub = [np.ascontiguousarray(t[a:b]) for t in hu]
        hs = [np.zeros_like(sub[0]) for _ in range(3)]
        rs = oracle_ld.explicit_terms(gs, *sub, np.zeros_like(sub[0]), *hs, gdt, rdt, adt, beta, f=tuple(fsub[gi]))
        for c in range(3):
            assert np.array_equal(r[c][a + lo:a + hi].cpu().numpy(), rs[c][lo:hi]), ("rhs", gi, c)
            assert np.array_equal(h[c][a + lo:a + hi].cpu().numpy(), hs[c][lo:hi]), ("H", gi, c)
    del h, fsub
    # ---- implicit viscous step on the whole grid
    hr = [t.cpu().numpy() for t in r]
    plan.viscous_step(u, v, w, *r, beta)
    assert plan.last_launch_count == 3                                                     # tables + the two fused passes
    torch.cuda.synchronize()
    q0max = [float(np.abs(a).max()) for a in hu]
    q0 = [a[nz // 2].copy() for a in hu]
    oracle_ld.viscous_step(g, *hu, *hr, beta)
    del hr
    for c, t in enumerate((u, v, w)):
        got = t.cpu().numpy()
        scale = float(np.abs(hu[c][nz // 2] - q0[c]).max())                                # size of the increment (one plane is enough)
        err = float(np.abs(got - hu[c]).max())
        print(f"cfg 4 FULL viscous comp {c}: max err {err:.2e}  increment ~{scale:.2e}  max|q| {q0max[c]:.2e}")
        assert err <= 1e-12 * scale + 2 * EPS * q0max[c], c
        del got
    plan.destroy()


# ---------------------------------------------------------------------------------------------
# degenerate and extreme cases of the fluid rows
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc", [((8192, 4, 3), (P, P)), ((4, 8192, 3), (P, P)), ((8192, 4, 3), (W, W)), ((4, 4, 2), (P, P)),
                                      ((4, 4, 2), (W, W)), ((8, 6, 1025), (P, W))])
def test_fluid_rows_at_extreme_sizes(oracle_ld, shape, bc):
    """the longest lines the plan accepts (8192), the smallest grid (4 x 4 x 2), a column longer than any other test's: explicit
    terms bit-exact, viscous step to rounding"""
    import torch
    g, f = _case(shape, bc, seed=46, n=7)
    u, v, w, p, h0, h1, h2 = f
    gdt, rdt, adt, beta = 1.5e-3, -0.5e-3, 1e-3, 2e-3
    ho = [h0.copy(), h1.copy(), h2.copy()]
    ro = oracle_ld.explicit_terms(g, u, v, w, p, *ho, gdt, rdt, adt, beta)
    plan = _plan(g)
    d = _dev(f)
    dr = [torch.empty_like(d[0]) for _ in range(3)]
    plan.explicit_terms(*d, *dr, gdt, rdt, adt, beta)
    torch.cuda.synchronize()
    for c in range(3):
        assert np.array_equal(dr[c].cpu().numpy(), ro[c]), ("rhs", c)
        assert np.array_equal(d[4 + c].cpu().numpy(), ho[c]), ("H", c)
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, *ro, beta)
    plan.viscous_step(d[0], d[1], d[2], *dr, beta)
    torch.cuda.synchronize()
    for c, (q0, qo) in enumerate(((u, uo), (v, vo), (w, wo))):
        assert np.abs(d[c].cpu().numpy() - qo).max() <= 1e-12 * np.abs(qo - q0).max() + 2 * EPS * np.abs(qo).max(), c
    plan.destroy()


@pytest.mark.parametrize("shape", [(64, 64, 9), (36, 16, 33)])
def test_fluid_rows_degenerate_inputs(shape):
    """beta = 0: the implicit operator is the identity, q += r exactly (both families).  u = v = w = 0, p = const: H = 0 and the rhs
    is exactly alpha dt f (0 without a force); rho dt Hprev passes through."""
    import torch
    from paper_2103_15187_b200 import binding
    g, f = _case(shape, (P, P), seed=47, n=9)
    for flags in (0, binding.VISC_GENERIC):
        plan = binding.Plan.from_grid(g, flags)
        d = _dev(f[:6])
        want = [d[c] + d[3 + c] for c in range(3)]
        want[2][0] = d[2][0]                                                       # the wall face of w is a fixed row (V7)
        plan.viscous_step(*d, 0.0)
        torch.cuda.synchronize()
        for c in range(3):
            assert torch.equal(d[c], want[c]), (flags, c)
        plan.destroy()
    plan = _plan(g)
    z = [torch.zeros(f[0].shape, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    p = torch.full_like(z[0], 3.25)
    hp = _dev(f[3:6])
    force = _dev(f[6:9])
    r = [torch.empty_like(z[0]) for _ in range(3)]
    hprev = [t.clone() for t in hp]
    plan.explicit_terms(*z, p, *hp, *r, 1.5e-3, -0.5e-3, 1e-3, 1e-4, f=tuple(force))
    torch.cuda.synchronize()
    for c in range(3):
        assert not bool(hp[c].any()), c                                           # H = 0
        want = (-0.5e-3 * hprev[c]) + 1e-3 * force[c]
        if c == 2:
            want[0] = 0                                                           # the wall face of w
        assert torch.equal(r[c], want), c
    plan.destroy()
