"""GPU parity of the IB-MLS transfer operators (include/fsei.h: fsei_mls_interpolate, fsei_mls_spread,
fsei_ibm_forcing) against the long-double oracle, through the C ABI.

Gates: the shape functions are the solution of a well-conditioned 4 x 4 system in marker-centred
scaled coordinates (condition number ~1e2), so fp64 gives phi to ~1e-14; interpolated values within 1e-12 * max|u|;
spread fields within 1e-12 * max|f| (the atomic sum over markers has no fixed order: a few ulp of the largest term).
"""
import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

pytestmark = pytest.mark.gpu
P, W = 0, 1


def _dev(arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in arrs]


def _setup(shape, bc, n, centre, radius, seed):
    nx, ny, nz = shape
    g = (nx, ny, nz, 1.0, 1.5, inputs.tanh_grid(nz, 2.5), bc[0], bc[1])
    u, v, w = (inputs.normal_field(60 + seed, c, (nz, ny, nx)) for c in range(3))
    xm, ym, zm, area, V = inputs.sphere_markers(n, centre, radius, seed=seed)
    return g, (u, v, w), (xm, ym, zm), area, V


CASES = [((32, 32, 32), (P, P), 500, (0.5, 0.75, 0.5), 0.3), ((48, 24, 20), (P, P), 777, (0.05, 1.45, 0.5), 0.35),
         ((36, 16, 33), (W, W), 300, (0.5, 0.75, 0.5), 0.48), ((64, 12, 7), (P, W), 64, (0.9, 0.7, 0.4), 0.3)]


@pytest.mark.parametrize("shape,bc,n,centre,radius", CASES)
def test_mls_interpolate_spread_forcing_vs_oracle(oracle_ld, shape, bc, n, centre, radius):
    import torch
    from paper_2103_15187_b200.binding import Plan
    g, vel, mk, area, V = _setup(shape, bc, n, centre, radius, seed=len(shape) + n)
    plan = Plan.from_grid(g)
    dvel, dmk, (darea,), dV = _dev(vel), _dev(mk), _dev([area]), _dev(V)
    # interpolation (Eq. 4)
    Ub = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.mls_interpolate(n, *dmk, *dvel, *Ub)
    Uo = oracle_ld.mls_interpolate(g, *mk, *vel)
    for c in range(3):
        assert np.abs(Ub[c].cpu().numpy() - Uo[c]).max() <= 1e-12 * np.abs(vel[c]).max(), c
    # spreading of given marker forces
    rng = np.random.default_rng(n)
    F = [rng.standard_normal(n) for _ in range(3)]
    fo = [np.zeros_like(vel[0]) for _ in range(3)]
    oracle_ld.mls_spread(g, *mk, area, F, fo)
    df = [torch.zeros_like(dvel[0]) for _ in range(3)]
    plan.mls_spread(n, *dmk, darea, *_dev(F), *df)
    for c in range(3):
        assert np.abs(df[c].cpu().numpy() - fo[c]).max() <= 1e-12 * np.abs(fo[c]).max(), c
    # the fused forcing call, accumulating on top of an existing field
    f0 = [inputs.normal_field(70, c, vel[0].shape) for c in range(3)]
    fo = [t.copy() for t in f0]
    Fo = oracle_ld.ibm_forcing(g, *mk, area, V, *vel, 500.0, fo)
    df = _dev(f0)
    dF = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.ibm_forcing(n, *dmk, darea, *dV, *dvel, 500.0, *dF, *df)
    torch.cuda.synchronize()
    for c in range(3):
        assert np.abs(dF[c].cpu().numpy() - Fo[c]).max() <= 1e-12 * np.abs(Fo[c]).max(), c
        assert np.abs(df[c].cpu().numpy() - fo[c]).max() <= 1e-12 * np.abs(fo[c]).max(), c
    plan.destroy()


def test_mls_linear_field_exact_on_gpu():
    """Property that holds at any size (no oracle): a linear field is interpolated exactly, for each component on its
    own staggered nodes of a stretched grid -- here at 256 x 128 x 192 with 200 000 markers."""
    import torch
    from paper_2103_15187_b200.binding import Plan
    nx, ny, nz = 256, 128, 192
    zc = inputs.tanh_grid(nz, 3.0)
    g = (nx, ny, nz, 1.0, 1.0, zc, W, W)
    plan = Plan.from_grid(g)
    zmid = 0.5 * (zc[:-1] + zc[1:])
    coef = [(0.3, 1.1, -0.7, 0.4), (-0.2, 0.5, 0.9, -1.3), (0.8, -0.6, 0.2, 0.7)]
    fields = []
    for c in range(3):
        x = (np.arange(nx) + (0 if c == 0 else 0.5)) / nx
        y = (np.arange(ny) + (0 if c == 1 else 0.5)) / ny
        z = zc[:-1] if c == 2 else zmid
        a, bx, by, bz = coef[c]
        fields.append(a + bx * x[None, None, :] + by * y[None, :, None] + bz * z[:, None, None])
    n = 200_000
    xm, ym, zm, area, V = inputs.sphere_markers(n, (0.5, 0.5, 0.5), 0.4, seed=9)
    d = _dev(fields)
    dm = _dev([xm, ym, zm])
    out = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.mls_interpolate(n, *dm, *d, *out)
    torch.cuda.synchronize()
    for c in range(3):
        a, bx, by, bz = coef[c]
        assert np.abs(out[c].cpu().numpy() - (a + bx * xm + by * ym + bz * zm)).max() < 1e-13, c
    # and the spreading conserves the total force: sum f dV = sum F area h_l
    F = _dev([np.ones(n)] * 3)
    f = [torch.zeros_like(d[0]) for _ in range(3)]
    plan.mls_spread(n, *dm, _dev([area])[0], *F, *f)
    torch.cuda.synchronize()
    dzc = np.diff(zc); dzm = np.r_[0.0, np.diff(zmid)]
    for c in range(3):
        dz = dzm if c == 2 else dzc
        z = zc[:-1] if c == 2 else zmid
        total = (f[c].cpu().numpy() * dz[:, None, None]).sum() / (nx * ny)
        kc = np.clip(np.abs(z[None, :] - zm[:2000, None]).argmin(axis=1), 1, nz - 2)      # h_l of a sample: the sphere is symmetric
        kc_all = np.clip(np.searchsorted(0.5 * (z[1:] + z[:-1]), zm), 1, nz - 2)
        assert np.array_equal(kc, kc_all[:2000])
        want = (area * (1 / nx + 1 / ny + dz[kc_all]) / 3).sum()
        assert abs(total - want) <= 1e-11 * want, c
    plan.destroy()


def test_substep_with_ib_forcing_vs_oracle(oracle_ld):
    """IB forcing -> explicit terms (f enters H) -> viscous step -> projection, against the same chain of the oracle."""
    import torch
    from paper_2103_15187_b200.binding import Plan
    g, vel, mk, area, V = _setup((48, 24, 20), (P, P), 400, (0.5, 0.75, 0.5), 0.3, seed=5)
    vel = [0.1 * t for t in vel]
    vel[2][0] = 0
    n = 400
    dt, Re = 2e-3, 200.0
    beta = dt / (2 * Re)
    plan = Plan.from_grid(g)
    d = _dev(vel) + [torch.zeros(vel[0].shape, dtype=torch.float64, device="cuda:0") for _ in range(11)]
    u, v, w, p, hu, hv, hw, ru, rv, rw, phi, fu, fv, fw = d
    dm, (da,), dV = _dev(mk), _dev([area]), _dev(V)
    dF = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.ibm_forcing(n, *dm, da, *dV, u, v, w, 1.0 / dt, *dF, fu, fv, fw)
    plan.fluid_substep(u, v, w, p, hu, hv, hw, ru, rv, rw, phi, 1.5 * dt, -0.5 * dt, dt, beta, f=(fu, fv, fw))
    torch.cuda.synchronize()
    uo, vo, wo = (t.copy() for t in vel)
    po = np.zeros_like(uo)
    fo = [np.zeros_like(uo) for _ in range(3)]
    ho = [np.zeros_like(uo) for _ in range(3)]
    oracle_ld.ibm_forcing(g, *mk, area, V, uo, vo, wo, 1.0 / dt, fo)
    r = oracle_ld.explicit_terms(g, uo, vo, wo, po, *ho, 1.5 * dt, -0.5 * dt, dt, beta, f=fo)
    oracle_ld.viscous_step(g, uo, vo, wo, *r, beta)
    oracle_ld.pressure_projection(g, uo, vo, wo, po, dt, beta)
    for c, (got, ref) in enumerate(zip((u, v, w, p), (uo, vo, wo, po))):
        assert np.abs(got.cpu().numpy() - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max()), c
    plan.destroy()


@pytest.mark.parametrize("shape,bc,n,centre,radius", CASES)
def test_apply_forcing_equals_dense_body_force(oracle_ld, shape, bc, n, centre, radius):
    """explicit terms without a force + fsei_ibm_apply_forcing on the markers' supports == explicit terms with the dense forcing
    fields: bit for bit given the same f (the same two operations per node), and against the oracle's chain; f is all-zero
    afterwards; a second apply is a no-op."""
    import torch
    from paper_2103_15187_b200.binding import Plan
    g, vel, mk, area, V = _setup(shape, bc, n, centre, radius, seed=7)
    if bc[0] == W: vel[0][:, :, 0] = 0
    if bc[1] == W: vel[1][:, 0, :] = 0
    vel[2][0] = 0
    dt, beta = 2e-3, 1e-5
    plan = Plan.from_grid(g)
    u, v, w = _dev(vel)
    z = lambda: torch.zeros_like(u)
    p, fu, fv, fw = z(), z(), z(), z()
    ha, hb, ra, rb = [z() for _ in range(3)], [z() for _ in range(3)], [z() for _ in range(3)], [z() for _ in range(3)]
    dm, (da,), dV = _dev(mk), _dev([area]), _dev(V)
    dF = [torch.empty(n, dtype=torch.float64, device="cuda:0") for _ in range(3)]
    plan.ibm_forcing(n, *dm, da, *dV, u, v, w, 1.0 / dt, *dF, fu, fv, fw)
    dense_f = [t.clone() for t in (fu, fv, fw)]
    plan.explicit_terms(u, v, w, p, *ha, *ra, 1.5 * dt, -0.5 * dt, dt, beta, f=(fu, fv, fw))            # dense path
    plan.explicit_terms(u, v, w, p, *hb, *rb, 1.5 * dt, -0.5 * dt, dt, beta)                            # sparse path
    plan.ibm_apply_forcing(n, *dm, fu, fv, fw, *rb, dt)
    assert plan.last_launch_count == 1
    torch.cuda.synchronize()
    for c in range(3):
        assert torch.equal(ra[c], rb[c]), c
        assert torch.equal(ha[c], hb[c]), c
        assert not (fu, fv, fw)[c].any(), c                                                              # cleared for the next substep
    keep = [t.clone() for t in rb]
    plan.ibm_apply_forcing(n, *dm, fu, fv, fw, *rb, dt)
    torch.cuda.synchronize()
    for c in range(3):
        assert torch.equal(keep[c], rb[c]), c
    # the oracle's chain (dense by definition); the spread's atomic order is the only difference
    fo = [np.zeros_like(vel[0]) for _ in range(3)]
    ho = [np.zeros_like(vel[0]) for _ in range(3)]
    oracle_ld.ibm_forcing(g, *mk, area, V, *vel, 1.0 / dt, fo)
    ro = oracle_ld.explicit_terms(g, *vel, np.zeros_like(vel[0]), *ho, 1.5 * dt, -0.5 * dt, dt, beta, f=fo)
    for c in range(3):
        assert np.abs(rb[c].cpu().numpy() - ro[c]).max() <= 1e-12 * max(1.0, np.abs(ro[c]).max()), c
        assert np.abs(dense_f[c].cpu().numpy() - fo[c]).max() <= 1e-12 * max(1.0, np.abs(fo[c]).max()), c
    plan.destroy()


def test_mls_edge_cases():
    import torch
    from paper_2103_15187_b200.binding import Plan, FseiError, ERR_ARG
    g, vel, mk, area, V = _setup((32, 32, 32), (P, P), 10, (0.5, 0.75, 0.5), 0.3, seed=1)
    plan = Plan.from_grid(g)
    d = _dev(vel)
    e = torch.empty(0, dtype=torch.float64, device="cuda:0")
    plan.mls_interpolate(0, e, e, e, *d, e, e, e)                       # no markers: no launch
    assert plan.last_launch_count == 0
    with pytest.raises(FseiError) as ex:
        plan.ibm_forcing(10, *_dev(mk), _dev([area])[0], *_dev(V), *d, 1.0, e, e, e, d[0], d[1], d[2])   # f aliases u
    assert ex.value.code == ERR_ARG
    plan.destroy()
