"""Memory-safety net for the round-2 kernels (compute-sanitizer is closed on this pool): every field lives in a buffer with
guard zones of a NaN bit pattern before and after it.  After each call the guards must be bit-for-bit untouched (no
out-of-bounds write) and every result finite and identical to the run on plain allocations (an out-of-bounds READ of a
guard that reaches the arithmetic shows up as NaN or as a difference) -- ragged and minimal shapes, all boundary mixes, both
viscous families, the slab stages with their halo planes."""
import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

pytestmark = pytest.mark.gpu
P, W = 0, 1
GUARD = 3                      # guard planes on either side of a field


class Guarded:
    """n fields of shape shp inside one buffer: [guard | field 0 | guard | field 1 | ... | guard]."""

    def __init__(self, shp, n, init):
        import torch
        self.shp, self.n = shp, n
        nz, ny, nx = shp
        self.plane = ny * nx
        self.stride = (nz + GUARD) * self.plane
        self.buf = torch.full((GUARD * self.plane + n * self.stride,), float("nan"), dtype=torch.float64, device="cuda:0")
        self.f = []
        for i in range(n):
            o = GUARD * self.plane + i * self.stride
            v = self.buf[o:o + nz * self.plane].view(nz, ny, nx)
            v.copy_(init[i])
            self.f.append(v)

    def guards_intact(self):
        import torch
        nz = self.shp[0]
        ok = bool(torch.isnan(self.buf[:GUARD * self.plane]).all())
        for i in range(self.n):
            o = GUARD * self.plane + i * self.stride + nz * self.plane
            ok = ok and bool(torch.isnan(self.buf[o:o + GUARD * self.plane]).all())
        return ok


def _fields(shape, bc, n, seed=77):
    import torch
    nx, ny, nz = shape
    g = (nx, ny, nz, 1.0, 1.5, inputs.tanh_grid(nz, 2.0), bc[0], bc[1])
    f = [torch.from_numpy(inputs.normal_field(seed, i, (nz, ny, nx))).to("cuda:0") for i in range(n)]
    f[2][0] = 0
    if bc[0] == W: f[0][:, :, 0] = 0
    if bc[1] == W: f[1][:, 0, :] = 0
    return g, f


SHAPES = [((32, 32, 32), (P, P)), ((36, 16, 5), (W, W)), ((48, 24, 7), (P, W)), ((4, 4, 2), (P, P)), ((4, 4, 3), (W, P)),
          ((64, 64, 9), (P, P)), ((128, 96, 4), (P, P)), ((24, 6, 33), (W, P))]


@pytest.mark.parametrize("shape,bc", SHAPES)
@pytest.mark.parametrize("generic", [False, True])
def test_fluid_substep_inside_guards(shape, bc, generic):
    import torch
    from paper_2103_15187_b200 import binding
    g, init = _fields(shape, bc, 14)
    for t in init[3:]:
        t.mul_(0.1)
    init[3].zero_()                                                   # p
    plan = binding.Plan.from_grid(g, binding.VISC_GENERIC if generic else 0)
    G = Guarded(init[0].shape, 14, init)
    plain = [t.clone() for t in init]
    args = dict(gamma_dt=1.5e-3, rho_dt=-0.5e-3, alpha_dt=1e-3, beta=2e-4)
    for F in (G.f, plain):
        u, v, w, p, hu, hv, hw, ru, rv, rw, phi, fu, fv, fw = F
        plan.fluid_substep(u, v, w, p, hu, hv, hw, ru, rv, rw, phi, f=(fu, fv, fw), **args)
    torch.cuda.synchronize()
    assert G.guards_intact()
    for i, (a, b) in enumerate(zip(G.f, plain)):
        if i in (7, 8, 9):
            continue                                                  # ru, rv, rw are scratch (documented)
        assert bool(torch.isfinite(a).all()), i
        assert torch.equal(a, b), i
    plan.destroy()


@pytest.mark.parametrize("shape,bc", [s for s in SHAPES if s[0][2] >= 3])
def test_ib_mls_inside_guards(shape, bc):
    import torch
    from paper_2103_15187_b200.binding import Plan
    g, init = _fields(shape, bc, 6)
    for t in init[3:]:
        t.zero_()
    plan = Plan.from_grid(g)
    n = 257
    xm, ym, zm, area, V = inputs.sphere_markers(n, (0.5, 0.75, 0.5), 0.45, seed=2)      # reaches the walls / seams
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    # marker arrays inside guards as well
    mk = torch.full((9 * (n + 16),), float("nan"), dtype=torch.float64, device="cuda:0")
    views = []
    for i, a in enumerate((xm, ym, zm, area, *V)):
        v = mk[8 + i * (n + 16): 8 + i * (n + 16) + n]; v.copy_(d(a)); views.append(v)
    Fm = torch.full((3 * (n + 16),), float("nan"), dtype=torch.float64, device="cuda:0")
    Fv = [Fm[8 + i * (n + 16): 8 + i * (n + 16) + n] for i in range(3)]
    G = Guarded(init[0].shape, 6, init)
    u, v, w, fu, fv, fw = G.f
    plan.ibm_forcing(n, *views[:4], *views[4:], u, v, w, 250.0, *Fv, fu, fv, fw)
    torch.cuda.synchronize()
    assert G.guards_intact()
    assert int(torch.isnan(Fm).sum()) == 3 * 16                      # only the guard slots are still NaN
    for t in (fu, fv, fw):
        assert bool(torch.isfinite(t).all())
    plan.destroy()


@pytest.mark.parametrize("world", [2, 3])
def test_slab_stages_inside_guards(world):
    """The slab stages read exactly one halo plane beyond their slab and nothing else."""
    import torch
    from paper_2103_15187_b200 import slab
    case = inputs.make_case(2, shape=(64, 32, 24))
    ranks = [slab.SlabProjection(case.grid, r, world) for r in range(world)]
    for r in ranks:
        r.load(case.u, case.v, case.w)
        # poison what a stage must never read: the halo plane of w above the top wall, the phi halos beyond the walls
        if r.x.k1 == r.x.nz:
            r.x.w_ext[r.x.nzl].fill_(float("nan"))
        r.x.phi_ext[0].fill_(float("nan")); r.x.phi_ext[r.x.nzl + 1].fill_(float("nan"))
    slab.project_local(ranks, case.alpha_dt, 0.0)                     # beta = 0: the upper phi halo is never exchanged nor read
    torch.cuda.synchronize()
    for r in ranks:
        for t in (r.u, r.v, r.w, r.p, r.phi):
            assert bool(torch.isfinite(t).all())
        r.destroy()


def test_slab_viscous_calls_reject_bad_arguments():
    import torch
    from paper_2103_15187_b200 import inputs
    from paper_2103_15187_b200.binding import FseiError, ERR_ARG, SlabPlan
    from tests.util import make_plan
    g = inputs.make_grid(2, shape=(32, 32, 16))
    sp = SlabPlan(g, 0, 8, 0, 8)
    a, b, c = (torch.zeros((8, 32, 32), dtype=torch.float64, device="cuda") for _ in range(3))
    pencil = torch.zeros((16, 32, 16), dtype=torch.float64, device="cuda")
    for call in (lambda: sp.slab_viscous_xy(a, a, c, 1e-3), lambda: sp.slab_viscous_xy(a, b, c, -1.0),
                 lambda: sp.pencil_viscous_z(pencil, 3, 1e-3), lambda: sp.pencil_viscous_z(pencil, 0, float("inf")),
                 lambda: sp.slab_field_add(a, a)):
        with pytest.raises(FseiError) as e:
            call()
        assert e.value.code == ERR_ARG
    sp.destroy()
    plan = make_plan(g)                                          # a whole-grid plan has no slab stages
    with pytest.raises(FseiError) as e:
        plan_call = SlabPlan.slab_viscous_xy
        plan_call(plan, a, b, c, 1e-3)
    assert e.value.code == ERR_ARG
    plan.destroy()
