"""fsei_viscous_step_noalloc (include/fsei.h): the implicit viscous step with its factorisation tables in a static device
array of libfsei, for callers that may not allocate.  Checked against the existing path (fsei_viscous_step) on two calls in
a row that share the array: different beta, then a different grid (shorter and longer lines than the call before, so stale
table entries would show), then a size beyond the limit.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

pytestmark = pytest.mark.gpu
P, W = 0, 1
EPS = 2.0 ** -52


def _case(shape, bc, seed):
    nx, ny, nz = shape
    g = (nx, ny, nz, 1.0, 1.5, inputs.tanh_grid(nz, 2.5), bc[0], bc[1])
    f = [inputs.normal_field(seed, i, (nz, ny, nx)) for i in range(6)]
    f[2][0] = 0
    if bc[0] == W: f[0][:, :, 0] = 0
    if bc[1] == W: f[1][:, 0, :] = 0
    return g, f


def _dev(arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in arrs]


def _check(shape, bc, beta, seed):
    """no-alloc entry against fsei_viscous_step: bit-identical to the generic family (same kernels, same tables), equal to
    rounding to the plan's default family (the tolerance of tests/test_gpu_fluid.py)."""
    import torch
    from paper_2103_15187_b200 import binding
    g, f = _case(shape, bc, seed)
    plan = binding.Plan.from_grid(g)
    pgen = binding.Plan.from_grid(g, binding.VISC_GENERIC)
    a, b, c = _dev(f), _dev(f), _dev(f)
    plan.viscous_step_noalloc(*a, beta)
    assert plan.last_launch_count == 10
    pgen.viscous_step(*b, beta)
    plan.viscous_step(*c, beta)
    torch.cuda.synchronize()
    for k in range(3):
        got, gen, dflt = a[k].cpu().numpy(), b[k].cpu().numpy(), c[k].cpu().numpy()
        assert np.array_equal(got, gen), k
        scale = np.abs(dflt - f[k]).max()
        assert np.abs(got - dflt).max() <= 1e-12 * scale + 2 * EPS * np.abs(dflt).max(), k
    plan.destroy(); pgen.destroy()


def test_noalloc_viscous_step_two_calls_in_a_row_match_existing_path():
    _check((64, 64, 40), (P, P), 3e-4, seed=81)              # fast family is the plan's default here
    _check((64, 64, 40), (P, P), 0.5, seed=82)               # same grid, other beta: the shared tables are rebuilt
    _check((36, 16, 33), (W, W), 2e-3, seed=83)              # shorter lines, walls: stale tails of the longer tables are not read
    _check((128, 48, 70), (P, W), 1e-3 / 6000.0, seed=84)    # longer lines again


def test_noalloc_same_plan_back_to_back_on_one_stream():
    """two calls of ONE plan enqueued with no sync in between (stream order serialises them on the shared array)"""
    import torch
    from paper_2103_15187_b200 import binding
    g, f = _case((48, 24, 20), (P, P), seed=85)
    plan = binding.Plan.from_grid(g)
    pgen = binding.Plan.from_grid(g, binding.VISC_GENERIC)
    a, b = _dev(f), _dev(f)
    for beta in (1e-3, 7e-2):
        plan.viscous_step_noalloc(*a, beta)
        a[3].copy_(a[0]); a[4].copy_(a[1]); a[5].copy_(a[2])         # a new rhs for the second call
    for beta in (1e-3, 7e-2):
        pgen.viscous_step(*b, beta)
        b[3].copy_(b[0]); b[4].copy_(b[1]); b[5].copy_(b[2])
    torch.cuda.synchronize()
    for k in range(3):
        assert torch.equal(a[k], b[k]), k
    plan.destroy(); pgen.destroy()


def test_noalloc_rejects_sizes_beyond_the_static_array_and_bad_arguments():
    import torch
    from paper_2103_15187_b200 import binding
    g = inputs.make_grid(2, shape=(2048, 8, 8))
    plan = binding.Plan.from_grid(g)
    t = [torch.zeros((8, 8, 2048), dtype=torch.float64, device="cuda:0") for _ in range(6)]
    with pytest.raises(binding.FseiError) as e:
        plan.viscous_step_noalloc(*t, 1e-3)
    assert e.value.code == binding.ERR_SIZE and "1024" in str(e.value)
    plan.viscous_step(*t, 1e-3)                                       # the allocating path takes the size
    plan.destroy()
    g = inputs.make_grid(2, shape=(32, 32, 16))
    plan = binding.Plan.from_grid(g)
    t = [torch.zeros((16, 32, 32), dtype=torch.float64, device="cuda:0") for _ in range(6)]
    for call in (lambda: plan.viscous_step_noalloc(t[0], t[1], t[2], t[0], t[4], t[5], 1e-3),
                 lambda: plan.viscous_step_noalloc(*t, -1.0)):
        with pytest.raises(binding.FseiError) as e:
            call()
        assert e.value.code == binding.ERR_ARG
    plan.destroy()
