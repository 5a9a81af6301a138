"""Pins for the IB-MLS oracle (oracle/fsei_ibm_oracle.c; Eq. 4) -- -m "not gpu".

The paper gives Eq. 4, the basis [1, x, y, z], "an exponential weight" and the 27-node support; everything else is a
reading (M1..M8).  What the mathematics fixes, independently of the oracle's code:
  * a moving-least-squares fit with a linear basis reproduces every linear field exactly (partition of unity,
    sum phi^k x_k = x_b) -- for each component on ITS staggered nodes, on a stretched z grid;
  * phi = p(x_b)^T A^-1 W_k p(x_k) may be formed in ANY affine parametrisation of the basis: a numpy dense solve in
    global unscaled coordinates must give the same numbers;
  * the spreading is the c_l-scaled transpose of the interpolation and conserves the total force.
"""
import math

import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

P, W = 0, 1


def grid(bc=(P, P), shape=(16, 12, 20), s=2.0, Lx=1.0, Ly=1.5):
    nx, ny, nz = shape
    return (nx, ny, nz, Lx, Ly, inputs.tanh_grid(nz, s), bc[0], bc[1])


def nodes(g, comp):
    """Coordinates of the nodes of component comp (M7), from the staggering definition."""
    nx, ny, nz, Lx, Ly, zc, _, _ = g
    x = (np.arange(nx) + (0 if comp == 0 else 0.5)) * Lx / nx
    y = (np.arange(ny) + (0 if comp == 1 else 0.5)) * Ly / ny
    z = zc[:-1].copy() if comp == 2 else 0.5 * (zc[:-1] + zc[1:])
    return x, y, z


def unravel(g, idx):
    nx, ny = g[0], g[1]
    return idx % nx, (idx // nx) % ny, idx // (nx * ny)


def unwrap(c, cb, L):
    return c - L * np.round((c - cb) / L)


MARKERS = [(0.37, 0.61, 0.45), (0.52, 0.93, 0.30), (0.11, 0.20, 0.71), (0.805, 1.21, 0.52)]


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("mk", MARKERS)
def test_MP1_partition_of_unity_and_linear_reproduction(oracle_ld, comp, mk):
    g = grid()
    idx, phi = oracle_ld.mls_weights(g, comp, *mk)
    i, j, k = unravel(g, idx)
    x, y, z = nodes(g, comp)
    assert abs(phi.sum() - 1) < 1e-14
    assert abs((phi * unwrap(x[i], mk[0], g[3])).sum() - mk[0]) < 1e-14
    assert abs((phi * unwrap(y[j], mk[1], g[4])).sum() - mk[1]) < 1e-14
    assert abs((phi * z[k]).sum() - mk[2]) < 1e-14
    # the support is the 3x3x3 block around the nearest node of this component's own grid
    assert len(set(idx.tolist())) == 27
    assert sorted(set(k.tolist())) == list(range(k.min(), k.min() + 3))
    kc = k.min() + 1
    assert abs(z[kc] - mk[2]) == np.abs(z - mk[2]).min()
    assert np.abs(unwrap(x[i], mk[0], g[3]) - mk[0]).max() <= 1.5 * g[3] / g[0] + 1e-12


@pytest.mark.parametrize("comp", [0, 1, 2])
def test_MP2_phi_vs_numpy_in_global_coordinates(oracle_ld, comp):
    g = grid()
    nx, ny, nz, Lx, Ly, zc, _, _ = g
    for mk in MARKERS:
        idx, phi = oracle_ld.mls_weights(g, comp, *mk)
        i, j, k = unravel(g, idx)
        x, y, z = nodes(g, comp)
        X = np.stack([np.ones(27), unwrap(x[i], mk[0], Lx), unwrap(y[j], mk[1], Ly), z[k]], axis=1)   # p(x_k), GLOBAL coordinates
        kc = np.sort(np.unique(k))[1]
        h = np.array([Lx / nx, Ly / ny, 0.5 * (z[kc + 1] - z[kc - 1])])
        r2 = (((X[:, 1:] - np.array(mk)) / (1.5 * h)) ** 2).sum(axis=1)
        Wt = np.exp(-r2 / 0.3**2)
        A = (X * Wt[:, None]).T @ X
        lam = np.linalg.solve(A, np.array([1.0, *mk]))
        want = Wt * (X @ lam)
        assert np.abs(phi - want).max() < 1e-10          # A is badly scaled in global coordinates: numpy's own error


def test_MP3_linear_field_is_interpolated_exactly(oracle_ld):
    g = grid(bc=(W, P), shape=(12, 16, 24), s=2.5)
    nx, ny, nz = g[:3]
    coef = [(0.3, 1.1, -0.7, 0.4), (-0.2, 0.5, 0.9, -1.3), (0.8, -0.6, 0.2, 0.7)]
    fields = []
    for c in range(3):
        x, y, z = nodes(g, c)
        a, bx, by, bz = coef[c]
        fields.append(np.ascontiguousarray(a + bx * x[None, None, :] + by * y[None, :, None] + bz * z[:, None, None]))
    # markers away from the periodic seam of y and at least 1.5 cells from the x walls (a linear field is not periodic)
    xm, ym, zm, area, V = inputs.sphere_markers(200, (0.5, 0.75, 0.5), 0.22, seed=1)
    out = oracle_ld.mls_interpolate(g, xm, ym, zm, *fields)
    for c in range(3):
        a, bx, by, bz = coef[c]
        assert np.abs(out[c] - (a + bx * xm + by * ym + bz * zm)).max() < 1e-13, c


def test_MP4_spreading_conserves_the_total_force(oracle_ld):
    g = grid(shape=(16, 12, 20))
    nx, ny, nz, Lx, Ly, zc, _, _ = g
    xm, ym, zm, area, V = inputs.sphere_markers(300, (0.5, 0.75, 0.5), 0.3, seed=2)
    rng = np.random.default_rng(5)
    F = [rng.standard_normal(300) for _ in range(3)]
    f = [np.zeros((nz, ny, nx)) for _ in range(3)]
    oracle_ld.mls_spread(g, xm, ym, zm, area, F, f)
    dzc = np.diff(zc); zmid = 0.5 * (zc[:-1] + zc[1:]); dzm = np.r_[0.0, np.diff(zmid)]
    dxdy = (Lx / nx) * (Ly / ny)
    for c in range(3):
        dz = dzm if c == 2 else dzc
        total = (f[c] * dz[:, None, None]).sum() * dxdy
        z = nodes(g, c)[2]
        kc = np.clip(np.abs(z[None, :] - zm[:, None]).argmin(axis=1), 1, nz - 2)
        hl = (Lx / nx + Ly / ny + dz[kc]) / 3
        want = (F[c] * area * hl).sum()
        assert abs(total - want) < 1e-13 * np.abs(F[c] * area * hl).sum(), c


def test_MP5_spreading_is_the_scaled_transpose_of_interpolation(oracle_ld):
    g = grid(shape=(16, 12, 20))
    nx, ny, nz, Lx, Ly, zc, _, _ = g
    n = 150
    xm, ym, zm, area, V = inputs.sphere_markers(n, (0.3, 1.2, 0.55), 0.25, seed=3)      # crosses the periodic seam of y
    rng = np.random.default_rng(6)
    F = [rng.standard_normal(n) for _ in range(3)]
    gf = [rng.standard_normal((nz, ny, nx)) for _ in range(3)]
    f = [np.zeros((nz, ny, nx)) for _ in range(3)]
    oracle_ld.mls_spread(g, xm, ym, zm, area, F, f)
    dzc = np.diff(zc); zmid = 0.5 * (zc[:-1] + zc[1:]); dzm = np.r_[0.0, np.diff(zmid)]
    dxdy = (Lx / nx) * (Ly / ny)
    vol = [np.broadcast_to((dzm if c == 2 else dzc)[:, None, None] * dxdy, (nz, ny, nx)).copy() for c in range(3)]
    Ig = oracle_ld.mls_interpolate(g, xm, ym, zm, *gf)
    Iv = oracle_ld.mls_interpolate(g, xm, ym, zm, *vol)
    for c in range(3):
        dz = dzm if c == 2 else dzc
        z = nodes(g, c)[2]
        kc = np.clip(np.abs(z[None, :] - zm[:, None]).argmin(axis=1), 1, nz - 2)
        cl = area * (Lx / nx + Ly / ny + dz[kc]) / 3 / Iv[c]
        lhs, rhs = (f[c] * gf[c]).sum(), (cl * F[c] * Ig[c]).sum()
        assert abs(lhs - rhs) < 1e-12 * np.abs(cl * F[c] * Ig[c]).sum(), c


def test_MP6_periodic_translation_invariance(oracle_ld):
    g = grid()
    for comp in range(3):
        a = oracle_ld.mls_weights(g, comp, 0.01, 1.49, 0.4)          # support wraps in x and in y
        b = oracle_ld.mls_weights(g, comp, 0.01 + g[3], 1.49 - 2 * g[4], 0.4)
        assert np.array_equal(a[0], b[0]) and np.abs(a[1] - b[1]).max() < 1e-13
        i, j, k = unravel(g, a[0])
        assert set(i.tolist()) == {15, 0, 1}          # nx = 16: the support wraps around the seam
        assert abs(a[1].sum() - 1) < 1e-14


def test_MP7_symmetry_on_a_uniform_grid(oracle_ld):
    nx = ny = nz = 12
    g = (nx, ny, nz, 1.0, 1.0, inputs.tanh_grid(nz, 0.0), P, P)
    x, y, z = nodes(g, 2)
    idx, phi = oracle_ld.mls_weights(g, 2, x[5], y[6], z[4])         # marker ON a w-node
    ph = phi.reshape(3, 3, 3)
    assert np.abs(ph - ph[::-1]).max() < 1e-15 and np.abs(ph - ph[:, ::-1]).max() < 1e-15 and np.abs(ph - ph[:, :, ::-1]).max() < 1e-15
    assert np.abs(ph - ph.transpose(1, 0, 2)).max() < 1e-15          # cubic symmetry (dx = dy = dz)
    assert ph[1, 1, 1] == ph.max() and ph[1, 1, 1] > 0.9              # eps = 0.3: the centre node dominates


def test_MP8_forcing_is_interpolate_then_spread(oracle_ld, oracle_d):
    g = grid(bc=(P, P), shape=(16, 12, 20))
    nx, ny, nz = g[:3]
    xm, ym, zm, area, V = inputs.sphere_markers(120, (0.5, 0.75, 0.5), 0.28, seed=4)
    u, v, w = (inputs.normal_field(50, c, (nz, ny, nx)) for c in range(3))
    inv_dt = 1.0 / 2e-3
    f = [np.zeros((nz, ny, nx)) for _ in range(3)]
    F = oracle_ld.ibm_forcing(g, xm, ym, zm, area, V, u, v, w, inv_dt, f)
    U = oracle_ld.mls_interpolate(g, xm, ym, zm, u, v, w)
    f2 = [np.zeros((nz, ny, nx)) for _ in range(3)]
    for c in range(3):
        assert np.array_equal(F[c], (V[c] - U[c]) * inv_dt)
    oracle_ld.mls_spread(g, xm, ym, zm, area, F, f2)
    for c in range(3):
        assert np.array_equal(f[c], f2[c])
    fd = [np.zeros((nz, ny, nx)) for _ in range(3)]
    oracle_d.ibm_forcing(g, xm, ym, zm, area, V, u, v, w, inv_dt, fd)
    for c in range(3):
        assert np.abs(fd[c] - f[c]).max() <= 1e-12 * np.abs(f[c]).max()
