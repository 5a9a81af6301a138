"""Pins for the fluid-substep oracle (oracle/fsei_fluid_oracle.c): the implicit viscous step (SURVEY 8(f) NEXT-1,
P:L208, Eq. 3) and the explicit terms (NEXT-2) -- run with -m "not gpu".

The paper prints Eq. 3 and names the algorithms (approximate factorisation, Thomas, Sherman-Morrison, second-order
central differences on a staggered mesh) but no discrete formula, so every pin is built independently of the oracle's
code from what the mathematics fixes: dense 1-D operators assembled from the COORDINATES of the staggered positions
(not from the oracle's reciprocal tables), numpy dense solves, closed-form eigenvalues, convergence to the analytic
operator, conservation laws.  Pin numbers V-P*/E-P* are those of DESIGN.md sec. 5.
"""
import math

import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

P, W = 0, 1
ALL_BC = [(P, P), (W, W), (P, W), (W, P)]
U, V, WW = 0, 1, 2


# ------------------------------------------------------------------------------------------
# independent dense 1-D second-difference operators, from the coordinates of the positions
# ------------------------------------------------------------------------------------------
def d2_uniform(n, h, kind):
    """kind: 'periodic' | 'normal' (row 0 is the wall face, value 0 and fixed; not-stored face n is 0) |
    'tangential' (cell centred, no-slip walls half a cell outside: ghost = -first interior)."""
    A = np.zeros((n, n))
    for m in range(n):
        if kind == "normal" and m == 0:
            continue                                   # fixed row
        ext = {}                                       # coefficient of stored unknown s in q_{m-1}, q_m, q_{m+1}
        for off, wgt in ((-1, 1.0), (0, -2.0), (1, 1.0)):
            t = m + off
            sgn = 1.0
            if t < 0 or t >= n:
                if kind == "periodic":
                    t %= n
                elif kind == "normal":
                    continue                           # wall face: value 0
                else:
                    t = 0 if t < 0 else n - 1; sgn = -1.0
            ext[t] = ext.get(t, 0.0) + sgn * wgt
        for t, c in ext.items():
            A[m, t] += c / h**2
    return A


def d2_z_centres(zc):
    """u, v along z: values at cell centres, walls (value 0) at zc[0], zc[nz]; flux form."""
    nz = len(zc) - 1
    zm = 0.5 * (zc[:-1] + zc[1:])
    A = np.zeros((nz, nz))
    for k in range(nz):
        # gradient at face k+1 (above) and face k (below), each as a row over the unknowns
        up, dn = np.zeros(nz), np.zeros(nz)
        if k + 1 < nz:
            up[k + 1] += 1 / (zm[k + 1] - zm[k]); up[k] -= 1 / (zm[k + 1] - zm[k])
        else:
            up[k] -= 1 / (zc[nz] - zm[k])              # (0 - q_k) / half cell
        if k > 0:
            dn[k] += 1 / (zm[k] - zm[k - 1]); dn[k - 1] -= 1 / (zm[k] - zm[k - 1])
        else:
            dn[k] += 1 / (zm[0] - zc[0])
        A[k] = (up - dn) / (zc[k + 1] - zc[k])
    return A


def d2_z_faces(zc):
    """w along z: values at faces zc[0..nz-1] stored (face 0 = wall, fixed), face nz = wall (0, not stored)."""
    nz = len(zc) - 1
    zm = 0.5 * (zc[:-1] + zc[1:])
    A = np.zeros((nz, nz))
    for k in range(1, nz):
        up, dn = np.zeros(nz), np.zeros(nz)            # gradients at cell centres k and k-1
        if k + 1 < nz:
            up[k + 1] += 1 / (zc[k + 1] - zc[k])
        up[k] -= 1 / (zc[k + 1] - zc[k])
        dn[k] += 1 / (zc[k] - zc[k - 1]); dn[k - 1] -= 1 / (zc[k] - zc[k - 1])
        A[k] = (up - dn) / (zm[k] - zm[k - 1])
    A[:, 0] = 0.0                                      # w_0 = 0
    return A


def ops_1d(g, comp):
    """(A_x, A_y, A_z, fixed_x, fixed_y, fixed_z) of component comp."""
    nx, ny, nz, Lx, Ly, zc, bcx, bcy = g
    kx = "periodic" if bcx == P else ("normal" if comp == U else "tangential")
    ky = "periodic" if bcy == P else ("normal" if comp == V else "tangential")
    Ax, Ay = d2_uniform(nx, Lx / nx, kx), d2_uniform(ny, Ly / ny, ky)
    Az = d2_z_faces(zc) if comp == WW else d2_z_centres(zc)
    fx = np.zeros(nx, bool); fy = np.zeros(ny, bool); fz = np.zeros(nz, bool)
    if kx == "normal": fx[0] = True
    if ky == "normal": fy[0] = True
    if comp == WW: fz[0] = True
    return Ax, Ay, Az, fx, fy, fz


def dense_viscous(g, comp, beta, rhs):
    """[(1-b Ax)(1-b Ay)(1-b Az)]^-1 rhs with identity rows / zero right-hand side on the wall faces."""
    Ax, Ay, Az, fx, fy, fz = ops_1d(g, comp)
    out = rhs.copy()
    for axis, (A, fixed) in zip((2, 1, 0), ((Ax, fx), (Ay, fy), (Az, fz))):
        M = np.eye(A.shape[0]) - beta * A
        M[fixed] = 0; M[fixed, fixed] = 1
        out = np.moveaxis(out, axis, 0).copy()
        out[fixed] = 0
        out = np.linalg.solve(M, out.reshape(out.shape[0], -1)).reshape(out.shape)
        out = np.moveaxis(out, 0, axis)
    return out


def small_grid(bc, shape=(6, 5, 7), s=2.0, Lx=1.0, Ly=1.5):
    nx, ny, nz = shape
    return (nx, ny, nz, Lx, Ly, inputs.tanh_grid(nz, s), bc[0], bc[1])


def rand_fields(g, seed, n=3):
    shp = (g[2], g[1], g[0])
    return [inputs.normal_field(seed, s, shp) for s in range(n)]


def zero_walls(g, u, v, w):
    w[0] = 0
    if g[6] == W: u[:, :, 0] = 0
    if g[7] == W: v[:, 0, :] = 0


# ------------------------------------------------------------------------------------------
# V-P1: cyclic Thomas + Sherman-Morrison against a dense solve of the cyclic matrix
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 8, 17, 64, 257])
def test_VP1_cyclic_thomas_vs_dense(oracle_ld, n):
    rng = np.random.default_rng(n)
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)          # asymmetric: a transposed a/c fails
    b = 2.5 + np.abs(a) + np.abs(c) + rng.uniform(0, 1, n)
    d = rng.standard_normal(n)
    A = np.zeros((n, n))
    for k in range(n):
        A[k, k] += b[k]; A[k, (k - 1) % n] += a[k]; A[k, (k + 1) % n] += c[k]
    x = oracle_ld.cyclic_thomas(a, b, c, d)
    assert np.allclose(x, np.linalg.solve(A, d), rtol=0, atol=1e-14 * max(1, np.abs(d).max()))


def test_VP1_cyclic_thomas_constant_coefficients_circulant(oracle_ld):
    """Constant-coefficient periodic operator: the solution is a circular convolution -> numpy FFT closed form."""
    n, r = 48, 7.3
    d = np.random.default_rng(3).standard_normal(n)
    x = oracle_ld.cyclic_thomas(np.full(n, -r), np.full(n, 1 + 2 * r), np.full(n, -r), d)
    sym = 1 + 2 * r - 2 * r * np.cos(2 * np.pi * np.arange(n) / n)
    assert np.allclose(x, np.fft.ifft(np.fft.fft(d) / sym).real, rtol=0, atol=1e-14)


# ------------------------------------------------------------------------------------------
# V-P2: the whole implicit step against the dense Kronecker-factored operator (all bc, all components)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("beta", [1e-3, 0.7])
def test_VP2_viscous_step_vs_dense(oracle_ld, bc, beta):
    g = small_grid(bc)
    u, v, w, ru, rv, rw = rand_fields(g, 21, 6)
    zero_walls(g, u, v, w)
    ref = [q + dense_viscous(g, c, beta, r) for c, (q, r) in enumerate(((u, ru), (v, rv), (w, rw)))]
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, ru, rv, rw, beta)
    for c, (got, want) in enumerate(zip((uo, vo, wo), ref)):
        assert np.abs(got - want).max() <= 2e-13 * np.abs(want).max(), (c, np.abs(got - want).max())
    # wall faces never move
    assert np.array_equal(wo[0], w[0])
    if bc[0] == W: assert np.array_equal(uo[:, :, 0], u[:, :, 0])
    if bc[1] == W: assert np.array_equal(vo[:, 0, :], v[:, 0, :])


def test_VP2_radix_free_sizes(oracle_ld):
    """No size restriction: a 7 x 3 x 5 grid (prime lengths), periodic x, walls in y."""
    g = small_grid((P, W), shape=(7, 3, 5))
    u, v, w, ru, rv, rw = rand_fields(g, 22, 6)
    zero_walls(g, u, v, w)
    ref = [q + dense_viscous(g, c, 0.3, r) for c, (q, r) in enumerate(((u, ru), (v, rv), (w, rw)))]
    oracle_ld.viscous_step(g, u, v, w, ru, rv, rw, 0.3)
    for got, want in zip((u, v, w), ref):
        assert np.abs(got - want).max() <= 2e-13 * np.abs(want).max()


# ------------------------------------------------------------------------------------------
# V-P3: discrete eigenfunctions on a uniform grid: dq = rhs / prod(1 - beta lambda)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("comp", [U, V, WW])
def test_VP3_eigenfunctions_periodic(oracle_ld, comp):
    nx, ny, nz, Lx, Ly = 16, 12, 10, 1.0, 2.0
    zc = inputs.tanh_grid(nz, 0.0)
    g = (nx, ny, nz, Lx, Ly, zc, P, P)
    k1, k2, m, beta = 3, 2, 4, 2e-3
    x = (np.arange(nx) + (0 if comp == U else 0.5)) * Lx / nx
    y = (np.arange(ny) + (0 if comp == V else 0.5)) * Ly / ny
    dz = 1.0 / nz
    if comp == WW:
        z = np.arange(nz) * dz                                   # faces; sin(pi m z) vanishes on both walls
    else:
        z = (np.arange(nz) + 0.5) * dz                           # centres; ghost = -value <=> sin(pi m z)
    f = np.sin(math.pi * m * z)[:, None, None] * np.cos(2 * math.pi * k2 * y / Ly + 0.3)[None, :, None] * \
        np.cos(2 * math.pi * k1 * x / Lx + 0.7)[None, None, :]
    lam = [(2 * math.cos(2 * math.pi * k1 / nx) - 2) / (Lx / nx)**2, (2 * math.cos(2 * math.pi * k2 / ny) - 2) / (Ly / ny)**2,
           (2 * math.cos(math.pi * m / nz) - 2) / dz**2]
    want = f / ((1 - beta * lam[0]) * (1 - beta * lam[1]) * (1 - beta * lam[2]))
    q = [np.zeros_like(f) for _ in range(3)]
    r = [np.zeros_like(f) for _ in range(3)]
    r[comp] = f.copy()
    oracle_ld.viscous_step(g, *q, *r, beta)
    assert np.abs(q[comp] - want).max() <= 1e-14
    for c in range(3):
        if c != comp: assert np.abs(q[c]).max() == 0.0


def test_VP3_eigenfunctions_walls_xy(oracle_ld):
    """Wall-bounded x,y: normal component ~ sin(pi k x/L) on faces, tangential ~ sin(pi k (i+1/2)/n) at centres,
    both with eigenvalue (2 cos(pi k/n) - 2)/h^2."""
    nx, ny, nz = 12, 10, 8
    g = (nx, ny, nz, 1.0, 1.0, inputs.tanh_grid(nz, 0.0), W, W)
    k1, k2, m, beta = 5, 3, 2, 5e-3
    xf, xc = np.arange(nx) / nx, (np.arange(nx) + 0.5) / nx
    yf, yc = np.arange(ny) / ny, (np.arange(ny) + 0.5) / ny
    zf, zcn = np.arange(nz) / nz, (np.arange(nz) + 0.5) / nz
    s = lambda k, t: np.sin(math.pi * k * t)
    lam = (2 * math.cos(math.pi * k1 / nx) - 2) * nx**2, (2 * math.cos(math.pi * k2 / ny) - 2) * ny**2, \
          (2 * math.cos(math.pi * m / nz) - 2) * nz**2
    den = (1 - beta * lam[0]) * (1 - beta * lam[1]) * (1 - beta * lam[2])
    f = [s(m, zcn)[:, None, None] * s(k2, yc)[None, :, None] * s(k1, xf)[None, None, :],
         s(m, zcn)[:, None, None] * s(k2, yf)[None, :, None] * s(k1, xc)[None, None, :],
         s(m, zf)[:, None, None] * s(k2, yc)[None, :, None] * s(k1, xc)[None, None, :]]
    q = [np.zeros_like(f[0]) for _ in range(3)]
    oracle_ld.viscous_step(g, *q, *[np.ascontiguousarray(t) for t in f], beta)
    for c in range(3):
        assert np.abs(q[c] - f[c] / den).max() <= 1e-14, c


# ------------------------------------------------------------------------------------------
# V-P4 / V-P5: beta = 0 is the identity; the three factors commute; double and long double builds agree
# ------------------------------------------------------------------------------------------
def test_VP4_beta_zero_is_identity(oracle_ld):
    g = small_grid((P, P))
    u, v, w, ru, rv, rw = rand_fields(g, 23, 6)
    zero_walls(g, u, v, w)
    rw2 = rw.copy(); rw2[0] = 0
    uo, vo, wo = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, uo, vo, wo, ru, rv, rw, 0.0)
    assert np.abs(uo - (u + ru)).max() <= 2.3e-16 * 8 and np.abs(vo - (v + rv)).max() <= 2.3e-16 * 8
    assert np.abs(wo - (w + rw2)).max() <= 2.3e-16 * 8           # the rhs of the wall face is ignored


@pytest.mark.parametrize("bc", [(P, P), (W, P)])
def test_VP5_sweeps_commute(oracle_ld, bc):
    g = small_grid(bc, shape=(8, 6, 9))
    (f,) = rand_fields(g, 24, 1)
    for comp in (U, V, WW):
        ref = None
        for order in ((0, 1, 2), (2, 1, 0), (1, 2, 0)):
            t = f.copy()
            for d in order:
                t = oracle_ld.viscous_sweep(g, comp, d, 0.4, t)
            if ref is None: ref = t
            assert np.abs(t - ref).max() <= 1e-14


def test_VP5_double_and_long_double_builds_agree(oracle_ld, oracle_d):
    g = inputs.make_grid(2, shape=(16, 12, 64))
    u, v, w, ru, rv, rw = rand_fields(g, 25, 6)
    zero_walls(g, u, v, w)
    a = [t.copy() for t in (u, v, w)]; b = [t.copy() for t in (u, v, w)]
    beta = 1e-3 / (2 * 100.0)                                    # wall cells: beta/dz^2 ~ 1e3
    oracle_ld.viscous_step(g, *a, ru, rv, rw, beta)
    oracle_d.viscous_step(g, *b, ru, rv, rw, beta)
    for x, y in zip(a, b):
        assert np.abs(x - y).max() <= 1e-13 * np.abs(x).max()


# ------------------------------------------------------------------------------------------
# V-P6: implicit rows and explicit Laplacian are the same operator: (A^-1 r - r)/beta -> lap r
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
def test_VP6_implicit_matches_explicit_laplacian(oracle_ld, bc):
    g = small_grid(bc, shape=(8, 6, 9))
    r = rand_fields(g, 26, 3)
    zero_walls(g, *r)
    beta = 1e-9
    q = [np.zeros_like(t) for t in r]
    oracle_ld.viscous_step(g, *q, *r, beta)
    for c in range(3):
        lap = oracle_ld.velocity_laplacian(g, c, r[c])
        got = (q[c] - r[c]) / beta
        assert np.abs(got - lap).max() <= 2e-4 * np.abs(lap).max(), c       # O(beta |lap|^2) + cancellation


# ------------------------------------------------------------------------------------------
# E-P1: explicit velocity Laplacian against the dense operators built from the coordinates
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
def test_EP1_velocity_laplacian_vs_dense(oracle_ld, bc):
    g = small_grid(bc)
    q = rand_fields(g, 31, 3)
    zero_walls(g, *q)
    for c in range(3):
        Ax, Ay, Az, fx, fy, fz = ops_1d(g, c)
        want = np.einsum("ab,kjb->kja", Ax, q[c]) + np.einsum("ab,kbi->kai", Ay, q[c]) + np.einsum("ab,bji->aji", Az, q[c])
        want[fz] = 0; want[:, fy] = 0; want[:, :, fx] = 0
        got = oracle_ld.velocity_laplacian(g, c, q[c])
        assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max(), c


# ------------------------------------------------------------------------------------------
# E-P2: convective term against a ghost-padded numpy construction from the staggering definition
# ------------------------------------------------------------------------------------------
def _pad(q, comp, g):
    """q with one ghost layer on every side, by the boundary conventions (arrays are [z][y][x])."""
    nx, ny, nz, Lx, Ly, zc, bcx, bcy = g
    e = np.zeros((nz + 2, ny + 2, nx + 2))
    e[1:-1, 1:-1, 1:-1] = q
    # x
    if bcx == P: e[:, :, 0] = e[:, :, -2]; e[:, :, -1] = e[:, :, 1]
    elif comp == U: e[:, :, -1] = 0; e[:, :, 0] = np.nan          # face -1 does not exist
    else: e[:, :, 0] = -e[:, :, 1]; e[:, :, -1] = -e[:, :, -2]
    if bcy == P: e[:, 0, :] = e[:, -2, :]; e[:, -1, :] = e[:, 1, :]
    elif comp == V: e[:, -1, :] = 0; e[:, 0, :] = np.nan
    else: e[:, 0, :] = -e[:, 1, :]; e[:, -1, :] = -e[:, -2, :]
    if comp == WW: e[-1] = 0; e[0] = np.nan
    else: e[0] = -e[1]; e[-1] = -e[-2]
    return e


def numpy_convective(g, u, v, w):
    nx, ny, nz, Lx, Ly, zc, bcx, bcy = g
    dx, dy = Lx / nx, Ly / ny
    dzc = np.diff(zc); zm = 0.5 * (zc[:-1] + zc[1:]); dzm = np.r_[np.nan, np.diff(zm)]
    ue, ve, we = _pad(u, U, g), _pad(v, V, g), _pad(w, WW, g)
    C = slice(1, -1)
    sh = lambda e, dk=0, dj=0, di=0: e[1 + dk:e.shape[0] - 1 + dk, 1 + dj:e.shape[1] - 1 + dj, 1 + di:e.shape[2] - 1 + di]
    # --- H_u at (face i, centre j, centre k)
    uc_p = 0.5 * (sh(ue) + sh(ue, di=1)); uc_m = 0.5 * (sh(ue, di=-1) + sh(ue))
    fx = (uc_p**2 - uc_m**2) / dx
    fy_hi = 0.5 * (sh(ue) + sh(ue, dj=1)) * 0.5 * (sh(ve, dj=1, di=-1) + sh(ve, dj=1))
    fy_lo = 0.5 * (sh(ue, dj=-1) + sh(ue)) * 0.5 * (sh(ve, di=-1) + sh(ve))
    if bcy == W: fy_hi[:, -1, :] = 0; fy_lo[:, 0, :] = 0
    fz_hi = 0.5 * (sh(ue) + sh(ue, dk=1)) * 0.5 * (sh(we, dk=1, di=-1) + sh(we, dk=1))
    fz_lo = 0.5 * (sh(ue, dk=-1) + sh(ue)) * 0.5 * (sh(we, di=-1) + sh(we))
    fz_hi[-1] = 0; fz_lo[0] = 0
    hu = -(fx + (fy_hi - fy_lo) / dy + (fz_hi - fz_lo) / dzc[:, None, None])
    if bcx == W: hu[:, :, 0] = 0
    # --- H_v
    vc_p = 0.5 * (sh(ve) + sh(ve, dj=1)); vc_m = 0.5 * (sh(ve, dj=-1) + sh(ve))
    gy = (vc_p**2 - vc_m**2) / dy
    gx_hi = 0.5 * (sh(ve) + sh(ve, di=1)) * 0.5 * (sh(ue, di=1, dj=-1) + sh(ue, di=1))
    gx_lo = 0.5 * (sh(ve, di=-1) + sh(ve)) * 0.5 * (sh(ue, dj=-1) + sh(ue))
    if bcx == W: gx_hi[:, :, -1] = 0; gx_lo[:, :, 0] = 0
    gz_hi = 0.5 * (sh(ve) + sh(ve, dk=1)) * 0.5 * (sh(we, dk=1, dj=-1) + sh(we, dk=1))
    gz_lo = 0.5 * (sh(ve, dk=-1) + sh(ve)) * 0.5 * (sh(we, dj=-1) + sh(we))
    gz_hi[-1] = 0; gz_lo[0] = 0
    hv = -((gx_hi - gx_lo) / dx + gy + (gz_hi - gz_lo) / dzc[:, None, None])
    if bcy == W: hv[:, 0, :] = 0
    # --- H_w at (centre i, centre j, face k)
    wc_p = 0.5 * (sh(we) + sh(we, dk=1)); wc_m = 0.5 * (sh(we, dk=-1) + sh(we))
    hz = (wc_p**2 - wc_m**2) / dzm[:, None, None]
    hx_hi = 0.5 * (sh(we) + sh(we, di=1)) * 0.5 * (sh(ue, di=1, dk=-1) + sh(ue, di=1))
    hx_lo = 0.5 * (sh(we, di=-1) + sh(we)) * 0.5 * (sh(ue, dk=-1) + sh(ue))
    if bcx == W: hx_hi[:, :, -1] = 0; hx_lo[:, :, 0] = 0
    hy_hi = 0.5 * (sh(we) + sh(we, dj=1)) * 0.5 * (sh(ve, dj=1, dk=-1) + sh(ve, dj=1))
    hy_lo = 0.5 * (sh(we, dj=-1) + sh(we)) * 0.5 * (sh(ve, dk=-1) + sh(ve))
    if bcy == W: hy_hi[:, -1, :] = 0; hy_lo[:, 0, :] = 0
    hw = -((hx_hi - hx_lo) / dx + (hy_hi - hy_lo) / dy + hz)
    hw[0] = 0
    return hu, hv, hw


@pytest.mark.parametrize("bc", ALL_BC)
def test_EP2_convective_vs_padded_numpy(oracle_ld, bc):
    g = small_grid(bc, shape=(8, 6, 7))
    u, v, w = rand_fields(g, 32, 3)
    zero_walls(g, u, v, w)
    got = oracle_ld.convective(g, u, v, w)
    want = numpy_convective(g, u, v, w)
    for c in range(3):
        assert not np.isnan(want[c]).any()
        assert np.abs(got[c] - want[c]).max() <= 1e-12 * np.abs(want[c]).max(), c


# ------------------------------------------------------------------------------------------
# E-P3: second-order convergence of H to the analytic -div(u u) on smooth fields (stretched z)
# ------------------------------------------------------------------------------------------
def _analytic_fields(g):
    nx, ny, nz, Lx, Ly, zc, _, _ = g
    zm = 0.5 * (zc[:-1] + zc[1:])
    a, b = 2 * math.pi / Lx, 2 * math.pi / Ly
    X = lambda st: (np.arange(nx) + st) * Lx / nx
    Y = lambda st: (np.arange(ny) + st) * Ly / ny
    fu = lambda x, y, z: np.sin(a * x + 0.3) * np.cos(b * y) * np.sin(math.pi * z) + 0.5
    fv = lambda x, y, z: np.cos(a * x) * np.sin(b * y + 0.2) * np.sin(math.pi * z)
    fw = lambda x, y, z: np.cos(a * x + 0.1) * np.cos(b * y + 0.4) * np.sin(math.pi * z)**2
    mesh = lambda x, y, z: (x[None, None, :], y[None, :, None], z[:, None, None])
    pos = {U: mesh(X(0), Y(.5), zm), V: mesh(X(.5), Y(0), zm), WW: mesh(X(.5), Y(.5), zc[:-1])}
    return (fu, fv, fw), pos, (a, b)


def _analytic_H(fs, pos, comp, ab):
    """-d(q u)/dx - d(q v)/dy - d(q w)/dz at the positions of comp, by high-order (complex-step free) finite
    differences of the ANALYTIC functions with a tiny step -- independent of any grid stencil."""
    fu, fv, fw = fs
    x, y, z = pos[comp]
    q = fs[comp]
    h = 1e-4
    def d(fun, ax):
        e = [0, 0, 0]; e[ax] = h
        return (-fun(x + 2 * e[0], y + 2 * e[1], z + 2 * e[2]) + 8 * fun(x + e[0], y + e[1], z + e[2])
                - 8 * fun(x - e[0], y - e[1], z - e[2]) + fun(x - 2 * e[0], y - 2 * e[1], z - 2 * e[2])) / (12 * h)
    return -(d(lambda *t: q(*t) * fu(*t), 0) + d(lambda *t: q(*t) * fv(*t), 1) + d(lambda *t: q(*t) * fw(*t), 2))


def test_EP3_convective_second_order_convergence(oracle_ld):
    errs = []
    for n in (16, 32, 64):
        g = (n, n, n, 1.0, 2.0, inputs.tanh_grid(n, 1.2), P, P)
        fs, pos, ab = _analytic_fields(g)
        u, v, w = (np.broadcast_to(fs[c](*pos[c]), (n, n, n)).copy() for c in (U, V, WW))
        w[0] = 0
        H = oracle_ld.convective(g, u, v, w)
        e = []
        for c in (U, V, WW):
            want = np.broadcast_to(_analytic_H(fs, pos, c, ab), (n, n, n))
            sl = slice(1, None) if c == WW else slice(None)
            e.append(np.abs(H[c][sl] - want[sl]).max() / np.abs(want).max())
        errs.append(e)
    errs = np.array(errs)
    rate = np.log2(errs[:-1] / errs[1:])
    assert (errs[-1] < 2e-2).all(), errs
    assert (rate[-1] > 1.7).all() and (rate[-1] < 2.4).all(), (errs, rate)


# ------------------------------------------------------------------------------------------
# E-P4 / E-P5: conservation of momentum (any field) and of kinetic energy (solenoidal field, uniform grid)
# ------------------------------------------------------------------------------------------
def test_EP4_momentum_conservation(oracle_ld):
    g = small_grid((P, P), shape=(12, 10, 9), s=2.0)
    u, v, w = rand_fields(g, 33, 3)
    zero_walls(g, u, v, w)
    hu, hv, hw = oracle_ld.convective(g, u, v, w)
    dzc = np.diff(g[5])[:, None, None]
    scale = (np.abs(hu) * dzc).sum()
    assert abs((hu * dzc).sum()) <= 1e-13 * scale and abs((hv * dzc).sum()) <= 1e-13 * scale


@pytest.mark.parametrize("bc", [(P, P), (W, W)])
def test_EP5_energy_conservation_solenoidal_uniform(oracle_ld, bc):
    nx, ny, nz = 12, 10, 8
    g = (nx, ny, nz, 1.0, 1.0, inputs.tanh_grid(nz, 0.0), bc[0], bc[1])
    u, v, w = rand_fields(g, 34, 3)
    zero_walls(g, u, v, w)
    p = np.zeros_like(u)
    oracle_ld.pressure_projection(g, u, v, w, p, 1.0, 0.0)          # discretely solenoidal, walls respected
    assert np.abs(oracle_ld.divergence(g, u, v, w, 1.0)).max() < 1e-12
    hu, hv, hw = oracle_ld.convective(g, u, v, w)
    prod = (u * hu).sum() + (v * hv).sum() + (w * hw).sum()
    scale = np.abs(u * hu).sum() + np.abs(v * hv).sum() + np.abs(w * hw).sum()
    assert abs(prod) <= 1e-12 * scale, prod / scale


# ------------------------------------------------------------------------------------------
# E-P6: assembly of the right-hand side, one term at a time
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P, P), (W, P)])
def test_EP6_rhs_assembly_term_by_term(oracle_ld, bc):
    from tests.test_oracle_pins import dense_ops
    g = small_grid(bc, shape=(6, 4, 5))
    u, v, w, p, h0, h1, h2 = rand_fields(g, 35, 7)
    zero_walls(g, u, v, w)
    zero_walls(g, h0, h1, h2)
    Z = lambda: np.zeros_like(u)
    H = oracle_ld.convective(g, u, v, w)
    # (a) only the convective term: rhs = gdt H, and H is stored
    hh = [Z(), Z(), Z()]
    r = oracle_ld.explicit_terms(g, u, v, w, Z(), *hh, 0.7, 0.0, 0.0, 0.0)
    for c in range(3):
        assert np.allclose(r[c], 0.7 * H[c], rtol=1e-15, atol=0) and np.array_equal(hh[c], H[c])
    # (b) only the previous H: zero velocity, rhs = rdt Hprev, and H becomes 0
    hh = [h0.copy(), h1.copy(), h2.copy()]
    r = oracle_ld.explicit_terms(g, Z(), Z(), Z(), Z(), *hh, 0.9, -0.4, 0.0, 0.0)
    for c, hp in enumerate((h0, h1, h2)):
        assert np.allclose(r[c], -0.4 * hp, rtol=1e-15, atol=0) and np.abs(hh[c]).max() == 0
    # (c) only the pressure gradient: rhs = -adt G p with the projection's own dense G
    _, (Gu, Gv, Gw) = dense_ops(*g)
    r = oracle_ld.explicit_terms(g, Z(), Z(), Z(), p, Z(), Z(), Z(), 0.0, 0.0, 0.3, 0.0)
    for c, G in enumerate((Gu, Gv, Gw)):
        want = -0.3 * (G @ p.ravel()).reshape(p.shape)
        assert np.abs(r[c] - want).max() <= 1e-13 * np.abs(want).max()
    # (d) only the explicit half of Crank-Nicolson: rhs = 2 beta lap q  (convective term switched off by gdt = 0)
    r = oracle_ld.explicit_terms(g, u, v, w, Z(), Z(), Z(), Z(), 0.0, 0.0, 0.0, 0.25)
    for c, q in enumerate((u, v, w)):
        assert np.allclose(r[c], 0.5 * oracle_ld.velocity_laplacian(g, c, q), rtol=1e-15, atol=0)
    # (e) the body force stands outside the [gamma, rho] bracket of Eq. 3: weight alpha dt in the rhs, H unchanged
    f = [h0, h1, h2]
    hh = [Z(), Z(), Z()]
    r = oracle_ld.explicit_terms(g, u, v, w, Z(), *hh, 0.0, 0.0, 0.3, 0.0, f=f)
    for c in range(3):
        assert np.array_equal(hh[c], H[c]) and np.allclose(r[c], 0.3 * f[c], rtol=1e-15, atol=0)


# ------------------------------------------------------------------------------------------
# E-P7: one whole substep (explicit terms -> implicit step -> projection) on a pure shear mode decays by the
# closed-form Crank-Nicolson factor  1 + 2 beta lam / ((1 - beta lam_y)(1 - beta lam_z))
# ------------------------------------------------------------------------------------------
def test_EP7_shear_mode_decay_closed_form(oracle_ld):
    nx, ny, nz = 8, 12, 10
    g = (nx, ny, nz, 1.0, 1.0, inputs.tanh_grid(nz, 0.0), P, P)
    k2, m = 2, 3
    y = (np.arange(ny) + 0.5) / ny; z = (np.arange(nz) + 0.5) / nz
    u = np.broadcast_to(np.sin(math.pi * m * z)[:, None, None] * np.cos(2 * math.pi * k2 * y)[None, :, None],
                        (nz, ny, nx)).copy()
    v, w, p = np.zeros_like(u), np.zeros_like(u), np.zeros_like(u)
    dt, Re = 0.05, 40.0
    beta = dt / (2 * Re)
    h = [np.zeros_like(u) for _ in range(3)]
    r = oracle_ld.explicit_terms(g, u, v, w, p, *h, 1.5 * dt, -0.5 * dt, dt, beta)
    assert np.abs(h[0]).max() <= 1e-15 and np.abs(h[1]).max() == 0 and np.abs(h[2]).max() == 0   # u(y,z) only: no convection
    u1, v1, w1 = u.copy(), v.copy(), w.copy()
    oracle_ld.viscous_step(g, u1, v1, w1, *r, beta)
    oracle_ld.pressure_projection(g, u1, v1, w1, p, dt, beta)
    ly = (2 * math.cos(2 * math.pi * k2 / ny) - 2) * ny**2
    lz = (2 * math.cos(math.pi * m / nz) - 2) * nz**2
    fac = 1 + 2 * beta * (ly + lz) / ((1 - beta * ly) * (1 - beta * lz))
    assert 0 < fac < 1
    assert np.abs(u1 - fac * u).max() <= 1e-14 and np.abs(v1).max() <= 1e-14 and np.abs(w1).max() <= 1e-14
