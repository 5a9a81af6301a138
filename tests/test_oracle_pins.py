"""Pins for the CPU oracle (oracle/fsei_oracle.c) -- run with -m "not gpu".

The paper (arXiv 2103.15187) prints no worked example, equation or number for the pressure
projection (finding 1), so the oracle is pinned to what the mathematics
fixes, each pin built independently of the oracle's own code (numpy dense algebra, closed
forms, O(n^2) definitions).  Pin numbers P1..P13 are those of SURVEY.md sec. 8(c) / DESIGN.md
sec. 5.  A plausible mistake anywhere in the oracle (dropped term, wrong sign or index,
transposed operand, wrong wavenumber/coefficients/gauge) fails at least one of them.
"""
import math

import numpy as np
import pytest

from paper_2103_15187_b200 import inputs

P, N = 0, 1


# ------------------------------------------------------------------------------------------
# independent dense construction of D, G, L = D G from the staggered-grid definitions
# ------------------------------------------------------------------------------------------
def dense_ops(nx, ny, nz, Lx, Ly, zc, bcx, bcy):
    """G: phi -> (gu,gv,gw) on stored faces (wall faces: zero rows); D: (u,v,w) -> div.  Loops only."""
    n = nx * ny * nz
    dx, dy = Lx / nx, Ly / ny
    dzc = np.diff(zc)
    zm = 0.5 * (zc[:-1] + zc[1:])
    idx = lambda i, j, k: (k * ny + j) * nx + i
    Gu, Gv, Gw = np.zeros((n, n)), np.zeros((n, n)), np.zeros((n, n))
    Du, Dv, Dw = np.zeros((n, n)), np.zeros((n, n)), np.zeros((n, n))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                r = idx(i, j, k)
                # gradient on the low faces of cell (i,j,k)
                if i > 0 or bcx == P:
                    Gu[r, r] += 1 / dx; Gu[r, idx((i - 1) % nx, j, k)] -= 1 / dx
                if j > 0 or bcy == P:
                    Gv[r, r] += 1 / dy; Gv[r, idx(i, (j - 1) % ny, k)] -= 1 / dy
                if k > 0:
                    Gw[r, r] += 1 / (zm[k] - zm[k - 1]); Gw[r, idx(i, j, k - 1)] -= 1 / (zm[k] - zm[k - 1])
                # divergence of cell (i,j,k): high face minus low face
                Du[r, r] -= 1 / dx
                if i + 1 < nx: Du[r, idx(i + 1, j, k)] += 1 / dx
                elif bcx == P: Du[r, idx(0, j, k)] += 1 / dx
                Dv[r, r] -= 1 / dy
                if j + 1 < ny: Dv[r, idx(i, j + 1, k)] += 1 / dy
                elif bcy == P: Dv[r, idx(i, 0, k)] += 1 / dy
                Dw[r, r] -= 1 / dzc[k]
                if k + 1 < nz: Dw[r, idx(i, j, k + 1)] += 1 / dzc[k]
    return (Du, Dv, Dw), (Gu, Gv, Gw)


def vol_mean(phi, zc):
    dzc = np.diff(zc)[:, None, None]
    return (phi * dzc).sum() / (dzc.sum() * phi.shape[1] * phi.shape[2])


def small_case(bc, n=8, s=2.0, seed=11, Lx=1.0, Ly=1.5):
    nx, ny, nz = (n, n, n) if isinstance(n, int) else n
    zc = inputs.tanh_grid(nz, s)
    g = (nx, ny, nz, Lx, Ly, zc, bc[0], bc[1])
    u = inputs.normal_field(seed, 0, (nz, ny, nx))
    v = inputs.normal_field(seed, 1, (nz, ny, nx))
    w = inputs.normal_field(seed, 2, (nz, ny, nx))
    w[0] = 0
    if bc[0] == N: u[:, :, 0] = 0
    if bc[1] == N: v[:, 0, :] = 0
    return g, u, v, w


ALL_BC = [(P, P), (N, N), (P, N), (N, P)]


# ------------------------------------------------------------------------------------------
# P11: DFT / DCT against their O(n^2) definitions (reading R15)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 18, 24, 27, 30, 32, 48, 64, 96])
def test_P11_dft_vs_definition(oracle_ld, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    jk = np.outer(np.arange(n), np.arange(n))
    F = np.exp(-2j * np.pi * jk / n)                       # forward: e^{-i...}, unnormalised
    X = oracle_ld.dft(x, -1)
    assert np.allclose(X, F @ x, rtol=0, atol=2e-14 * n)
    xb = oracle_ld.dft(x, +1)                              # inverse carries 1/n
    assert np.allclose(xb, np.conj(F) @ x / n, rtol=0, atol=2e-14)
    assert np.allclose(oracle_ld.dft(X, +1), x, rtol=0, atol=1e-14)   # round trip
    # Parseval and delta <-> constant
    assert abs((abs(X) ** 2).sum() / n - (abs(x) ** 2).sum()) < 1e-12 * n
    d = np.zeros(n, complex); d[0] = 1
    assert np.allclose(oracle_ld.dft(d, -1), np.ones(n), atol=1e-15)


@pytest.mark.parametrize("n", [256, 384, 768, 1024])
def test_P11_dft_long_lengths_vs_numpy(oracle_ld, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert np.allclose(oracle_ld.dft(x, -1), np.fft.fft(x), rtol=0, atol=1e-12)
    assert np.allclose(oracle_ld.dft(x, +1), np.fft.ifft(x), rtol=0, atol=1e-14)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 6, 8, 9, 12, 16, 24, 32, 48, 64, 96])
def test_P11_dct_vs_definition(oracle_ld, n):
    rng = np.random.default_rng(100 + n)
    x = rng.standard_normal(n)
    k = np.arange(n)[:, None]; j = np.arange(n)[None, :]
    C = np.cos(np.pi * k * (j + 0.5) / n)                  # X_k = sum_j x_j cos(pi k (j+1/2)/n)
    X = oracle_ld.dct(x)
    assert np.allclose(X, C @ x, rtol=0, atol=2e-14 * n)
    wgt = np.full(n, 2.0); wgt[0] = 1.0                    # x_j = (X_0 + 2 sum_{k>=1} X_k cos)/n
    xi = oracle_ld.dct(x, inverse=True)
    assert np.allclose(xi, (C.T * wgt) @ x / n, rtol=0, atol=2e-14)
    assert np.allclose(oracle_ld.dct(X, inverse=True), x, rtol=0, atol=1e-14)
    assert np.allclose(oracle_ld.dct(np.ones(n)), np.r_[n, np.zeros(n - 1)], atol=1e-13)


def test_P11_dct_768_roundtrip_and_scipy(oracle_ld):
    import scipy.fft
    x = np.random.default_rng(5).standard_normal(768)
    X = oracle_ld.dct(x)
    assert np.allclose(X, scipy.fft.dct(x, type=2) / 2, rtol=0, atol=1e-12)
    assert np.allclose(oracle_ld.dct(X, inverse=True), x, rtol=0, atol=1e-14)


# ------------------------------------------------------------------------------------------
# P12: Thomas vs dense solve; prefix-sum gauge column vs pinned dense solve; z coefficients
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nz,s", [(8, 2.0), (32, 2.0), (96, 3.0)])
def test_P12_zcoef_and_thomas_vs_dense(oracle_ld, nz, s):
    zc = inputs.tanh_grid(nz, s)
    dzc, dzm, a, c = oracle_ld.zcoef(zc)
    zm = 0.5 * (zc[:-1] + zc[1:])
    assert np.allclose(dzc, np.diff(zc), rtol=1e-12)
    # fp64 cancellation in this reference: eps * z / dz  ~ 1e-12 on the clustered grids
    assert np.allclose(dzm[1:], np.diff(zm), rtol=1e-11)
    assert a[0] == 0 and c[-1] == 0
    assert np.allclose(a[1:], 1 / (np.diff(zm) * dzc[1:]), rtol=1e-11)
    assert np.allclose(c[:-1], 1 / (np.diff(zm) * dzc[:-1]), rtol=1e-11)
    rng = np.random.default_rng(nz)
    for lam in (-0.5, -39.478, -4.0e4):
        b = -(a + c) + lam
        T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
        d = rng.standard_normal(nz)
        x = oracle_ld.thomas(a, b, c, d)
        xd = np.linalg.solve(T, d)
        assert np.linalg.norm(x - xd) <= 1e-11 * np.linalg.norm(xd)
        assert np.linalg.norm(T @ x - d) <= 1e-12 * np.linalg.norm(d) * max(1.0, np.linalg.cond(T) * 1e-4)


def test_P12_thomas_asymmetric_offdiagonals(oracle_ld):
    """a (sub) and c (super) must not be interchangeable."""
    n = 7
    a = np.r_[0.0, np.arange(1, n)] * 0.3
    c = np.r_[np.arange(1, n) * -0.7, 0.0]
    b = np.full(n, 5.0)
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    d = np.arange(1.0, n + 1)
    assert np.allclose(oracle_ld.thomas(a, b, c, d), np.linalg.solve(T, d), rtol=1e-13)


@pytest.mark.parametrize("nz,s", [(8, 2.0), (64, 3.0), (384, 3.0)])
def test_P12_gauge_column_vs_pinned_dense(oracle_ld, nz, s):
    zc = inputs.tanh_grid(nz, s)
    dzc, dzm, a, c = oracle_ld.zcoef(zc)
    rng = np.random.default_rng(nz + 1)
    d = rng.standard_normal(nz)
    d -= (d * dzc).sum() / dzc.sum()                       # compatible: sum d dzc = 0
    x = oracle_ld.gauge_column(zc, d)
    T = np.diag(-(a + c)) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    # residual of the singular system, and the volume-weighted zero-mean gauge (R7)
    assert np.linalg.norm(T @ x - d) <= 1e-9 * np.linalg.norm(d) * (nz / 8)
    assert abs((x * dzc).sum()) <= 1e-14 * (abs(x) * dzc).sum()
    # pinned dense solve in extended precision: replace row 0 by x_0 = 0, then same gauge
    Tp = T.astype(np.longdouble); dp = d.astype(np.longdouble)
    Tp[0, :] = 0; Tp[0, 0] = 1; dp[0] = 0
    if nz <= 64:
        xp = np.linalg.solve(Tp.astype(np.float64), dp.astype(np.float64))
        xp -= (xp * dzc).sum() / dzc.sum()
        assert np.linalg.norm(x - xp) <= 1e-9 * np.linalg.norm(xp)


# ------------------------------------------------------------------------------------------
# modified wavenumbers (R6): formula of B:north_star and eigenvalues of the dense 1-D operators
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,L", [(8, 1.0), (12, 2.0), (32, 0.5)])
def test_modified_wavenumbers(oracle_ld, n, L):
    h = L / n
    k = np.arange(n)
    assert np.allclose(oracle_ld.modified_wavenumbers(n, L, P), (2 * np.cos(2 * np.pi * k / n) - 2) / h**2, rtol=1e-14, atol=1e-12)
    assert np.allclose(oracle_ld.modified_wavenumbers(n, L, N), (2 * np.cos(np.pi * k / n) - 2) / h**2, rtol=1e-14, atol=1e-12)
    # they are the eigenvalues of the periodic / Neumann second-difference matrices
    A = (np.diag(-2.0 * np.ones(n)) + np.diag(np.ones(n - 1), 1) + np.diag(np.ones(n - 1), -1))
    Ap = A.copy(); Ap[0, -1] = Ap[-1, 0] = 1
    An = A.copy(); An[0, 0] = An[-1, -1] = -1
    assert np.allclose(np.sort(np.linalg.eigvalsh(Ap / h**2)), np.sort(oracle_ld.modified_wavenumbers(n, L, P)), atol=1e-9 / h**2)
    assert np.allclose(np.sort(np.linalg.eigvalsh(An / h**2)), np.sort(oracle_ld.modified_wavenumbers(n, L, N)), atol=1e-9 / h**2)


# ------------------------------------------------------------------------------------------
# stencils vs the dense operators: divergence (a1), laplacian = D G, projection (a7)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
def test_stencils_vs_dense(oracle_ld, bc):
    g, u, v, w = small_case(bc, n=(6, 5, 7))
    nx, ny, nz = g[:3]
    (Du, Dv, Dw), (Gu, Gv, Gw) = dense_ops(*g)
    adt = 2.5e-3
    rhs = oracle_ld.divergence(g, u, v, w, adt)
    ref = (Du @ u.ravel() + Dv @ v.ravel() + Dw @ w.ravel()) / adt
    assert np.allclose(rhs.ravel(), ref, rtol=0, atol=1e-12 * abs(ref).max())
    phi = inputs.normal_field(3, 7, (nz, ny, nx))
    Ld = Du @ Gu + Dv @ Gv + Dw @ Gw
    lap = oracle_ld.laplacian(g, phi)
    assert np.allclose(lap.ravel(), Ld @ phi.ravel(), rtol=0, atol=1e-12 * abs(lap).max())
    # projection with beta != 0
    beta = 0.37
    u2, v2, w2, p2 = u.copy(), v.copy(), w.copy(), inputs.normal_field(3, 8, (nz, ny, nx))
    p0 = p2.copy()
    oracle_ld.project(g, u2, v2, w2, p2, phi, adt, beta)
    assert np.allclose(u2.ravel(), u.ravel() - adt * (Gu @ phi.ravel()), atol=1e-13)
    assert np.allclose(v2.ravel(), v.ravel() - adt * (Gv @ phi.ravel()), atol=1e-13)
    assert np.allclose(w2.ravel(), w.ravel() - adt * (Gw @ phi.ravel()), atol=1e-13)
    assert np.allclose(p2.ravel(), p0.ravel() + phi.ravel() - beta * (Ld @ phi.ravel()), atol=1e-10)
    # wall faces untouched
    assert np.array_equal(w2[0], w[0])
    if bc[0] == N: assert np.array_equal(u2[:, :, 0], u[:, :, 0])
    if bc[1] == N: assert np.array_equal(v2[:, 0, :], v[:, 0, :])


# ------------------------------------------------------------------------------------------
# P2: dense brute-force solve of the 7-point staggered Laplacian on 8x8x8
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
def test_P2_dense_bruteforce_8x8x8(oracle_ld, bc):
    g, u, v, w = small_case(bc, n=8, s=2.0, Ly=1.0)
    nx, ny, nz, Lx, Ly, zc = g[:6]
    (Du, Dv, Dw), (Gu, Gv, Gw) = dense_ops(*g)
    Ld = Du @ Gu + Dv @ Gv + Dw @ Gw
    assert np.linalg.matrix_rank(Ld, tol=1e-8 * abs(Ld).max()) == nx * ny * nz - 1
    Wd = np.repeat(np.diff(zc), nx * ny)
    assert abs(Wd[:, None] * Ld - (Wd[:, None] * Ld).T).max() <= 1e-9           # diag(dzc) L symmetric (P10)
    assert abs(Ld.sum(axis=1)).max() <= 1e-9 * abs(Ld).max()                      # constants in the null space
    adt = 1e-3
    rhs = oracle_ld.divergence(g, u, v, w, adt)
    phi = oracle_ld.poisson_solve(g, rhs)
    ref = np.linalg.lstsq(Ld, rhs.ravel(), rcond=None)[0].reshape(rhs.shape)
    ref -= vol_mean(ref, zc)
    assert np.linalg.norm(phi - ref) <= 5e-13 * np.linalg.norm(ref)
    assert abs(vol_mean(phi, zc)) <= 1e-15 * abs(phi).max() * 10                  # P5 gauge


def test_P2_dense_bruteforce_nonsquare_radix3(oracle_ld):
    """nx != ny != nz, a radix-3 length and Lx != Ly: catches transposed axes / swapped lengths."""
    g, u, v, w = small_case((P, N), n=(6, 4, 5), s=1.5, Lx=0.7, Ly=1.3)
    nx, ny, nz, Lx, Ly, zc = g[:6]
    (Du, Dv, Dw), (Gu, Gv, Gw) = dense_ops(*g)
    Ld = Du @ Gu + Dv @ Gv + Dw @ Gw
    rhs = oracle_ld.divergence(g, u, v, w, 1e-2)
    phi = oracle_ld.poisson_solve(g, rhs)
    ref = np.linalg.lstsq(Ld, rhs.ravel(), rcond=None)[0].reshape(rhs.shape)
    ref -= vol_mean(ref, zc)
    assert np.linalg.norm(phi - ref) <= 5e-13 * np.linalg.norm(ref)


# ------------------------------------------------------------------------------------------
# P1: exact discrete eigenfunctions with the modified wavenumbers (uniform z)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,k1,k2,m", [((16, 16, 16), 1, 2, 3), ((32, 24, 12), 5, 0, 1), ((24, 32, 20), 0, 7, 0),
                                           ((32, 32, 16), 16, 16, 15)])
def test_P1_eigenfunction_periodic_uniform(oracle_ld, shape, k1, k2, m):
    nx, ny, nz = shape
    Lx, Ly, Lz = 1.0, 2.0, 1.0
    zc = inputs.tanh_grid(nz, 0.0, Lz)
    g = (nx, ny, nz, Lx, Ly, zc, P, P)
    dx, dy, dz = Lx / nx, Ly / ny, Lz / nz
    x = (np.arange(nx) + 0.5) * dx; y = (np.arange(ny) + 0.5) * dy; kk = np.arange(nz)
    rhs = (np.cos(2 * np.pi * k1 * x / Lx + 0.3)[None, None, :] * np.cos(2 * np.pi * k2 * y / Ly + 1.1)[None, :, None]
           * np.cos(np.pi * m * (kk + 0.5) / nz)[:, None, None])
    lam = ((2 * math.cos(2 * math.pi * k1 / nx) - 2) / dx**2 + (2 * math.cos(2 * math.pi * k2 / ny) - 2) / dy**2
           + (2 * math.cos(math.pi * m / nz) - 2) / dz**2)
    assert lam < 0
    phi = oracle_ld.poisson_solve(g, np.ascontiguousarray(rhs))
    assert np.linalg.norm(phi - rhs / lam) <= 1e-13 * np.linalg.norm(rhs / lam)


def test_P1_eigenfunction_neumann_uniform(oracle_ld):
    nx, ny, nz = 24, 16, 12
    Lx, Ly = 1.5, 1.0
    zc = inputs.tanh_grid(nz, 0.0)
    g = (nx, ny, nz, Lx, Ly, zc, N, N)
    dx, dy, dz = Lx / nx, Ly / ny, 1.0 / nz
    k1, k2, m = 5, 3, 2
    rhs = (np.cos(np.pi * k1 * (np.arange(nx) + 0.5) / nx)[None, None, :] * np.cos(np.pi * k2 * (np.arange(ny) + 0.5) / ny)[None, :, None]
           * np.cos(np.pi * m * (np.arange(nz) + 0.5) / nz)[:, None, None])
    lam = (2 * math.cos(math.pi * k1 / nx) - 2) / dx**2 + (2 * math.cos(math.pi * k2 / ny) - 2) / dy**2 + (2 * math.cos(math.pi * m / nz) - 2) / dz**2
    phi = oracle_ld.poisson_solve(g, np.ascontiguousarray(rhs))
    assert np.linalg.norm(phi - rhs / lam) <= 1e-13 * np.linalg.norm(rhs / lam)


# ------------------------------------------------------------------------------------------
# P3: manufactured solution on stretched grids, P5 gauge, P10 self-adjointness
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc,shape,s", [((P, P), (32, 16, 48), 3.0), ((N, N), (24, 24, 64), 3.0), ((P, N), (16, 12, 32), 2.0),
                                        ((N, P), (12, 16, 32), 2.0), ((P, P), (8, 8, 384), 3.0)])
def test_P3_manufactured_solution(oracle_ld, bc, shape, s):
    nx, ny, nz = shape
    zc = inputs.tanh_grid(nz, s)
    g = (nx, ny, nz, 1.0, 1.0, zc, bc[0], bc[1])
    phi_true = inputs.normal_field(21, 0, (nz, ny, nx))
    phi_true -= vol_mean(phi_true, zc)
    rhs = oracle_ld.laplacian(g, phi_true)
    phi = oracle_ld.poisson_solve(g, rhs)
    assert np.linalg.norm(phi - phi_true) <= 2e-12 * np.linalg.norm(phi_true)
    assert abs(vol_mean(phi, zc)) <= 1e-14 * abs(phi).max()
    psi = inputs.normal_field(21, 1, (nz, ny, nx))
    dzc = np.diff(zc)[:, None, None]
    lhs = (psi * oracle_ld.laplacian(g, phi_true) * dzc).sum(); rhs2 = (oracle_ld.laplacian(g, psi) * phi_true * dzc).sum()
    assert abs(lhs - rhs2) <= 1e-12 * max(abs(lhs), abs(rhs2), 1.0) * 100


# ------------------------------------------------------------------------------------------
# P4/P6/P7/P8/P13: properties of the whole projection
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
def test_P4_P6_projection_divergence_free_and_idempotent(oracle_ld, bc):
    g, u, v, w = small_case(bc, n=(16, 12, 24), s=2.0)
    adt = 1e-3
    p = np.zeros_like(u)
    pre = abs(oracle_ld.divergence(g, u, v, w, 1.0)).max()
    phi1 = oracle_ld.pressure_projection(g, u, v, w, p, adt)
    post = abs(oracle_ld.divergence(g, u, v, w, 1.0)).max()
    assert post <= 1e-13 * pre
    assert np.array_equal(p, phi1)                                    # beta = 0: p += phi
    phi2 = oracle_ld.pressure_projection(g, u, v, w, p, adt)          # P6: projecting again does nothing
    assert np.linalg.norm(phi2) <= 1e-12 * np.linalg.norm(phi1)


def test_P7_pure_gradient_input(oracle_ld):
    nx, ny, nz = 16, 16, 32
    zc = inputs.tanh_grid(nz, 2.0)
    g = (nx, ny, nz, 1.0, 1.0, zc, P, P)
    chi = inputs.normal_field(9, 0, (nz, ny, nx)); chi -= vol_mean(chi, zc)
    u, v, w, p = (np.zeros((nz, ny, nx)) for _ in range(4))
    oracle_ld.project(g, u, v, w, p, chi, -1.0)                       # u = +G chi
    adt = 2e-3
    umax = max(abs(u).max(), abs(v).max(), abs(w).max())
    p[:] = 0
    phi = oracle_ld.pressure_projection(g, u, v, w, p, adt)
    assert max(abs(u).max(), abs(v).max(), abs(w).max()) <= 1e-12 * umax
    assert np.linalg.norm(adt * phi - chi) <= 1e-12 * np.linalg.norm(chi)


def test_P8_solenoidal_input_unchanged(oracle_ld):
    """u* = discrete curl of a vector potential (zero normal component at the walls) has D u* = 0."""
    nx, ny, nz = 16, 12, 20
    Lx, Ly = 1.0, 1.0
    zc = inputs.tanh_grid(nz, 2.0)
    g = (nx, ny, nz, Lx, Ly, zc, P, P)
    dx, dy = Lx / nx, Ly / ny
    dzc = np.diff(zc)
    # stream function psi_y on (x-face, z-face) edges: u = d psi/dz, w = -d psi/dx ; psi = 0 on the walls
    psi = np.zeros((nz + 1, ny, nx)); psi[1:nz] = inputs.normal_field(4, 0, (nz - 1, ny, nx))
    u = (psi[1:] - psi[:-1]) / dzc[:, None, None]
    w = -(np.roll(psi, -1, axis=2) - psi)[:nz] / dx
    # and psi_z on (x-face, y-face) edges: u += -d/dy, v += d/dx
    pz = inputs.normal_field(4, 1, (nz, ny, nx))
    u = u - (np.roll(pz, -1, axis=1) - pz) / dy
    v = (np.roll(pz, -1, axis=2) - pz) / dx
    u, v, w = (np.ascontiguousarray(t) for t in (u, v, w))
    assert abs(w[0]).max() == 0
    rhs = oracle_ld.divergence(g, u, v, w, 1.0)
    scale = max(abs(u).max(), abs(v).max(), abs(w).max()) / min(dx, dy, dzc.min())
    assert abs(rhs).max() <= 1e-14 * scale * 10
    u0, v0, w0 = u.copy(), v.copy(), w.copy()
    p = np.zeros_like(u)
    oracle_ld.pressure_projection(g, u, v, w, p, 1e-3)
    assert max(abs(u - u0).max(), abs(v - v0).max(), abs(w - w0).max()) <= 1e-11 * abs(u0).max()


def test_P9_translation_and_mirror(oracle_ld):
    nx, ny, nz = 16, 8, 12
    zc = inputs.tanh_grid(nz, 2.0)                                    # symmetric about z = 1/2
    g = (nx, ny, nz, 1.0, 1.0, zc, P, P)
    rhs = inputs.normal_field(13, 0, (nz, ny, nx))
    rhs -= vol_mean(rhs, zc)
    phi = oracle_ld.poisson_solve(g, rhs)
    sh = oracle_ld.poisson_solve(g, np.ascontiguousarray(np.roll(np.roll(rhs, 3, axis=2), 5, axis=1)))
    assert np.allclose(sh, np.roll(np.roll(phi, 3, axis=2), 5, axis=1), rtol=0, atol=1e-13 * abs(phi).max())
    mz = oracle_ld.poisson_solve(g, np.ascontiguousarray(rhs[::-1]))
    assert np.allclose(mz, phi[::-1], rtol=0, atol=1e-12 * abs(phi).max())


def test_P13_beta_term(oracle_ld):
    g, u, v, w = small_case((P, P), n=(16, 16, 16), s=2.0)
    adt, beta = 1e-3, 0.25
    rhs = oracle_ld.divergence(g, u, v, w, adt)
    phi = oracle_ld.poisson_solve(g, rhs)
    p = np.zeros_like(u)
    oracle_ld.project(g, u, v, w, p, phi, adt, beta)
    assert np.linalg.norm((p - phi) + beta * rhs) <= 1e-10 * np.linalg.norm(beta * rhs)


# ------------------------------------------------------------------------------------------
# the two flavours of the same source agree; config 1 end to end (values of SURVEY appendix A)
# ------------------------------------------------------------------------------------------
def test_double_and_long_double_builds_agree(oracle_ld, oracle_d):
    assert oracle_ld.mant_bits == 64 and oracle_d.mant_bits == 53
    c = inputs.make_case(1)
    rhs = oracle_ld.divergence(c.grid, c.u, c.v, c.w, c.alpha_dt)
    assert np.array_equal(rhs, oracle_d.divergence(c.grid, c.u, c.v, c.w, c.alpha_dt))   # stencils are double in both
    a, b = oracle_ld.poisson_solve(c.grid, rhs), oracle_d.poisson_solve(c.grid, rhs)
    assert np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(a)


def test_config1_end_to_end(oracle_ld):
    c = inputs.make_case(1)
    u, v, w, p = c.u.copy(), c.v.copy(), c.w.copy(), np.zeros_like(c.u)
    pre = abs(oracle_ld.divergence(c.grid, u, v, w, 1.0)).max()
    phi = oracle_ld.pressure_projection(c.grid, u, v, w, p, c.alpha_dt)
    post = abs(oracle_ld.divergence(c.grid, u, v, w, 1.0)).max()
    assert post <= 1e-10 and post <= 1e-14 * pre * 10                 # B:north_star's absolute gate holds on config 1
    assert abs(vol_mean(phi, c.zc)) <= 1e-15 * abs(phi).max() * 10
    assert np.array_equal(w[0], np.zeros_like(w[0]))
