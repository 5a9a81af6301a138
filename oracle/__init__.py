"""CPU oracle for the pressure projection -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It builds and loads oracle/fsei_oracle.c (plain C,
its own DFT/DCT/Thomas) in two flavours of the same source:

  kind="ld"  real_t = long double (x87 80-bit): the parity reference
  kind="d"   real_t = double: the timed CPU baseline

It shares nothing with paper_2103_15187_b200/ except the seeded input generators
(paper_2103_15187_b200_inputs), which hold none of the method's arithmetic.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fsei_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "fsei_fluid_oracle.c"),    # projection; viscous step + explicit terms;
         os.path.join(_HERE, "fsei_ibm_oracle.c")]            # IB-MLS transfer operators
BC_PERIODIC, BC_NEUMANN = 0, 1

_dp = ctypes.POINTER(ctypes.c_double)


def lib_path(kind: str) -> str:
    return os.path.join(_HERE, f"liboracle_{kind}.so")


def build(force: bool = False) -> None:
    """gcc -O2 -ffp-contract=off -fopenmp, once per flavour (rebuilt when the source is newer)."""
    for kind, defs in (("ld", ["-DORACLE_LONG_DOUBLE"]), ("d", [])):
        out = lib_path(kind)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= max(os.path.getmtime(f) for f in _SRCS):
            continue
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", *defs, *_SRCS, "-o", out, "-lm"]
        subprocess.run(cmd, check=True)


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"], "oracle wants contiguous float64"
    return a.ctypes.data_as(_dp)


class Oracle:
    """Thin ctypes view of one flavour of the oracle library."""

    def __init__(self, kind: str = "ld"):
        build()
        self.kind = kind
        self.lib = ctypes.CDLL(lib_path(kind))
        self.mant_bits = int(self.lib.oracle_real_mant_bits())
        L = self.lib
        i, d = ctypes.c_int, ctypes.c_double
        grid = [i, i, i, d, d, _dp, i, i]
        L.oracle_divergence.argtypes = grid + [_dp, _dp, _dp, d, _dp]
        L.oracle_laplacian.argtypes = grid + [_dp, _dp]
        L.oracle_project.argtypes = grid + [_dp, _dp, _dp, _dp, _dp, d, d]
        L.oracle_poisson_solve.argtypes = grid + [_dp, _dp]
        L.oracle_pressure_projection.argtypes = grid + [_dp, _dp, _dp, _dp, _dp, d, d]
        L.oracle_dft.argtypes = [i, i, _dp, _dp, _dp, _dp]
        L.oracle_dct.argtypes = [i, i, _dp, _dp]
        L.oracle_thomas.argtypes = [i, _dp, _dp, _dp, _dp, _dp]
        L.oracle_zcoef.argtypes = [i, _dp, _dp, _dp, _dp, _dp]
        L.oracle_gauge_column.argtypes = [i, _dp, _dp, _dp]
        L.oracle_modified_wavenumbers.argtypes = [i, d, i, _dp]
        # fsei_fluid_oracle.c: implicit viscous step (NEXT-1) and explicit terms (NEXT-2)
        L.oracle_viscous_step.argtypes = grid + [_dp] * 6 + [d]
        L.oracle_viscous_sweep.argtypes = grid + [i, i, d, _dp]
        L.oracle_cyclic_thomas.argtypes = [i, _dp, _dp, _dp, _dp, _dp]
        L.oracle_convective.argtypes = grid + [_dp] * 3 + [_dp] * 3
        L.oracle_velocity_laplacian.argtypes = grid + [i, _dp, _dp]
        L.oracle_explicit_terms.argtypes = grid + [_dp] * 4 + [ctypes.c_void_p] * 3 + [_dp] * 6 + [d, d, d, d]

    # -- grid tuple helper: g = (nx, ny, nz, Lx, Ly, zc, bc_x, bc_y) ------------------------
    @staticmethod
    def _g(g):
        nx, ny, nz, Lx, Ly, zc, bcx, bcy = g
        zc = np.ascontiguousarray(zc, dtype=np.float64)
        assert zc.shape == (nz + 1,)
        return (int(nx), int(ny), int(nz), float(Lx), float(Ly), _ptr(zc), int(bcx), int(bcy)), zc

    @staticmethod
    def _chk(rc, what):
        if rc != 0:
            raise RuntimeError(f"oracle {what} failed with code {rc}")

    def divergence(self, g, u, v, w, alpha_dt):
        a, keep = self._g(g)
        rhs = np.empty_like(u)
        self._chk(self.lib.oracle_divergence(*a, _ptr(u), _ptr(v), _ptr(w), float(alpha_dt), _ptr(rhs)), "divergence")
        return rhs

    def laplacian(self, g, phi):
        a, keep = self._g(g)
        out = np.empty_like(phi)
        self._chk(self.lib.oracle_laplacian(*a, _ptr(phi), _ptr(out)), "laplacian")
        return out

    def poisson_solve(self, g, rhs):
        a, keep = self._g(g)
        phi = np.empty_like(rhs)
        self._chk(self.lib.oracle_poisson_solve(*a, _ptr(rhs), _ptr(phi)), "poisson_solve")
        return phi

    def project(self, g, u, v, w, p, phi, alpha_dt, beta=0.0):
        """In place on u, v, w, p."""
        a, keep = self._g(g)
        self._chk(self.lib.oracle_project(*a, _ptr(u), _ptr(v), _ptr(w), _ptr(p), _ptr(phi),
                                          float(alpha_dt), float(beta)), "project")

    def pressure_projection(self, g, u, v, w, p, alpha_dt, beta=0.0):
        """In place on u, v, w, p; returns phi."""
        a, keep = self._g(g)
        phi = np.empty_like(u)
        self._chk(self.lib.oracle_pressure_projection(*a, _ptr(u), _ptr(v), _ptr(w), _ptr(p), _ptr(phi),
                                                      float(alpha_dt), float(beta)), "pressure_projection")
        return phi

    # -- fluid substep: explicit terms, implicit viscous step ----------------------------------
    def viscous_step(self, g, u, v, w, ru, rv, rw, beta):
        """In place on u, v, w: q += [(1-b dxx)(1-b dyy)(1-b dzz)]^-1 rhs_q."""
        a, keep = self._g(g)
        self._chk(self.lib.oracle_viscous_step(*a, _ptr(u), _ptr(v), _ptr(w), _ptr(ru), _ptr(rv), _ptr(rw),
                                               float(beta)), "viscous_step")

    def viscous_sweep(self, g, comp, direction, beta, f):
        """Returns [(1 - beta d2_dir)]^-1 f for component comp (0,1,2 = u,v,w), direction 0,1,2 = x,y,z."""
        a, keep = self._g(g)
        out = np.ascontiguousarray(f, dtype=np.float64).copy()
        self._chk(self.lib.oracle_viscous_sweep(*a, int(comp), int(direction), float(beta), _ptr(out)), "viscous_sweep")
        return out

    def cyclic_thomas(self, a, b, c, d):
        a, b, c, d = (np.ascontiguousarray(t, dtype=np.float64) for t in (a, b, c, d))
        x = np.empty_like(d)
        self.lib.oracle_cyclic_thomas(d.shape[0], _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x))
        return x

    @staticmethod
    def _opt(a):
        return None if a is None else a.ctypes.data

    def convective(self, g, u, v, w):
        """H = -div(uu): returns hu, hv, hw."""
        a, keep = self._g(g)
        h = [np.empty_like(u) for _ in range(3)]
        self._chk(self.lib.oracle_convective(*a, _ptr(u), _ptr(v), _ptr(w), *[_ptr(x) for x in h]), "convective")
        return h

    def velocity_laplacian(self, g, comp, q):
        a, keep = self._g(g)
        out = np.empty_like(q)
        self._chk(self.lib.oracle_velocity_laplacian(*a, int(comp), _ptr(q), _ptr(out)), "velocity_laplacian")
        return out

    def explicit_terms(self, g, u, v, w, p, hu, hv, hw, gamma_dt, rho_dt, alpha_dt, beta, f=(None, None, None)):
        """hu, hv, hw: H^{n-1} in, H^n out (in place).  Returns ru, rv, rw."""
        a, keep = self._g(g)
        r = [np.empty_like(u) for _ in range(3)]
        self._chk(self.lib.oracle_explicit_terms(*a, _ptr(u), _ptr(v), _ptr(w), _ptr(p), *[self._opt(x) for x in f],
                                                 _ptr(hu), _ptr(hv), _ptr(hw), *[_ptr(x) for x in r],
                                                 float(gamma_dt), float(rho_dt), float(alpha_dt), float(beta)),
                  "explicit_terms")
        return r

    # -- IB-MLS transfer operators (fsei_ibm_oracle.c) --------------------------------------------
    def mls_weights(self, g, comp, xb, yb, zb):
        """(idx[27], phi[27]) of one marker for component comp."""
        a, keep = self._g(g)
        idx = np.empty(27, dtype=np.int64); phi = np.empty(27)
        self.lib.oracle_mls_weights.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 2 + [_dp] + [ctypes.c_int] * 3 + \
            [ctypes.c_double] * 3 + [ctypes.c_void_p, _dp]
        self._chk(self.lib.oracle_mls_weights(*a, int(comp), float(xb), float(yb), float(zb), idx.ctypes.data, _ptr(phi)), "mls_weights")
        return idx, phi

    def _markers(self, xm, ym, zm):
        m = [np.ascontiguousarray(t, dtype=np.float64) for t in (xm, ym, zm)]
        return m, ctypes.c_long(m[0].shape[0])

    def mls_interpolate(self, g, xm, ym, zm, u, v, w):
        a, keep = self._g(g)
        m, n = self._markers(xm, ym, zm)
        out = [np.empty(n.value) for _ in range(3)]
        self.lib.oracle_mls_interpolate.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 2 + [_dp] + [ctypes.c_int] * 2 + \
            [ctypes.c_long] + [_dp] * 9
        self._chk(self.lib.oracle_mls_interpolate(*a, n, *[_ptr(t) for t in m], _ptr(u), _ptr(v), _ptr(w), *[_ptr(t) for t in out]),
                  "mls_interpolate")
        return out

    def mls_spread(self, g, xm, ym, zm, area, F, f):
        """f (3 fields) += spread of the marker forces F (3 arrays), in place."""
        a, keep = self._g(g)
        m, n = self._markers(xm, ym, zm)
        area = np.ascontiguousarray(area, dtype=np.float64)
        self.lib.oracle_mls_spread.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 2 + [_dp] + [ctypes.c_int] * 2 + \
            [ctypes.c_long] + [_dp] * 10
        self._chk(self.lib.oracle_mls_spread(*a, n, *[_ptr(t) for t in m], _ptr(area), *[_ptr(np.ascontiguousarray(t)) for t in F],
                                             *[_ptr(t) for t in f]), "mls_spread")

    def ibm_forcing(self, g, xm, ym, zm, area, V, u, v, w, inv_dt, f):
        """f (3 fields) += IB forcing; returns the marker forces F (3 arrays)."""
        a, keep = self._g(g)
        m, n = self._markers(xm, ym, zm)
        area = np.ascontiguousarray(area, dtype=np.float64)
        F = [np.empty(n.value) for _ in range(3)]
        self.lib.oracle_ibm_forcing.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 2 + [_dp] + [ctypes.c_int] * 2 + \
            [ctypes.c_long] + [_dp] * 10 + [ctypes.c_double] + [_dp] * 6
        self._chk(self.lib.oracle_ibm_forcing(*a, n, *[_ptr(t) for t in m], _ptr(area), *[_ptr(np.ascontiguousarray(t)) for t in V],
                                              _ptr(u), _ptr(v), _ptr(w), float(inv_dt), *[_ptr(t) for t in F], *[_ptr(t) for t in f]),
                  "ibm_forcing")
        return F

    # -- building blocks ---------------------------------------------------------------------
    def dft(self, x: np.ndarray, sign: int) -> np.ndarray:
        x = np.asarray(x, dtype=np.complex128)
        n = x.shape[0]
        xr, xi = np.ascontiguousarray(x.real), np.ascontiguousarray(x.imag)
        yr, yi = np.empty(n), np.empty(n)
        self.lib.oracle_dft(n, int(sign), _ptr(xr), _ptr(xi), _ptr(yr), _ptr(yi))
        return yr + 1j * yi

    def dct(self, x: np.ndarray, inverse: bool = False) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.empty_like(x)
        self.lib.oracle_dct(x.shape[0], int(inverse), _ptr(x), _ptr(y))
        return y

    def thomas(self, a, b, c, d):
        a, b, c, d = (np.ascontiguousarray(t, dtype=np.float64) for t in (a, b, c, d))
        x = np.empty_like(d)
        self.lib.oracle_thomas(d.shape[0], _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x))
        return x

    def zcoef(self, zc):
        zc = np.ascontiguousarray(zc, dtype=np.float64)
        nz = zc.shape[0] - 1
        out = [np.empty(nz) for _ in range(4)]
        self.lib.oracle_zcoef(nz, _ptr(zc), *[_ptr(o) for o in out])
        return tuple(out)  # dzc, dzm, a, c

    def gauge_column(self, zc, d):
        zc = np.ascontiguousarray(zc, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        x = np.empty_like(d)
        self.lib.oracle_gauge_column(d.shape[0], _ptr(zc), _ptr(d), _ptr(x))
        return x

    def modified_wavenumbers(self, n, L, bc):
        lam = np.empty(n)
        self.lib.oracle_modified_wavenumbers(int(n), float(L), int(bc), _ptr(lam))
        return lam
