"""Seeded synthetic inputs for the pressure projection.

A module of its own: it serves the CUDA path's tests/bench AND the oracle's tests, and
holds none of the method's arithmetic -- only the grid recipe (tanh stretching), a
counter-based random stream and smooth-field synthesis.  Everything is generated once on
the host in float64, so both sides see identical bits.

The paper's workloads need its heart geometry (not available); these stand in for its
double-precision, periodic-x,y, wall-normal-z boxes at the shapes of
BASELINE.json's configs.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libfsei_inputs.so")
BC_PERIODIC, BC_NEUMANN = 0, 1
_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> None:
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return
    subprocess.run(["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", _SRC, "-o", _LIB, "-lm"],
                   check=True)


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.fsei_gen_raw.restype = ctypes.c_uint64
        _lib.fsei_gen_raw.argtypes = [ctypes.c_uint64] * 3
        _lib.fsei_gen_normal.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_size_t, ctypes.c_double,
                                         ctypes.c_int, _dp]
        _lib.fsei_gen_separable.argtypes = [ctypes.c_int] * 4 + [_dp] * 5
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


# --------------------------------------------------------------------------------------------
# grid
# --------------------------------------------------------------------------------------------
def tanh_grid(nz: int, s: float, Lz: float = 1.0) -> np.ndarray:
    """z-FACE coordinates zc[0..nz], two-sided tanh clustering (reading R3):
    zc[k] = Lz/2 (1 + tanh(s (2k/nz - 1)) / tanh(s)); s = 0 gives the uniform grid."""
    k = np.arange(nz + 1, dtype=np.float64)
    if s == 0:
        zc = Lz * k / nz
    else:
        zc = Lz * 0.5 * (1.0 + np.tanh(s * (2.0 * k / nz - 1.0)) / math.tanh(s))
    zc[0], zc[-1] = 0.0, Lz
    return zc


# --------------------------------------------------------------------------------------------
# random streams
# --------------------------------------------------------------------------------------------
def normal_field(seed: int, stream: int, shape, sigma: float = 1.0, out: np.ndarray | None = None,
                 accumulate: bool = False) -> np.ndarray:
    """sigma * N(0,1), element idx = linear C-order index, from stream (seed, stream)."""
    if out is None:
        out = np.empty(shape, dtype=np.float64)
        accumulate = False
    assert out.shape == tuple(shape)
    _load().fsei_gen_normal(seed, stream, out.size, float(sigma), int(accumulate), _p(out))
    return out


class _Scalar:
    """Sequential scalar draws from stream (seed, stream) -- for the handful of mode parameters."""

    def __init__(self, seed: int, stream: int):
        self.seed, self.stream, self.n = seed, stream, 0
        self.lib = _load()

    def raw(self) -> int:
        v = int(self.lib.fsei_gen_raw(self.seed, self.stream, self.n))
        self.n += 1
        return v

    def uniform(self) -> float:
        return (self.raw() >> 11) * 2.0 ** -53

    def normal(self) -> float:
        u1 = ((self.raw() >> 11) + 1) * 2.0 ** -53
        u2 = (self.raw() >> 11) * 2.0 ** -53
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def integer(self, lo: int, hi: int) -> int:
        return lo + self.raw() % (hi - lo + 1)


def smooth_field(seed: int, stream: int, comp: str, grid, K: int, M: int = 48, out: np.ndarray | None = None):
    """Band-limited smooth component `comp` in {'u','v','w'} evaluated at ITS staggered position:
    (1/sqrt(M)) sum_m A_m X_m(x) Y_m(y) Z_m(z), integer wavevector 0 < |k| <= K by rejection.
    Periodic direction: cos(2 pi k x/L + theta).  Wall direction: sin(pi k x/L) for the component
    normal to that wall (no penetration), cos(pi k x/L) otherwise.  z is always a wall direction."""
    nx, ny, nz, Lx, Ly, zc, bcx, bcy = grid
    rng = _Scalar(seed, stream)
    dx, dy = Lx / nx, Ly / ny
    x = (np.arange(nx) + (0.0 if comp == "u" else 0.5)) * dx
    y = (np.arange(ny) + (0.0 if comp == "v" else 0.5)) * dy
    z = zc[:-1].copy() if comp == "w" else 0.5 * (zc[:-1] + zc[1:])
    Lz = zc[-1] - zc[0]
    amp = np.empty(M)
    fx, fy, fz = np.empty((M, nx)), np.empty((M, ny)), np.empty((M, nz))
    for m in range(M):
        while True:
            k1, k2, k3 = rng.integer(-K, K), rng.integer(-K, K), rng.integer(-K, K)
            if 0 < k1 * k1 + k2 * k2 + k3 * k3 <= K * K:
                break
        amp[m] = rng.normal() / math.sqrt(M)
        th, ps = 2 * math.pi * rng.uniform(), 2 * math.pi * rng.uniform()
        if bcx == BC_PERIODIC:
            fx[m] = np.cos(2 * math.pi * k1 * x / Lx + th)
        else:
            fx[m] = np.sin(math.pi * k1 * x / Lx) if comp == "u" else np.cos(math.pi * k1 * x / Lx)
        if bcy == BC_PERIODIC:
            fy[m] = np.cos(2 * math.pi * k2 * y / Ly + ps)
        else:
            fy[m] = np.sin(math.pi * k2 * y / Ly) if comp == "v" else np.cos(math.pi * k2 * y / Ly)
        fz[m] = np.sin(math.pi * k3 * (z - zc[0]) / Lz) if comp == "w" else np.cos(math.pi * k3 * (z - zc[0]) / Lz)
    if out is None:
        out = np.empty((nz, ny, nx), dtype=np.float64)
    _load().fsei_gen_separable(nx, ny, nz, M, _p(amp), _p(fx), _p(fy), _p(fz), _p(out))
    return out


# --------------------------------------------------------------------------------------------
# synthetic Lagrangian markers (stand-in for the paper's triangulated wet surfaces)
# --------------------------------------------------------------------------------------------
def sphere_markers(n: int, centre, radius: float, seed: int = 0, omega=(0.3, -0.2, 0.5), vel=(0.1, 0.0, -0.05)):
    """n markers on a sphere (golden-angle spiral, rotated by a seeded phase): positions xm, ym, zm, the area each
    marker stands for (4 pi R^2 / n, the paper's triangle areas) and the velocity of a rigid body (translation `vel` +
    rotation `omega` about the centre) at each marker.  Returns (xm, ym, zm, area, (Vu, Vv, Vw)) as float64 arrays."""
    rng = _Scalar(seed, 900)
    ph0 = 2 * math.pi * rng.uniform()
    l = np.arange(n, dtype=np.float64)
    ct = 1.0 - 2.0 * (l + 0.5) / n
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = ph0 + l * math.pi * (3.0 - math.sqrt(5.0))
    rx, ry, rz = radius * st * np.cos(ph), radius * st * np.sin(ph), radius * ct
    xm, ym, zm = centre[0] + rx, centre[1] + ry, centre[2] + rz
    area = np.full(n, 4.0 * math.pi * radius * radius / n)
    V = (vel[0] + omega[1] * rz - omega[2] * ry, vel[1] + omega[2] * rx - omega[0] * rz, vel[2] + omega[0] * ry - omega[1] * rx)
    return (np.ascontiguousarray(xm), np.ascontiguousarray(ym), np.ascontiguousarray(zm), area,
            tuple(np.ascontiguousarray(t) for t in V))


# --------------------------------------------------------------------------------------------
# BASELINE.json configs (recipe table of DESIGN.md sec. 4)
# --------------------------------------------------------------------------------------------
RK3_ALPHA = (8.0 / 15.0, 2.0 / 15.0, 1.0 / 3.0)      # reading R10

CONFIGS = {
    1: dict(shape=(32, 32, 32), L=(1.0, 1.0, 1.0), s=2.0, bc=(0, 0), kind="white", seed=0, projections=1),
    2: dict(shape=(256, 256, 256), L=(1.0, 1.0, 1.0), s=3.0, bc=(0, 0), kind="smooth+noise", K=16, sigma=1e-3,
            seed=1, projections=1),
    3: dict(shape=(512, 512, 384), L=(2.0, 2.0, 1.0), s=3.0, bc=(0, 0), kind="white", seed=2, projections=3),
    4: dict(shape=(1024, 1024, 768), L=(1.0, 1.0, 1.0), s=3.5, bc=(0, 0), kind="white", seed=3, projections=10),
    5: dict(shape=(768, 768, 1024), L=(1.0, 1.0, 1.0), s=3.0, bc=(1, 1), kind="smooth", K=32, seed=4,
            projections=1),
}


@dataclass
class Case:
    cfg: int
    nx: int
    ny: int
    nz: int
    Lx: float
    Ly: float
    zc: np.ndarray
    bc_x: int
    bc_y: int
    alpha_dt: float
    beta: float
    u: np.ndarray = field(repr=False, default=None)
    v: np.ndarray = field(repr=False, default=None)
    w: np.ndarray = field(repr=False, default=None)

    @property
    def grid(self):
        return (self.nx, self.ny, self.nz, self.Lx, self.Ly, self.zc, self.bc_x, self.bc_y)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


def make_grid(cfg: int, shape=None, bc=None):
    c = CONFIGS[cfg]
    nx, ny, nz = shape if shape is not None else c["shape"]
    bcx, bcy = bc if bc is not None else c["bc"]
    Lx, Ly, Lz = c["L"]
    return (nx, ny, nz, Lx, Ly, tanh_grid(nz, c["s"], Lz), bcx, bcy)


def make_case(cfg: int, shape=None, substep: int = 0, bc=None, out=None, fields: bool = True) -> Case:
    """Inputs of BASELINE.json config `cfg` (1..5); `shape=(nx,ny,nz)` gives the same recipe at other
    extents (parity cases the oracle finishes in seconds).  `out=(u,v,w)` fills caller arrays
    (e.g. pinned host memory).  `substep` selects the independent provisional triple of config 3."""
    c = CONFIGS[cfg]
    grid = make_grid(cfg, shape, bc)
    nx, ny, nz, Lx, Ly, zc, bcx, bcy = grid
    alpha = RK3_ALPHA[substep] if cfg == 3 else 1.0
    case = Case(cfg, nx, ny, nz, Lx, Ly, zc, bcx, bcy, alpha_dt=alpha * 1e-3, beta=0.0)
    if not fields:
        return case
    shp = (nz, ny, nx)
    seed = c["seed"]
    arrs = list(out) if out is not None else [np.empty(shp, dtype=np.float64) for _ in range(3)]
    for ci, comp in enumerate("uvw"):
        a = arrs[ci]
        assert a.shape == shp and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        stream = ci + 3 * substep
        if c["kind"] == "white":
            normal_field(seed, stream, shp, 1.0, out=a)
        else:
            smooth_field(seed, 100 + stream, comp, grid, c["K"], out=a)
            if c["kind"] == "smooth+noise":
                normal_field(seed, stream, shp, c["sigma"], out=a, accumulate=True)
    u, v, w = arrs
    w[0, :, :] = 0.0                       # low z wall: no penetration
    if bcx == BC_NEUMANN:
        u[:, :, 0] = 0.0
    if bcy == BC_NEUMANN:
        v[:, 0, :] = 0.0
    case.u, case.v, case.w = u, v, w
    return case
