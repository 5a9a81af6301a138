"""Helpers shared by the tests: run the CUDA path / the host stepping harness on a seeded case."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_EMU_SRC = os.path.join(ROOT, "tests", "emu", "emu.cpp")
_EMU_LIB = os.path.join(ROOT, "tests", "emu", "libfsei_emu.so")
_dp = ctypes.POINTER(ctypes.c_double)


def emu_lib():
    """tests/emu/emu.cpp: the device phases of libfsei stepped thread by thread on the host."""
    csrc = os.path.join(ROOT, "paper_2103_15187_b200", "csrc")
    deps = [_EMU_SRC] + [os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith((".cuh", ".hpp"))]
    if not os.path.exists(_EMU_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_EMU_LIB) for d in deps):
        subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wno-unknown-pragmas",
                        _EMU_SRC, "-o", _EMU_LIB], check=True)
    L = ctypes.CDLL(_EMU_LIB)
    i, d = ctypes.c_int, ctypes.c_double
    L.emu_pressure_projection.argtypes = [i, i, i, d, d, _dp, i, i, _dp, _dp, _dp, _dp, _dp, d, d]
    L.emu_poisson_solve.argtypes = [i, i, i, d, d, _dp, i, i, _dp, _dp]
    L.emu_plan_radices.argtypes = [i, ctypes.POINTER(ctypes.c_int)]
    L.emu_plan_check.argtypes = [i, i, i, d, d, _dp, i, i]
    return L


_EMUF_SRC = os.path.join(ROOT, "tests", "emu", "emu_fast.cpp")
_EMUF_LIB = os.path.join(ROOT, "tests", "emu", "libfsei_emu_fast.so")


def emu_fast_lib():
    """tests/emu/emu_fast.cpp: the fast-path kernels of libfsei run on the host (a CTA = a team of host threads)."""
    csrc = os.path.join(ROOT, "paper_2103_15187_b200", "csrc")
    deps = [_EMUF_SRC, os.path.join(ROOT, "tests", "emu", "cuda_shim.hpp")] + \
        [os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith((".cuh", ".hpp"))]
    if not os.path.exists(_EMUF_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_EMUF_LIB) for d in deps):
        subprocess.run(["g++", "-std=c++20", "-O1", "-ffp-contract=off", "-fPIC", "-shared", "-pthread", "-Wno-unknown-pragmas",
                        "-I" + os.path.join(ROOT, "tests", "emu"), _EMUF_SRC, "-o", _EMUF_LIB], check=True)
    L = ctypes.CDLL(_EMUF_LIB)
    i, d = ctypes.c_int, ctypes.c_double
    L.emu_fast_pressure_projection.argtypes = [i, i, i, d, d, _dp, i, i, _dp, _dp, _dp, _dp, _dp, d, d, i]
    L.emu_fast_supported.argtypes = [i, i]
    L.emu_fused_pressure_projection.argtypes = [i, i, i, d, d, _dp, i, i, _dp, _dp, _dp, _dp, _dp, d, d, i]
    L.emu_fused_supported.argtypes = [i, i]
    return L


def emu_fast_projection(case, beta=0.0, split=False, fused=False):
    L = emu_fast_lib()
    u, v, w = case.u.copy(), case.v.copy(), case.w.copy()
    p, phi = np.zeros_like(u), np.empty_like(u)
    zc = np.ascontiguousarray(case.zc)
    fn = L.emu_fused_pressure_projection if fused else L.emu_fast_pressure_projection
    rc = fn(case.nx, case.ny, case.nz, case.Lx, case.Ly, _p(zc), case.bc_x, case.bc_y,
                                        _p(u), _p(v), _p(w), _p(p), _p(phi), case.alpha_dt, beta, int(split))
    assert rc == 0, rc
    return u, v, w, p, phi


def _p(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def emu_projection(case, beta=0.0):
    L = emu_lib()
    u, v, w = case.u.copy(), case.v.copy(), case.w.copy()
    p, phi = np.zeros_like(u), np.empty_like(u)
    zc = np.ascontiguousarray(case.zc)
    rc = L.emu_pressure_projection(case.nx, case.ny, case.nz, case.Lx, case.Ly, _p(zc), case.bc_x, case.bc_y,
                                   _p(u), _p(v), _p(w), _p(p), _p(phi), case.alpha_dt, beta)
    assert rc == 0
    return u, v, w, p, phi


def oracle_projection(orc, case, beta=0.0, p=None):
    u, v, w = case.u.copy(), case.v.copy(), case.w.copy()
    p = np.zeros_like(u) if p is None else p
    phi = orc.pressure_projection(case.grid, u, v, w, p, case.alpha_dt, beta)
    return u, v, w, p, phi


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def op_norm_inf(case):
    """||L||_inf = 4/dx^2 + 4/dy^2 + max_k 2(a_k + c_k)   (SURVEY 8(c) A17 / DESIGN.md R17)."""
    dzc = np.diff(case.zc)
    zm = 0.5 * (case.zc[:-1] + case.zc[1:])
    dzm = np.diff(zm)
    a = np.zeros(case.nz); c = np.zeros(case.nz)
    a[1:] = 1.0 / (dzm * dzc[1:]); c[:-1] = 1.0 / (dzm * dzc[:-1])
    dx, dy = case.Lx / case.nx, case.Ly / case.ny
    return 4 / dx**2 + 4 / dy**2 + 2 * (a + c).max()


def div_gate(case, phi_absmax):
    """R17: max|D u_new| <= max(1e-10, 4 * 2^-52 * ||L||_inf * alpha_dt * ||phi||_inf)."""
    return max(1e-10, 4 * 2.0**-52 * op_norm_inf(case) * abs(case.alpha_dt) * phi_absmax)


# ---- CUDA path -----------------------------------------------------------------------------------
def plan_flags() -> int:
    """Test-only switches, read HERE (the library itself reads no environment variable): FSEI_PATH = generic|fast|fused
    and FSEI_TWIST = 0|1 become flags of fsei_plan_create_ex."""
    from paper_2103_15187_b200 import binding as b
    f = {"generic": b.PATH_GENERIC, "fast": b.PATH_FAST, "fused": b.PATH_FUSED}.get(os.environ.get("FSEI_PATH", ""), 0)
    tw = os.environ.get("FSEI_TWIST")
    if tw is not None:
        f |= b.TWIST_ON if tw == "1" else b.TWIST_OFF
    return f


def make_plan(grid):
    from paper_2103_15187_b200.binding import Plan
    return Plan.from_grid(grid, plan_flags())



def gpu_fields(case):
    import torch
    dev = torch.device("cuda:0")
    return [torch.from_numpy(a).to(dev) for a in (case.u, case.v, case.w)]


def gpu_projection(case, beta=0.0, plan=None, p=None, split=False):
    """Run the CUDA path through the C ABI; returns numpy u, v, w, p, phi."""
    import torch
    from paper_2103_15187_b200.binding import Plan
    own = plan is None
    plan = plan or Plan.from_grid(case.grid, plan_flags())
    u, v, w = gpu_fields(case)
    p = torch.zeros_like(u) if p is None else p
    phi = torch.empty_like(u)
    if split:
        plan.divergence(u, v, w, case.alpha_dt, phi)
        plan.poisson_solve(phi, phi)
        plan.project(u, v, w, p, phi, case.alpha_dt, beta)
    else:
        plan.pressure_projection(u, v, w, p, phi, case.alpha_dt, beta)
    torch.cuda.synchronize()
    out = [t.cpu().numpy() for t in (u, v, w, p, phi)]
    if own:
        plan.destroy()
    return out
