"""Thin ctypes binding over the C ABI of libfsei.so (include/fsei.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library.  PyTorch is used by callers for
device memory and streams; this module only needs integer device pointers.  There is no CPU
fallback: if libfsei.so is missing or cannot be loaded, importing `lib()` raises.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

BC_PERIODIC, BC_NEUMANN = 0, 1
OK, ERR_ARG, ERR_SIZE, ERR_GRID, ERR_ALLOC, ERR_CUDA = 0, 1, 2, 3, 4, 5

PATH_GENERIC, PATH_FAST, PATH_FUSED, TWIST_OFF, TWIST_ON, HOST_FIELDS, VISC_GENERIC = 1, 2, 3, 4, 8, 16, 32     # fsei_plan_create_ex flags

EXPORTS = ("fsei_plan_create", "fsei_plan_create_ex", "fsei_plan_kernel_family", "fsei_plan_destroy", "fsei_last_error", "fsei_last_error_code",
           "fsei_plan_workspace_bytes", "fsei_divergence", "fsei_poisson_solve", "fsei_project",
           "fsei_pressure_projection", "fsei_pressure_projection_host", "fsei_plan_last_launch_count",
           "fsei_plan_profile", "fsei_plan_profile_read",
           "fsei_explicit_terms", "fsei_viscous_step", "fsei_viscous_step_noalloc", "fsei_fluid_substep",
           "fsei_mls_interpolate", "fsei_mls_spread", "fsei_ibm_forcing", "fsei_ibm_apply_forcing",
           "fsei_slab_plan_create", "fsei_slab_set_peers", "fsei_slab_forward", "fsei_pencil_solve", "fsei_slab_backward", "fsei_slab_project",
           "fsei_slab_viscous_xy", "fsei_pencil_viscous_z", "fsei_slab_field_add")

_lib = None
_vp, _d, _i = ctypes.c_void_p, ctypes.c_double, ctypes.c_int


class FseiError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libfsei error {code}: {msg}")
        self.code = code


def lib() -> ctypes.CDLL:
    """Load libfsei.so (building it first if nvcc is here and the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.stale():
        try:
            _build.build()
        except RuntimeError as e:  # raised by build._nvcc(): no nvcc on this box -> use the shipped .so if there is one
            if not os.path.exists(path):
                raise RuntimeError(f"libfsei.so is missing and cannot be built ({e}); there is no CPU fallback") from e
        # a compile error (subprocess.CalledProcessError) propagates: never run a stale binary against new sources
    L = ctypes.CDLL(path)
    L.fsei_plan_create.restype = _vp
    L.fsei_plan_create.argtypes = [_i, _i, _i, _d, _d, _vp, _i, _i]
    L.fsei_plan_create_ex.restype = _vp
    L.fsei_plan_create_ex.argtypes = [_i, _i, _i, _d, _d, _vp, _i, _i, ctypes.c_uint]
    L.fsei_plan_kernel_family.restype = _i
    L.fsei_plan_kernel_family.argtypes = [_vp]
    L.fsei_plan_destroy.restype = None
    L.fsei_plan_destroy.argtypes = [_vp]
    L.fsei_last_error.restype = ctypes.c_char_p
    L.fsei_last_error.argtypes = []
    L.fsei_last_error_code.restype = _i
    L.fsei_last_error_code.argtypes = []
    L.fsei_plan_workspace_bytes.restype = ctypes.c_size_t
    L.fsei_plan_workspace_bytes.argtypes = [_vp]
    L.fsei_plan_last_launch_count.restype = _i
    L.fsei_plan_last_launch_count.argtypes = [_vp]
    L.fsei_divergence.restype = _i
    L.fsei_divergence.argtypes = [_vp, _vp, _vp, _vp, _d, _vp, _vp]
    L.fsei_poisson_solve.restype = _i
    L.fsei_poisson_solve.argtypes = [_vp, _vp, _vp, _vp]
    L.fsei_project.restype = _i
    L.fsei_project.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _d, _d, _vp]
    L.fsei_pressure_projection.restype = _i
    L.fsei_pressure_projection.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _d, _d, _vp]
    L.fsei_pressure_projection_host.restype = _i
    L.fsei_pressure_projection_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _d, _d, _vp]
    L.fsei_plan_profile.restype = _i
    L.fsei_plan_profile.argtypes = [_vp, _i]
    L.fsei_plan_profile_read.restype = _i
    L.fsei_plan_profile_read.argtypes = [_vp, _i, ctypes.POINTER(_d), ctypes.POINTER(ctypes.c_long), ctypes.POINTER(ctypes.c_char_p)]
    L.fsei_explicit_terms.restype = _i
    L.fsei_explicit_terms.argtypes = [_vp] * 14 + [_d] * 4 + [_vp]
    L.fsei_viscous_step.restype = _i
    L.fsei_viscous_step.argtypes = [_vp] * 7 + [_d, _vp]
    L.fsei_viscous_step_noalloc.restype = _i
    L.fsei_viscous_step_noalloc.argtypes = [_vp] * 7 + [_d, _vp]
    L.fsei_fluid_substep.restype = _i
    L.fsei_fluid_substep.argtypes = [_vp] * 15 + [_d] * 4 + [_vp]
    L.fsei_mls_interpolate.restype = _i
    L.fsei_mls_interpolate.argtypes = [_vp, ctypes.c_long] + [_vp] * 9 + [_vp]
    L.fsei_mls_spread.restype = _i
    L.fsei_mls_spread.argtypes = [_vp, ctypes.c_long] + [_vp] * 10 + [_vp]
    L.fsei_ibm_forcing.restype = _i
    L.fsei_ibm_forcing.argtypes = [_vp, ctypes.c_long] + [_vp] * 10 + [_d] + [_vp] * 6 + [_vp]
    L.fsei_ibm_apply_forcing.restype = _i
    L.fsei_ibm_apply_forcing.argtypes = [_vp, ctypes.c_long] + [_vp] * 9 + [_d, _vp]
    L.fsei_slab_plan_create.restype = _vp
    L.fsei_slab_plan_create.argtypes = [_i, _i, _i, _d, _d, _vp, _i, _i, _i, _i, _i, _i]
    L.fsei_slab_set_peers.restype = _i
    L.fsei_slab_set_peers.argtypes = [_vp, _i, ctypes.POINTER(_vp), ctypes.POINTER(_vp), ctypes.POINTER(_i), ctypes.POINTER(_i)]
    L.fsei_slab_forward.restype = _i
    L.fsei_slab_forward.argtypes = [_vp, _vp, _vp, _vp, _d, _vp, _vp]
    L.fsei_pencil_solve.restype = _i
    L.fsei_pencil_solve.argtypes = [_vp, _vp, _vp]
    L.fsei_slab_backward.restype = _i
    L.fsei_slab_backward.argtypes = [_vp, _vp, _vp, _vp]
    L.fsei_slab_project.restype = _i
    L.fsei_slab_project.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _d, _d, _vp]
    L.fsei_slab_viscous_xy.restype = _i
    L.fsei_slab_viscous_xy.argtypes = [_vp, _vp, _vp, _vp, _d, _vp]
    L.fsei_pencil_viscous_z.restype = _i
    L.fsei_pencil_viscous_z.argtypes = [_vp, _vp, _i, _d, _vp]
    L.fsei_slab_field_add.restype = _i
    L.fsei_slab_field_add.argtypes = [_vp, _vp, _vp, _vp]
    _lib = L
    return L


def _ptr(t) -> int:
    """Integer address of a torch tensor / numpy array / int."""
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous() and t.element_size() == 8, "fields must be contiguous float64"
        return t.data_ptr()
    assert t.flags["C_CONTIGUOUS"] and t.itemsize == 8
    return t.ctypes.data


def _optr(t):
    return None if t is None else _ptr(t)


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return int(getattr(stream, "cuda_stream", stream))


def last_error() -> str:
    return lib().fsei_last_error().decode()


def _chk(rc: int):
    if rc != OK:
        raise FseiError(rc, last_error())


class Plan:
    """fsei_plan_create(nx, ny, nz, Lx, Ly, zc[], bc_x, bc_y); zc is a host float64 array of nz+1 faces."""

    def __init__(self, nx, ny, nz, Lx, Ly, zc, bc_x=BC_PERIODIC, bc_y=BC_PERIODIC, flags=0):
        import numpy as np
        L = lib()
        zc = np.ascontiguousarray(zc, dtype=np.float64)
        if zc.shape != (nz + 1,):
            raise FseiError(ERR_ARG, f"zc must hold nz+1 = {nz + 1} face coordinates")
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        if flags:
            self._h = L.fsei_plan_create_ex(self.nx, self.ny, self.nz, float(Lx), float(Ly), zc.ctypes.data, int(bc_x), int(bc_y),
                                            int(flags))
        else:
            self._h = L.fsei_plan_create(self.nx, self.ny, self.nz, float(Lx), float(Ly), zc.ctypes.data, int(bc_x), int(bc_y))
        if not self._h:
            raise FseiError(L.fsei_last_error_code(), last_error())

    @classmethod
    def from_grid(cls, grid, flags=0):
        nx, ny, nz, Lx, Ly, zc, bcx, bcy = grid
        return cls(nx, ny, nz, Lx, Ly, zc, bcx, bcy, flags)

    @property
    def kernel_family(self) -> int:
        """0 generic, 1 fast, 2 fused; +4 with the twisted factorisation."""
        return int(lib().fsei_plan_kernel_family(self._h))

    def destroy(self):
        if getattr(self, "_h", None):
            lib().fsei_plan_destroy(self._h)
            self._h = None

    __del__ = destroy

    @property
    def workspace_bytes(self) -> int:
        return int(lib().fsei_plan_workspace_bytes(self._h))

    @property
    def last_launch_count(self) -> int:
        return int(lib().fsei_plan_last_launch_count(self._h))

    def profile(self, enable: bool):
        _chk(lib().fsei_plan_profile(self._h, int(enable)))

    def profile_read(self) -> dict:
        """{kernel name: (summed ms, launches)} since the last read (waits for the recorded events)."""
        n = 32
        ms, cnt, names = (_d * n)(), (ctypes.c_long * n)(), (ctypes.c_char_p * n)()
        k = lib().fsei_plan_profile_read(self._h, n, ms, cnt, names)
        if k < 0:
            raise FseiError(-k, last_error())
        return {names[i].decode(): (float(ms[i]), int(cnt[i])) for i in range(k) if cnt[i] > 0}

    def divergence(self, u, v, w, alpha_dt, rhs, stream=None):
        _chk(lib().fsei_divergence(self._h, _ptr(u), _ptr(v), _ptr(w), float(alpha_dt), _ptr(rhs), _stream(stream)))

    def poisson_solve(self, rhs, phi, stream=None):
        _chk(lib().fsei_poisson_solve(self._h, _ptr(rhs), _ptr(phi), _stream(stream)))

    def project(self, u, v, w, p, phi, alpha_dt, beta=0.0, stream=None):
        _chk(lib().fsei_project(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), _ptr(phi), float(alpha_dt), float(beta),
                                _stream(stream)))

    def pressure_projection(self, u, v, w, p, phi, alpha_dt, beta=0.0, stream=None):
        _chk(lib().fsei_pressure_projection(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), _ptr(phi), float(alpha_dt),
                                            float(beta), _stream(stream)))

    def pressure_projection_host(self, u, v, w, p, alpha_dt, beta=0.0, stream=None):
        """u, v, w, p: HOST float64 arrays/tensors (pinned for speed), updated in place; synchronous."""
        _chk(lib().fsei_pressure_projection_host(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), float(alpha_dt),
                                                 float(beta), _stream(stream)))

    def explicit_terms(self, u, v, w, p, hu, hv, hw, ru, rv, rw, gamma_dt, rho_dt, alpha_dt, beta, f=(None, None, None),
                       stream=None):
        _chk(lib().fsei_explicit_terms(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), *[_optr(t) for t in f], _ptr(hu), _ptr(hv),
                                       _ptr(hw), _ptr(ru), _ptr(rv), _ptr(rw), float(gamma_dt), float(rho_dt), float(alpha_dt),
                                       float(beta), _stream(stream)))

    def viscous_step(self, u, v, w, ru, rv, rw, beta, stream=None):
        _chk(lib().fsei_viscous_step(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(ru), _ptr(rv), _ptr(rw), float(beta),
                                     _stream(stream)))

    def viscous_step_noalloc(self, u, v, w, ru, rv, rw, beta, stream=None):
        _chk(lib().fsei_viscous_step_noalloc(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(ru), _ptr(rv), _ptr(rw), float(beta),
                                             _stream(stream)))

    def fluid_substep(self, u, v, w, p, hu, hv, hw, ru, rv, rw, phi, gamma_dt, rho_dt, alpha_dt, beta, f=(None, None, None),
                      stream=None):
        _chk(lib().fsei_fluid_substep(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), *[_optr(t) for t in f], _ptr(hu), _ptr(hv),
                                      _ptr(hw), _ptr(ru), _ptr(rv), _ptr(rw), _ptr(phi), float(gamma_dt), float(rho_dt),
                                      float(alpha_dt), float(beta), _stream(stream)))

    def mls_interpolate(self, n, xm, ym, zm, u, v, w, ub, vb, wb, stream=None):
        _chk(lib().fsei_mls_interpolate(self._h, int(n), _ptr(xm), _ptr(ym), _ptr(zm), _ptr(u), _ptr(v), _ptr(w), _ptr(ub),
                                        _ptr(vb), _ptr(wb), _stream(stream)))

    def ibm_apply_forcing(self, n, xm, ym, zm, fu, fv, fw, ru, rv, rw, alpha_dt, stream=None):
        _chk(lib().fsei_ibm_apply_forcing(self._h, int(n), _ptr(xm), _ptr(ym), _ptr(zm), _ptr(fu), _ptr(fv), _ptr(fw), _ptr(ru), _ptr(rv),
                                          _ptr(rw), float(alpha_dt), _stream(stream)))

    def mls_spread(self, n, xm, ym, zm, area, Fu, Fv, Fw, fu, fv, fw, stream=None):
        _chk(lib().fsei_mls_spread(self._h, int(n), _ptr(xm), _ptr(ym), _ptr(zm), _ptr(area), _ptr(Fu), _ptr(Fv), _ptr(Fw),
                                   _ptr(fu), _ptr(fv), _ptr(fw), _stream(stream)))

    def ibm_forcing(self, n, xm, ym, zm, area, Vu, Vv, Vw, u, v, w, inv_dt, Fu, Fv, Fw, fu, fv, fw, stream=None):
        _chk(lib().fsei_ibm_forcing(self._h, int(n), _ptr(xm), _ptr(ym), _ptr(zm), _ptr(area), _ptr(Vu), _ptr(Vv), _ptr(Vw),
                                    _ptr(u), _ptr(v), _ptr(w), float(inv_dt), _ptr(Fu), _ptr(Fv), _ptr(Fw), _ptr(fu), _ptr(fv),
                                    _ptr(fw), _stream(stream)))


class SlabPlan(Plan):
    """fsei_slab_plan_create: this rank's share of a multi-GPU projection -- planes [k0, k1) and x-slots [s0, s1)."""

    def __init__(self, grid, k0, k1, s0, s1):
        import numpy as np
        nx, ny, nz, Lx, Ly, zc, bcx, bcy = grid
        L = lib()
        zc = np.ascontiguousarray(zc, dtype=np.float64)
        if zc.shape != (nz + 1,):
            raise FseiError(ERR_ARG, f"zc must hold nz+1 = {nz + 1} face coordinates")
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.k0, self.k1, self.s0, self.s1 = int(k0), int(k1), int(s0), int(s1)
        self.shape = (self.k1 - self.k0, self.ny, self.nx)
        self._h = L.fsei_slab_plan_create(self.nx, self.ny, self.nz, float(Lx), float(Ly), zc.ctypes.data, int(bcx), int(bcy),
                                          self.k0, self.k1, self.s0, self.s1)
        if not self._h:
            raise FseiError(L.fsei_last_error_code(), last_error())

    def set_peers(self, pencils, specs, k0s, s0s):
        """Device addresses (ints) of every rank's pencil and slab spectrum + the range tables; [] switches peers off."""
        n = len(pencils)
        if n == 0:
            _chk(lib().fsei_slab_set_peers(self._h, 0, None, None, None, None))
            return
        pa, sa = (_vp * n)(*[int(x) for x in pencils]), (_vp * n)(*[int(x) for x in specs])
        ka, xa = (_i * (n + 1))(*[int(x) for x in k0s]), (_i * (n + 1))(*[int(x) for x in s0s])
        _chk(lib().fsei_slab_set_peers(self._h, n, pa, sa, ka, xa))

    def slab_forward(self, u, v, w, alpha_dt, spec, stream=None):
        _chk(lib().fsei_slab_forward(self._h, _ptr(u), _ptr(v), _ptr(w), float(alpha_dt), _ptr(spec), _stream(stream)))

    def pencil_solve(self, pencil, stream=None):
        _chk(lib().fsei_pencil_solve(self._h, _ptr(pencil), _stream(stream)))

    def slab_backward(self, spec, phi, stream=None):
        _chk(lib().fsei_slab_backward(self._h, _ptr(spec), _ptr(phi), _stream(stream)))

    def slab_project(self, u, v, w, p, phi, alpha_dt, beta=0.0, stream=None):
        _chk(lib().fsei_slab_project(self._h, _ptr(u), _ptr(v), _ptr(w), _ptr(p), _ptr(phi), float(alpha_dt), float(beta),
                                     _stream(stream)))

    def slab_viscous_xy(self, ru, rv, rw, beta, stream=None):
        _chk(lib().fsei_slab_viscous_xy(self._h, _ptr(ru), _ptr(rv), _ptr(rw), float(beta), _stream(stream)))

    def pencil_viscous_z(self, pencil, comp, beta, stream=None):
        _chk(lib().fsei_pencil_viscous_z(self._h, _ptr(pencil), int(comp), float(beta), _stream(stream)))

    def slab_field_add(self, q, r, stream=None):
        _chk(lib().fsei_slab_field_add(self._h, _ptr(q), _ptr(r), _stream(stream)))
