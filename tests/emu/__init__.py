"""Host emulator of the CUDA kernels (test infrastructure only; see cales_emu.cu)."""
import ctypes as C
import numpy as np

from . import build as _build

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.emu_last_error.restype = C.c_char_p
        L.emu_max_div.restype = C.c_double
        L.emu_cfl_dt.restype = C.c_double
        L.emu_destroy.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


class Emu:
    """Same surface as oracle.Oracle for the calls the parity tests use."""

    def __init__(self, nx, ny, nz, lx, ly, lz, **kw):
        from paper_2411_09364_b200.binding import CalesParams, PARAM_KEYS
        P = CalesParams()
        defaults = dict(nu=1e-3, cs=0.17, aplus=25.0, dsm_avg_xy_plane=1, kappa=0.41, B=5.2, wm_tol=1e-4, wm_maxit=50)
        defaults.update(kw)
        P.nx, P.ny, P.nz, P.lx, P.ly, P.lz = nx, ny, nz, lx, ly, lz
        for k, v in defaults.items():
            assert k in PARAM_KEYS, k
            setattr(P, k, v)
        self._h = C.c_void_p()
        rc = lib().emu_create(C.byref(P), C.byref(self._h))
        if rc:
            raise RuntimeError(lib().emu_last_error().decode())
        self.shape = (nz, ny, nx); self.nx, self.ny, self.nz = nx, ny, nz
        self.per_plane = defaults.get("dsm_avg_xy_plane", 1)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.emu_destroy(self._h); self._h = None

    def set(self, f, a):
        a = np.ascontiguousarray(a, dtype=np.float64); assert a.shape == self.shape
        lib().emu_set_field(self._h, f, _p(a))

    def get(self, f):
        a = np.empty(self.shape); lib().emu_get_field(self._h, f, _p(a)); return a

    def set_velocity(self, u, v, w):
        self.set(0, u); self.set(1, v); self.set(2, w)

    def step(self, dt):
        lib().emu_step(self._h, C.c_double(dt))

    def poisson_solve(self, rhs):
        rhs = np.ascontiguousarray(rhs, dtype=np.float64); phi = np.empty(self.shape)
        lib().emu_poisson_solve(self._h, _p(rhs), _p(phi)); return phi

    def eddy_viscosity(self, u=None, v=None, w=None):
        nut = np.empty(self.shape)
        if u is None:
            lib().emu_eddy_viscosity(self._h, None, None, None, _p(nut))
        else:
            u, v, w = (np.ascontiguousarray(q, dtype=np.float64) for q in (u, v, w))
            lib().emu_eddy_viscosity(self._h, _p(u), _p(v), _p(w), _p(nut))
        return nut

    def wall_stress(self):
        tau = np.empty((2, 2, self.ny, self.nx)); lib().emu_wall_stress(self._h, _p(tau)); return tau

    def wall_stress_y(self):
        tau = np.empty((2, 2, self.nz, self.nx)); lib().emu_wall_stress_y(self._h, _p(tau)); return tau

    def get_cs(self):
        cs = np.empty(self.nz if self.per_plane else self.nz * self.ny); lib().emu_get_cs(self._h, _p(cs)); return cs

    def transform(self, f, direction, inverse=False):
        a = np.ascontiguousarray(f, dtype=np.float64).copy()
        lib().emu_transform(self._h, _p(a), direction, 1 if inverse else 0); return a

    def project(self):
        lib().emu_project(self._h)

    def max_div(self):
        return lib().emu_max_div(self._h)

    def cfl_dt(self, cfl):
        return lib().emu_cfl_dt(self._h, C.c_double(cfl))

    def plane_stats(self):
        out = np.empty((8, self.nz)); lib().emu_plane_stats(self._h, _p(out)); return out
