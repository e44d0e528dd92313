"""Thin ctypes binding of libcales.so (include/cales.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used only for device memory
(the workspace blob and I/O tensors) and for the CUDA stream.  There is no CPU fallback: importing this
module builds/loads libcales.so and raises if that fails; constructing a Solver raises without a CUDA device.
"""
import ctypes as C

from . import build as _build

_dp = C.POINTER(C.c_double)


class CalesParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
        ("zstretch", C.c_int), ("zstretch_factor", C.c_double), ("zf_user", _dp),
        ("bc_y", C.c_int), ("bc_z", C.c_int),
        ("nu", C.c_double),
        ("sgs_model", C.c_int), ("cs", C.c_double), ("van_driest", C.c_int), ("aplus", C.c_double),
        ("dsm_avg_xy_plane", C.c_int), ("dsm_clip_total", C.c_int), ("dsm_alpha2d", C.c_double),
        ("wall_model", C.c_int), ("kappa", C.c_double), ("B", C.c_double), ("h_wm", C.c_double),
        ("wm_tol", C.c_double), ("wm_maxit", C.c_int),
        ("implicit_z", C.c_int),
        ("const_flow_rate", C.c_int), ("u_bulk", C.c_double),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("cuda_stream", C.c_void_p), ("device", C.c_int),
        ("wall_model_y", C.c_int), ("dsm_filter3d", C.c_int), ("implicit_xyz", C.c_int),
    ]


class CalesDiag(C.Structure):
    _fields_ = [("max_div", C.c_double), ("u_bulk", C.c_double), ("kinetic_energy", C.c_double), ("forcing", C.c_double),
                ("wm_max_iters", C.c_int), ("nan_count", C.c_int),
                ("ms_rhs", C.c_double), ("ms_implicit", C.c_double), ("ms_solver", C.c_double),
                ("ms_correction", C.c_double), ("ms_sgs", C.c_double), ("ms_wall", C.c_double)]


# every symbol include/cales.h declares
SYMBOLS = ["cales_default_params", "cales_workspace_bytes", "cales_create", "cales_create_basic", "cales_destroy",
           "cales_set_field", "cales_get_field", "cales_step", "cales_step_adaptive", "cales_last_dt", "cales_poisson_solve", "cales_eddy_viscosity",
           "cales_wall_stress", "cales_wall_stress_y", "cales_project", "cales_cfl_dt", "cales_cfl_dt_static", "cales_plane_stats", "cales_stats_reset", "cales_stats_accumulate", "cales_stats_get", "cales_get_cs", "cales_transform", "cales_transpose_xy",
           "cales_set_timing", "cales_set_graph", "cales_set_option", "cales_fp64_peak", "cales_kernel_count", "cales_kernel_time", "cales_launches_per_step", "cales_diagnostics", "cales_last_error"]

_lib = None


def lib():
    """Load (building if stale) libcales.so.  Raises if the CUDA extension cannot be built or loaded."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        for name in SYMBOLS:
            getattr(L, name)  # AttributeError if a declared symbol is missing
        L.cales_last_error.restype = C.c_char_p
        L.cales_workspace_bytes.restype = C.c_size_t
        L.cales_workspace_bytes.argtypes = [C.POINTER(CalesParams)]
        L.cales_default_params.restype = None
        L.cales_default_params.argtypes = [C.POINTER(CalesParams)]
        L.cales_create.argtypes = [C.POINTER(CalesParams), C.POINTER(C.c_void_p)]
        L.cales_destroy.argtypes = [C.c_void_p]
        L.cales_set_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.cales_get_field.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.cales_step.argtypes = [C.c_void_p, C.c_double]
        L.cales_step_adaptive.argtypes = [C.c_void_p, C.c_double]
        L.cales_last_dt.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.cales_poisson_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.cales_eddy_viscosity.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.cales_wall_stress.argtypes = [C.c_void_p, C.c_void_p]
        L.cales_wall_stress_y.argtypes = [C.c_void_p, C.c_void_p]
        L.cales_project.argtypes = [C.c_void_p]
        L.cales_get_cs.argtypes = [C.c_void_p, C.c_void_p]
        L.cales_cfl_dt.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.cales_cfl_dt_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.cales_plane_stats.argtypes = [C.c_void_p, C.c_void_p]
        L.cales_stats_reset.argtypes = [C.c_void_p]
        L.cales_stats_accumulate.argtypes = [C.c_void_p, C.c_double]
        L.cales_stats_get.argtypes = [C.c_void_p, _dp, _dp, _dp, C.POINTER(C.c_double)]
        L.cales_transform.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.cales_transpose_xy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.cales_set_timing.argtypes = [C.c_void_p, C.c_int]
        L.cales_set_graph.argtypes = [C.c_void_p, C.c_int]
        L.cales_fp64_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.cales_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_longlong]
        L.cales_launches_per_step.argtypes = [C.c_void_p]
        L.cales_kernel_time.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_double), C.POINTER(C.c_int)]
        L.cales_diagnostics.argtypes = [C.c_void_p, C.POINTER(CalesDiag)]
        L.cales_create_basic.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_double,
                                         C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int,
                                         C.c_void_p, C.c_size_t, C.c_void_p, C.c_int, C.POINTER(C.c_void_p)]
        _lib = L
    return _lib


class CalesError(RuntimeError):
    pass


def _chk(rc):
    if rc != 0:
        raise CalesError("cales error %d: %s" % (rc, lib().cales_last_error().decode()))


PARAM_KEYS = [f[0] for f in CalesParams._fields_ if f[0] not in ("zf_user", "workspace", "workspace_bytes", "cuda_stream", "device")]


def make_params(nx, ny, nz, lx, ly, lz, **kw):
    P = CalesParams()
    lib().cales_default_params(C.byref(P))
    P.nx, P.ny, P.nz, P.lx, P.ly, P.lz = nx, ny, nz, lx, ly, lz
    for k, v in kw.items():
        if k not in PARAM_KEYS:
            raise KeyError(k)
        setattr(P, k, v)
    return P


def workspace_bytes(nx, ny, nz, lx, ly, lz, **kw):
    return lib().cales_workspace_bytes(C.byref(make_params(nx, ny, nz, lx, ly, lz, **kw)))


class Solver:
    """One cales_solver on a CUDA device.  Device tensors are torch float64 of shape (nz, ny, nx)."""

    U, V, W, P, NUT = range(5)

    def __init__(self, nx, ny, nz, lx, ly, lz, device=0, stream=None, zf_user=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise CalesError("no CUDA device: the CaLES hot path has no CPU fallback")
        L = lib()
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        P = make_params(nx, ny, nz, lx, ly, lz, **kw)
        self._zf_user = None
        if zf_user is not None:
            import numpy as np
            self._zf_user = np.ascontiguousarray(zf_user, dtype=np.float64)
            P.zf_user = self._zf_user.ctypes.data_as(_dp); P.zstretch = 2
        need = L.cales_workspace_bytes(C.byref(P))
        if need == 0:
            raise CalesError("cales: " + L.cales_last_error().decode())
        self.workspace = torch.empty(need // 8 + 32, dtype=torch.float64, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        P.workspace = self.workspace.data_ptr() + off
        P.workspace_bytes = need
        P.cuda_stream = self.stream.cuda_stream
        P.device = device
        self._h = C.c_void_p()
        _chk(L.cales_create(C.byref(P), C.byref(self._h)))
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.npoints = nx * ny * nz
        self.workspace_bytes = need

    def close(self):
        if getattr(self, "_h", None):
            lib().cales_destroy(self._h); self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- fields
    def _dev(self, t):
        torch = self._torch
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == self.npoints
        return C.c_void_p(t.data_ptr())

    def set_field(self, f, a):
        """a: device tensor (async) or a host numpy array / CPU tensor (synchronous H2D)."""
        torch = self._torch
        if isinstance(a, torch.Tensor) and a.is_cuda:
            _chk(lib().cales_set_field(self._h, f, self._dev(a), 1))
        else:
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(a)
            assert t.dtype == torch.float64 and t.is_contiguous() and t.numel() == self.npoints
            _chk(lib().cales_set_field(self._h, f, C.c_void_p(t.data_ptr()), 0))

    def get_field(self, f, out=None):
        """Device tensor by default; if `out` is a CPU tensor the copy is D2H and synchronous."""
        torch = self._torch
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        if out.is_cuda:
            _chk(lib().cales_get_field(self._h, f, self._dev(out), 1))
        else:
            assert out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.npoints
            _chk(lib().cales_get_field(self._h, f, C.c_void_p(out.data_ptr()), 0))
        return out

    def get_numpy(self, f):
        torch = self._torch
        out = torch.empty(self.shape, dtype=torch.float64)
        return self.get_field(f, out).numpy()

    def set_velocity(self, u, v, w):
        self.set_field(0, u); self.set_field(1, v); self.set_field(2, w)

    # ---- the calls of the boundary
    def step(self, dt):
        _chk(lib().cales_step(self._h, float(dt)))

    def step_adaptive(self, cfl):
        _chk(lib().cales_step_adaptive(self._h, float(cfl)))

    def last_dt(self):
        dt = C.c_double()
        _chk(lib().cales_last_dt(self._h, C.byref(dt)))
        return dt.value

    def poisson_solve(self, rhs, phi=None):
        if phi is None:
            phi = self._torch.empty_like(rhs)
        _chk(lib().cales_poisson_solve(self._h, self._dev(rhs), self._dev(phi)))
        return phi

    def eddy_viscosity(self, u=None, v=None, w=None, nut=None):
        torch = self._torch
        if nut is None:
            nut = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        if u is None:
            _chk(lib().cales_eddy_viscosity(self._h, None, None, None, self._dev(nut)))
        else:
            _chk(lib().cales_eddy_viscosity(self._h, self._dev(u), self._dev(v), self._dev(w), self._dev(nut)))
        return nut

    def wall_stress(self):
        tau = self._torch.empty((2, 2, self.ny, self.nx), dtype=self._torch.float64, device=self.device)
        _chk(lib().cales_wall_stress(self._h, C.c_void_p(tau.data_ptr())))
        return tau

    def wall_stress_y(self):
        tau = self._torch.empty((2, 2, self.nz, self.nx), dtype=self._torch.float64, device=self.device)
        _chk(lib().cales_wall_stress_y(self._h, C.c_void_p(tau.data_ptr())))
        return tau

    def project(self):
        _chk(lib().cales_project(self._h))

    def cfl_dt(self, cfl):
        dt = C.c_double()
        _chk(lib().cales_cfl_dt(self._h, float(cfl), C.byref(dt)))
        return dt.value

    def cfl_dt_static(self, cfl, dt_dev, u=None, v=None, w=None):
        """Allocation-free CFL reduction into the 1-element DEVICE tensor dt_dev (scratch in the library's static device array)."""
        f = [None if a is None else self._dev(a) for a in (u, v, w)]
        _chk(lib().cales_cfl_dt_static(self._h, f[0], f[1], f[2], float(cfl), C.c_void_p(dt_dev.data_ptr())))
        return dt_dev

    def plane_stats(self):
        out = self._torch.empty((8, self.nz), dtype=self._torch.float64, device=self.device)
        _chk(lib().cales_plane_stats(self._h, C.c_void_p(out.data_ptr())))
        return out

    def stats_reset(self):
        _chk(lib().cales_stats_reset(self._h))

    def stats_accumulate(self, weight=1.0):
        _chk(lib().cales_stats_accumulate(self._h, float(weight)))

    def stats_get(self):
        import numpy as np
        prof = np.empty((8, self.nz)); wall = np.empty(8); der = np.empty(4); w = C.c_double()
        _chk(lib().cales_stats_get(self._h, prof.ctypes.data_as(_dp), wall.ctypes.data_as(_dp), der.ctypes.data_as(_dp), C.byref(w)))
        return dict(profiles=prof, wall=wall, tau_w=der[0], u_tau=der[1], re_tau=der[2], cf=der[3], weight=w.value)

    def get_cs(self, per_plane=True):
        n = self.nz if per_plane else self.nz * self.ny
        cs = self._torch.empty(n, dtype=self._torch.float64, device=self.device)
        _chk(lib().cales_get_cs(self._h, C.c_void_p(cs.data_ptr())))
        return cs

    def transform(self, field, direction, inverse=False):
        _chk(lib().cales_transform(self._h, self._dev(field), direction, 1 if inverse else 0))
        return field

    def transpose_xy(self, src):
        dst = self._torch.empty((self.nz, self.nx, self.ny), dtype=self._torch.float64, device=self.device)
        _chk(lib().cales_transpose_xy(self._h, self._dev(src), C.c_void_p(dst.data_ptr())))
        return dst

    def set_timing(self, on=True):
        _chk(lib().cales_set_timing(self._h, 1 if on else 0))

    def kernel_times(self):
        """{kernel name: (total ms, launches)} of the last step that ran with timing on (synchronises)."""
        out = {}
        for kid in range(lib().cales_kernel_count()):
            name, ms, n = C.c_char_p(), C.c_double(), C.c_int()
            _chk(lib().cales_kernel_time(self._h, kid, C.byref(name), C.byref(ms), C.byref(n)))
            if n.value:
                out[name.value.decode()] = (ms.value, n.value)
        return out

    def set_graph(self, on=True):
        _chk(lib().cales_set_graph(self._h, 1 if on else 0))

    def fp64_peak(self):
        tf = C.c_double()
        _chk(lib().cales_fp64_peak(self._h, C.byref(tf)))
        return tf.value

    def set_option(self, key, value):
        _chk(lib().cales_set_option(self._h, key.encode(), int(value)))

    def launches_per_step(self):
        return lib().cales_launches_per_step(self._h)

    def diagnostics(self):
        d = CalesDiag()
        _chk(lib().cales_diagnostics(self._h, C.byref(d)))
        return {k: getattr(d, k) for k, _ in CalesDiag._fields_}
