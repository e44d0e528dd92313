"""ctypes binding of oracle/liboracle.so (argument marshalling only).  TEST INFRASTRUCTURE ONLY."""
import ctypes as C
import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)


class OracleParams(C.Structure):
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
        ("wall_model_y", C.c_int), ("dsm_filter3d", C.c_int), ("implicit_xyz", C.c_int),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_loglaw_hplus.restype = C.c_double
        L.oracle_loglaw_hplus.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_int)]
        L.oracle_rk3_coeffs.restype = None
        L.oracle_destroy.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _arr(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _chk(rc):
    if rc != 0:
        raise RuntimeError("oracle: " + lib().oracle_last_error().decode())


def num_threads():
    return lib().oracle_num_threads()


def fft_c2c(x, sign=-1):
    x = np.asarray(x, dtype=np.complex128)
    n = x.size
    re, im = _arr(x.real), _arr(x.imag)
    ro, io = np.empty(n), np.empty(n)
    _chk(lib().oracle_fft_c2c(n, _p(re), _p(im), _p(ro), _p(io), sign))
    return ro + 1j * io


def dct2(x):
    x = _arr(x); X = np.empty_like(x)
    _chk(lib().oracle_dct2(x.size, _p(x), _p(X))); return X


def dct3(X):
    X = _arr(X); x = np.empty_like(X)
    _chk(lib().oracle_dct3(X.size, _p(X), _p(x))); return x


def thomas(a, b, c, d, cyclic=False):
    a, b, c, d = map(_arr, (a, b, c, d)); x = np.empty_like(d)
    f = lib().oracle_thomas_cyclic if cyclic else lib().oracle_thomas
    _chk(f(d.size, _p(a), _p(b), _p(c), _p(d), _p(x))); return x


def loglaw_hplus(re_wm, kappa=0.41, B=5.2, tol=1e-4, maxit=50):
    it = C.c_int(0)
    h = lib().oracle_loglaw_hplus(float(re_wm), kappa, B, tol, maxit, C.byref(it))
    return h, it.value


def rk3_coeffs(k):
    a, b, g = C.c_double(), C.c_double(), C.c_double()
    lib().oracle_rk3_coeffs(k, C.byref(a), C.byref(b), C.byref(g))
    return a.value, b.value, g.value


PARAM_DEFAULTS = dict(
    zstretch=0, zstretch_factor=0.0, bc_y=0, bc_z=0, nu=1e-3, sgs_model=0, cs=0.17, van_driest=0, aplus=25.0,
    dsm_avg_xy_plane=1, dsm_clip_total=0, dsm_alpha2d=0.0, wall_model=0, kappa=0.41, B=5.2, h_wm=0.0,
    wm_tol=1e-4, wm_maxit=50, implicit_z=0, const_flow_rate=0, u_bulk=0.0, wall_model_y=0, dsm_filter3d=0, implicit_xyz=0)


class Oracle:
    """One oracle solver instance.  Arrays are numpy float64 of shape (nz, ny, nx)."""

    U, V, W, P, NUT = range(5)

    def __init__(self, nx, ny, nz, lx, ly, lz, zf_user=None, **kw):
        d = dict(PARAM_DEFAULTS); d.update(kw)
        self.params = dict(nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, **d)
        P = OracleParams()
        for k, v in self.params.items():
            setattr(P, k, v)
        self._zf_user = None
        if zf_user is not None:
            self._zf_user = _arr(zf_user); P.zf_user = _p(self._zf_user); P.zstretch = 2
        self._h = C.c_void_p()
        _chk(lib().oracle_create(C.byref(P), C.byref(self._h)))
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.zf, self.zc, self.dzf = np.empty(nz + 1), np.empty(nz), np.empty(nz)
        self._dzc = np.empty(nz + 1)
        _chk(lib().oracle_get_grid(self._h, _p(self.zf), _p(self.zc), _p(self.dzf), _p(self._dzc)))
        self.dx, self.dy = lx / nx, ly / ny

    def dzc(self, k):
        return self._dzc[k + 1]

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.oracle_destroy(self._h); self._h = None

    def set(self, f, a):
        a = _arr(a); assert a.shape == self.shape
        _chk(lib().oracle_set_field(self._h, f, _p(a)))

    def get(self, f):
        a = np.empty(self.shape); _chk(lib().oracle_get_field(self._h, f, _p(a))); return a

    def set_velocity(self, u, v, w):
        self.set(0, u); self.set(1, v); self.set(2, w)

    def velocity(self):
        return self.get(0), self.get(1), self.get(2)

    def step(self, dt):
        _chk(lib().oracle_step(self._h, C.c_double(dt)))

    def substep(self, rk, dt):
        _chk(lib().oracle_substep(self._h, C.c_int(rk), C.c_double(dt)))

    def ustar(self):
        out = [np.empty(self.shape) for _ in range(3)]
        for c in range(3):
            _chk(lib().oracle_get_ustar(self._h, c, _p(out[c])))
        return out

    def poisson_solve(self, rhs):
        rhs = _arr(rhs); phi = np.empty(self.shape)
        _chk(lib().oracle_poisson_solve(self._h, _p(rhs), _p(phi))); return phi

    def helmholtz_solve(self, comp, c, rhs):
        rhs = _arr(rhs); out = np.empty(self.shape)
        _chk(lib().oracle_helmholtz_solve(self._h, C.c_int(comp), C.c_double(c), _p(rhs), _p(out))); return out

    def laplacian(self, phi):
        phi = _arr(phi); out = np.empty(self.shape)
        _chk(lib().oracle_laplacian(self._h, _p(phi), _p(out))); return out

    def eddy_viscosity(self, u=None, v=None, w=None):
        nut = np.empty(self.shape)
        if u is None:
            _chk(lib().oracle_eddy_viscosity(self._h, None, None, None, _p(nut)))
        else:
            u, v, w = map(_arr, (u, v, w))
            _chk(lib().oracle_eddy_viscosity(self._h, _p(u), _p(v), _p(w), _p(nut)))
        return nut

    def wall_stress(self):
        tau = np.empty((2, 2, self.ny, self.nx)); _chk(lib().oracle_wall_stress(self._h, _p(tau))); return tau

    def wall_stress_y(self):
        tau = np.empty((2, 2, self.nz, self.nx)); _chk(lib().oracle_wall_stress_y(self._h, _p(tau))); return tau

    def _three(self, fn, *extra):
        a, b, c = (np.empty(self.shape) for _ in range(3))
        _chk(fn(self._h, _p(a), _p(b), _p(c), *extra)); return a, b, c

    def advection(self):
        return self._three(lib().oracle_advection)

    def diffusion(self, which=0):
        return self._three(lib().oracle_diffusion, C.c_int(which))

    def sgs_term(self):
        return self._three(lib().oracle_sgs_term)

    def divergence(self):
        d = np.empty(self.shape); _chk(lib().oracle_divergence(self._h, _p(d))); return d

    def strain(self):
        S = np.empty((6,) + self.shape); m = np.empty(self.shape)
        _chk(lib().oracle_strain(self._h, _p(S), _p(m))); return S, m

    def filter_xy(self, q):
        q = _arr(q); out = np.empty(self.shape)
        _chk(lib().oracle_filter_xy(self._h, _p(q), _p(out))); return out

    def test_filter(self, q, kind=0):
        q = _arr(q); out = np.empty(self.shape)
        _chk(lib().oracle_test_filter(self._h, _p(q), _p(out), C.c_int(kind))); return out

    def get_cs(self):
        n = self.nz if self.params["dsm_avg_xy_plane"] else self.nz * self.ny
        cs = np.empty(n); _chk(lib().oracle_get_cs(self._h, _p(cs))); return cs

    def dsm_tensors(self):
        L = np.empty((6,) + self.shape); M = np.empty((6,) + self.shape)
        _chk(lib().oracle_get_dsm_tensors(self._h, _p(L), _p(M))); return L, M

    def cfl_dt(self, cfl):
        dt = C.c_double(); _chk(lib().oracle_cfl_dt(self._h, C.c_double(cfl), C.byref(dt))); return dt.value

    def plane_stats(self):
        out = np.empty((8, self.nz)); _chk(lib().oracle_plane_stats(self._h, _p(out))); return out

    def stats_reset(self):
        _chk(lib().oracle_stats_reset(self._h))

    def stats_accumulate(self, weight=1.0):
        _chk(lib().oracle_stats_accumulate(self._h, C.c_double(weight)))

    def stats_get(self):
        prof = np.empty((8, self.nz)); wall = np.empty(8); der = np.empty(4); w = C.c_double()
        _chk(lib().oracle_stats_get(self._h, _p(prof), _p(wall), _p(der), C.byref(w)))
        return dict(profiles=prof, wall=wall, tau_w=der[0], u_tau=der[1], re_tau=der[2], cf=der[3], weight=w.value)

    def project(self):
        _chk(lib().oracle_project(self._h))

    def diagnostics(self):
        md, ub, ke, fo = (C.c_double() for _ in range(4)); it = C.c_int()
        _chk(lib().oracle_diagnostics(self._h, C.byref(md), C.byref(ub), C.byref(ke), C.byref(fo), C.byref(it)))
        return dict(max_div=md.value, u_bulk=ub.value, kinetic_energy=ke.value, forcing=fo.value, wm_max_iters=it.value)
