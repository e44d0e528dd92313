"""Seeded synthetic workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it only names the five BASELINE.json configurations (plus reduced replicas with the same
option set) and draws the seeded initial fields with numpy.  It imports neither the CUDA binding nor
the oracle.  The fields stand in for the paper's workloads (DIT PAPER.md:219-229, WRLES channel
PAPER.md:235-253, WMLES channel PAPER.md:275-342, duct PAPER.md:363-383), whose experimental / DNS
datasets are not available here.

Arrays are float64, shape (nz, ny, nx), x fastest; u on +x faces, v on +y faces, w on +z faces.
"""
import math
import numpy as np

KAPPA, BLOG = 0.41, 5.2


def _base(**kw):
    d = dict(zstretch=0, zstretch_factor=0.0, bc_y=0, bc_z=0, nu=1e-3, sgs_model=0, cs=0.17, van_driest=0,
             aplus=25.0, dsm_avg_xy_plane=1, dsm_clip_total=0, dsm_alpha2d=0.0, wall_model=0, kappa=KAPPA,
             B=BLOG, h_wm=0.0, wm_tol=1e-4, wm_maxit=50, implicit_z=0, const_flow_rate=0, u_bulk=0.0, wall_model_y=0, dsm_filter3d=0, implicit_xyz=0)
    d.update(kw)
    return d


def config(n, shape=None):
    """Return the description of BASELINE.json config n (1..5); `shape=(nx,ny,nz)` gives a reduced
    replica with the same box and option set.  Keys: name, params (solver keyword arguments), seed,
    steps, dt (fixed) or cfl, init (recipe name), retau / profile constants."""
    pi = math.pi
    if n == 1:
        nx, ny, nz = shape or (32, 32, 32)
        return dict(name="dit32" if shape is None else "dit", seed=1001, steps=10, dt=1e-3, cfl=None, init="dit",
                    params=dict(nx=nx, ny=ny, nz=nz, lx=2 * pi, ly=2 * pi, lz=2 * pi,
                                **_base(nu=1e-3, sgs_model=1, cs=0.17)))
    if n == 2:
        nx, ny, nz = shape or (192, 96, 64)
        return dict(name="wmles_channel_2000", seed=1002, steps=100, dt=None, cfl=0.5, init="loglaw", retau=2000.0,
                    params=dict(nx=nx, ny=ny, nz=nz, lx=2 * pi, ly=pi, lz=2.0,
                                **_base(bc_z=1, nu=1.0 / 2000.0, sgs_model=1, cs=0.1, wall_model=1, const_flow_rate=1)))
    if n == 3:
        nx, ny, nz = shape or (256, 256, 192)
        return dict(name="wrles_channel_550", seed=1003, steps=100, dt=None, cfl=0.5, init="poiseuille",
                    params=dict(nx=nx, ny=ny, nz=nz, lx=2 * pi, ly=pi, lz=2.0,
                                **_base(bc_z=1, zstretch=1, zstretch_factor=1.5, nu=1e-4, sgs_model=1, cs=0.1,
                                        van_driest=1, aplus=25.0, implicit_z=1, const_flow_rate=1, u_bulk=1.0)))
    if n == 4:
        nx, ny, nz = shape or (1024, 256, 256)
        return dict(name="duct_4410", seed=1004, steps=50, dt=None, cfl=0.5, init="duct",
                    params=dict(nx=nx, ny=ny, nz=nz, lx=6.0, ly=2.0, lz=2.0,
                                **_base(bc_y=1, bc_z=1, nu=1.0 / 4410.0, sgs_model=2, dsm_avg_xy_plane=0,
                                        dsm_clip_total=1, const_flow_rate=1, u_bulk=1.0)))
    if n == 5:
        nx, ny, nz = shape or (1536, 1024, 512)
        return dict(name="wmles_channel_5200", seed=1005, steps=20, dt=None, cfl=0.5, init="loglaw", retau=5200.0,
                    params=dict(nx=nx, ny=ny, nz=nz, lx=6 * pi, ly=2 * pi, lz=2.0,
                                **_base(bc_z=1, nu=1.0 / 5200.0, sgs_model=2, dsm_avg_xy_plane=1, dsm_clip_total=0,
                                        wall_model=1, const_flow_rate=1)))
    raise ValueError("config must be 1..5")


def z_faces(p):
    """z faces of the configuration's grid (uniform, or the two-sided tanh of DESIGN.md reading S16).
    Only used to place the initial profile; each solver builds its own grid."""
    nz, lz = p["nz"], p["lz"]
    k = np.arange(nz + 1, dtype=np.float64)
    if p["zstretch"] == 1:
        a = p["zstretch_factor"]
        zf = 0.5 * lz * (1.0 + np.tanh(a * (2.0 * k / nz - 1.0)) / math.tanh(a))
    else:
        zf = lz * k / nz
    zf[0], zf[-1] = 0.0, lz
    return zf


def _dit(p, rng):
    """Random-phase solenoidal field with E(k) ~ k^4 exp(-2 (k/4)^2), sampled at the staggered face
    positions by spectral phase shifts, scaled to u_rms = 1 (BASELINE.json config 1)."""
    nx, ny, nz = p["nx"], p["ny"], p["nz"]
    kx = np.fft.fftfreq(nx, 1.0 / nx) * (2 * math.pi / p["lx"])
    ky = np.fft.fftfreq(ny, 1.0 / ny) * (2 * math.pi / p["ly"])
    kz = np.fft.fftfreq(nz, 1.0 / nz) * (2 * math.pi / p["lz"])
    KZ, KY, KX = np.meshgrid(kz, ky, kx, indexing="ij")
    K2 = KX ** 2 + KY ** 2 + KZ ** 2
    K = np.sqrt(K2)
    a = rng.standard_normal((3, nz, ny, nx)) + 1j * rng.standard_normal((3, nz, ny, nx))
    K2s = np.where(K2 > 0, K2, 1.0)
    kdota = (KX * a[0] + KY * a[1] + KZ * a[2]) / K2s
    a[0] -= KX * kdota; a[1] -= KY * kdota; a[2] -= KZ * kdota
    E = K ** 4 * np.exp(-2.0 * (K / 4.0) ** 2)
    amp = np.sqrt(E / (4 * math.pi * K2s))
    amp[K2 == 0] = 0.0
    kmax = min(nx, ny, nz) // 2 * 0.95        # keep away from the Nyquist planes
    amp[K > kmax * (2 * math.pi / max(p["lx"], p["ly"], p["lz"]))] = 0.0
    dx, dy, dz = p["lx"] / nx, p["ly"] / ny, p["lz"] / nz
    # cell index (i,j,k) <-> centre ((i+1/2)dx, ...); u lives at (i+1)dx etc.
    cen = np.exp(1j * (KX * 0.5 * dx + KY * 0.5 * dy + KZ * 0.5 * dz))
    sh = [np.exp(1j * KX * 0.5 * dx), np.exp(1j * KY * 0.5 * dy), np.exp(1j * KZ * 0.5 * dz)]
    out = [np.real(np.fft.ifftn(a[c] * amp * cen * sh[c])) for c in range(3)]
    urms = math.sqrt(sum(float(np.mean(o * o)) for o in out) / 3.0)
    return [np.ascontiguousarray(o / urms) for o in out]


def _noise(rng, shape, amp):
    r = rng.random(shape)          # uniform in [-amp, amp), built in place (config 5 is 6.4 GB per field)
    r *= 2.0 * amp
    r -= amp
    return r


def initial_fields(cfg):
    """(u, v, w, u_bulk) for a configuration from config(); u_bulk is None where no flow rate is imposed."""
    p = cfg["params"]
    nx, ny, nz = p["nx"], p["ny"], p["nz"]
    rng = np.random.default_rng(cfg["seed"])
    shape = (nz, ny, nx)
    if cfg["init"] == "dit":
        u, v, w = _dit(p, rng)
        return u, v, w, None
    zf = z_faces(p)
    zc = 0.5 * (zf[:-1] + zf[1:])
    dzf = zf[1:] - zf[:-1]
    h = 0.5 * p["lz"]
    if cfg["init"] == "loglaw":
        dplus = np.minimum(zc, p["lz"] - zc) * cfg["retau"] / h
        prof = np.log(dplus) / KAPPA + BLOG
        ub = float(np.sum(prof * dzf) / p["lz"])
        U = np.broadcast_to(prof[:, None, None], shape)
    elif cfg["init"] == "poiseuille":
        ub = p["u_bulk"]
        prof = 1.5 * ub * (1.0 - ((zc - h) / h) ** 2)
        U = np.broadcast_to(prof[:, None, None], shape)
    elif cfg["init"] == "duct":
        ub = p["u_bulk"]
        yc = (np.arange(ny) + 0.5) * p["ly"] / ny
        hy = 0.5 * p["ly"]
        U = 2.25 * ub * (1.0 - ((zc[:, None, None] - h) / h) ** 2) * (1.0 - ((yc[None, :, None] - hy) / hy) ** 2)
        U = np.broadcast_to(U, shape)
    else:
        raise ValueError(cfg["init"])
    u = _noise(rng, shape, 0.1 * ub)
    u += U
    v = _noise(rng, shape, 0.1 * ub)
    w = _noise(rng, shape, 0.1 * ub)
    if p["bc_z"] == 1:
        w[nz - 1] = 0.0          # the top wall face
    if p["bc_y"] == 1:
        v[:, ny - 1, :] = 0.0    # the +y wall face
    return np.ascontiguousarray(u), np.ascontiguousarray(v), np.ascontiguousarray(w), ub


def time_step(cfg, u, v, w):
    """dt of the run (reading S18): the fixed value of the config, or CFL / max(|u|/dx+|v|/dy+|w|/dzf)
    from the initial field, fixed for the whole run; the same double goes to both implementations."""
    if cfg["dt"] is not None:
        return float(cfg["dt"])
    p = cfg["params"]
    zf = z_faces(p)
    dzf = (zf[1:] - zf[:-1])[:, None, None]
    dx, dy = p["lx"] / p["nx"], p["ly"] / p["ny"]
    rmax = 0.0
    step = max(1, (1 << 24) // (p["nx"] * p["ny"]))       # k-slabs of ~16 M points keep the temporaries small
    for k0 in range(0, p["nz"], step):
        sl = slice(k0, k0 + step)
        rmax = max(rmax, float((np.abs(u[sl]) / dx + np.abs(v[sl]) / dy + np.abs(w[sl]) / dzf[sl]).max()))
    return float(cfg["cfl"] / rmax)


def solver_kwargs(cfg, u_bulk):
    """Solver keyword arguments of a configuration with the imposed bulk velocity filled in."""
    p = dict(cfg["params"])
    if p["const_flow_rate"] and u_bulk is not None:
        p["u_bulk"] = float(u_bulk)
    return p
