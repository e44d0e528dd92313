"""CPU-only check of the DEVICE code's arithmetic: the kernels of libcales.so are __host__ __device__ phase
functions; tests/emu steps those same functions on the host in launch order.  Here that emulation is compared
with the CPU oracle on reduced replicas of all five configurations (same option sets), so that index / sign /
boundary mistakes in the kernels surface without a GPU.  The real parity gate is tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

from tests import parity_cases as pc


@pytest.fixture(scope="module")
def emu():
    from tests import emu as e
    return e


@pytest.mark.parametrize("case", sorted(pc.SMALL))
def test_emulated_kernels_match_oracle(oracle, emu, case):
    n, shape, steps = pc.SMALL[case][:3]
    cfg, kw, (u, v, w), dt = pc.prepare(oracle, n, shape, *pc.SMALL[case][3:])
    o = pc.make(oracle.Oracle, kw)
    e = pc.make(emu.Emu, kw)
    o.set_velocity(u, v, w); e.set_velocity(u, v, w)
    for s in range(steps):
        o.step(dt); e.step(dt)
        err = pc.field_errors([e.get(f) for f in range(5)], [o.get(f) for f in range(5)], o.dzf, kw["nu"])
        assert max(err.values()) <= 1e-11, (case, s, err)
    assert abs(e.cfl_dt(0.95) - o.cfl_dt(0.95)) <= 1e-12 * o.cfl_dt(0.95)
    sa, sb = e.plane_stats(), o.plane_stats()
    assert np.max(np.abs(sa - sb)) <= 1e-11 * np.max(np.abs(sb))
    # projection quality of the emulated device path (north_star: <= 1e-12 x velocity scale)
    scale = max(np.max(np.abs(o.get(0))), 1e-300) / min(o.dx, o.dy, float(np.min(o.dzf)))
    assert e.max_div() <= 1e-12 * scale * 10


@pytest.mark.parametrize("bc_y,bc_z,stretch", [(0, 0, 0), (0, 1, 0), (0, 1, 1), (1, 1, 0), (1, 1, 1)])
def test_emulated_poisson_matches_oracle(oracle, emu, bc_y, bc_z, stretch):
    nx, ny, nz = 24, 12, 10
    kw = dict(bc_y=bc_y, bc_z=bc_z, zstretch=stretch, zstretch_factor=1.5 if stretch else 0.0)
    o = oracle.Oracle(nx, ny, nz, 2.0, 1.5, 1.0, **kw)
    e = emu.Emu(nx, ny, nz, 2.0, 1.5, 1.0, **kw)
    rhs = np.random.default_rng(5).standard_normal((nz, ny, nx))
    a, b = e.poisson_solve(rhs), o.poisson_solve(rhs)
    assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))


@pytest.mark.parametrize("n", [2, 6, 8, 12, 32, 96, 192])
def test_emulated_transforms_match_numpy_scipy(emu, n):
    import scipy.fft
    rng = np.random.default_rng(n)
    # x direction: packed half-complex real FFT
    e = emu.Emu(n, 4, 4, 1.0, 1.0, 1.0)
    f = rng.standard_normal((4, 4, n))
    F = e.transform(f, 0)
    X = np.fft.rfft(f, axis=2)
    assert np.allclose(F[..., 0], X[..., 0].real, atol=1e-12) and np.allclose(F[..., 1], X[..., n // 2].real, atol=1e-12)
    if n > 2:
        assert np.allclose(F[..., 2::2], X[..., 1:n // 2].real, atol=1e-12)
        assert np.allclose(F[..., 3::2], X[..., 1:n // 2].imag, atol=1e-12)
    assert np.allclose(e.transform(F, 0, inverse=True), f, atol=1e-12)
    # y direction: FFT (periodic) and DCT-II (walls)
    for bc_y in (0, 1):
        e = emu.Emu(4, n, 4, 1.0, 1.0, 1.0, bc_y=bc_y, bc_z=1)
        f = rng.standard_normal((4, n, 4))
        F = e.transform(f, 1)
        if bc_y == 0:
            X = np.fft.rfft(f, axis=1)
            assert np.allclose(F[:, 0], X[:, 0].real, atol=1e-12) and np.allclose(F[:, 1], X[:, n // 2].real, atol=1e-12)
            if n > 2:
                assert np.allclose(F[:, 2::2], X[:, 1:n // 2].real, atol=1e-12)
                assert np.allclose(F[:, 3::2], X[:, 1:n // 2].imag, atol=1e-12)
        else:
            assert np.allclose(F, 0.5 * scipy.fft.dct(f, type=2, axis=1), atol=1e-12)
        assert np.allclose(e.transform(F, 1, inverse=True), f, atol=1e-12)


def _fuzz_cases():
    """Seeded random option sets on small, awkward grids (sizes of the form 2^a 3^b down to 2, all boundary combinations)."""
    rng = np.random.default_rng(20241109)
    sizes_xy = [2, 4, 6, 8, 12, 16, 18, 24, 32, 36, 48]
    out = []
    for t in range(14):
        bc_z = int(rng.integers(0, 2)); bc_y = int(rng.integers(0, 2)) if bc_z else 0
        nx, ny = int(rng.choice(sizes_xy)), int(rng.choice(sizes_xy)); nz = int(rng.integers(4, 14))
        stretch = int(bc_z and rng.integers(0, 2))
        sgs = int(rng.integers(0, 3))
        wm = int(bc_z and rng.integers(0, 2))
        imp = int(bc_z and rng.integers(0, 2))
        vd = int(sgs == 1 and bc_z and not bc_y and not wm and rng.integers(0, 2))
        kw = dict(bc_y=bc_y, bc_z=bc_z, zstretch=stretch, zstretch_factor=1.3 if stretch else 0.0, nu=float(rng.uniform(1e-3, 2e-2)),
                  sgs_model=sgs, cs=0.12, van_driest=vd, dsm_avg_xy_plane=int(rng.integers(0, 2)), dsm_clip_total=int(rng.integers(0, 2)),
                  wall_model=wm, h_wm=float(rng.choice([0.0, 0.12])) if wm else 0.0, implicit_z=imp,
                  const_flow_rate=int(rng.integers(0, 2)), u_bulk=1.0)
        out.append((t, nx, ny, nz, kw))
    rng = np.random.default_rng(20241128)           # dynamic model with the 3-D box test filter
    for t in range(14, 22):
        bc_z = int(rng.integers(0, 2)); bc_y = int(rng.integers(0, 2)) if bc_z else 0
        nx, ny = int(rng.choice(sizes_xy)), int(rng.choice(sizes_xy)); nz = int(rng.integers(4, 14))
        stretch = int(bc_z and rng.integers(0, 2))
        wm = int(bc_z and rng.integers(0, 2))
        kw = dict(bc_y=bc_y, bc_z=bc_z, zstretch=stretch, zstretch_factor=1.3 if stretch else 0.0, nu=float(rng.uniform(1e-3, 2e-2)),
                  sgs_model=2, dsm_filter3d=1, dsm_avg_xy_plane=int(rng.integers(0, 2)), dsm_clip_total=int(rng.integers(0, 2)),
                  wall_model=wm, wall_model_y=int(bc_y and rng.integers(0, 2)), h_wm=0.0, implicit_z=int(bc_z and rng.integers(0, 2)),
                  const_flow_rate=int(rng.integers(0, 2)), u_bulk=1.0)
        out.append((t, nx, ny, nz, kw))
    return out


@pytest.mark.parametrize("t,nx,ny,nz,kw", _fuzz_cases())
def test_fuzzed_option_sets_match_oracle(oracle, emu, t, nx, ny, nz, kw):
    rng = np.random.default_rng(100 + t)
    lz = 2.0
    u = 1.0 + 0.3 * rng.standard_normal((nz, ny, nx)); v = 0.3 * rng.standard_normal((nz, ny, nx)); w = 0.3 * rng.standard_normal((nz, ny, nx))
    if kw["bc_z"]:
        w[-1] = 0.0
    if kw["bc_y"]:
        v[:, -1, :] = 0.0
    o = oracle.Oracle(nx, ny, nz, 3.0, 2.0, lz, **kw)
    o.set_velocity(u, v, w); o.project(); u, v, w = o.velocity()
    if kw["const_flow_rate"]:
        kw = dict(kw, u_bulk=float(np.sum(u * o.dzf[:, None, None]) / (nx * ny * lz)))
        o = oracle.Oracle(nx, ny, nz, 3.0, 2.0, lz, **kw)
    e = emu.Emu(nx, ny, nz, 3.0, 2.0, lz, **kw)
    o.set_velocity(u, v, w); e.set_velocity(u, v, w)
    dt = 0.2 * min(3.0 / nx, 2.0 / ny, float(np.min(o.dzf))) / 2.0
    for s in range(2):
        o.step(dt); e.step(dt)
    err = pc.field_errors([e.get(f) for f in range(5)], [o.get(f) for f in range(5)], o.dzf, kw["nu"])
    assert max(err.values()) <= 1e-10, (t, nx, ny, nz, kw, err)
