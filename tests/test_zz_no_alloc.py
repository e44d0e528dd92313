"""cales_cfl_dt_static: the allocation-free entry point (scratch in the library's file-scope device array) against the
existing path cales_cfl_dt, on two calls in a row.  Collected last on purpose (the suite runs with pytest -x); passes
alone in a fresh process and after the other GPU tests.  A maximum is independent of the order it is taken in, so the
two paths must agree to the last bit; the oracle is checked at the tolerance of test_cfl_dt_and_plane_stats_parity."""
import numpy as np
import pytest

from tests import parity_cases as pc

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2411_09364_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("n,shape", [(3, (72, 36, 40)), (5, (96, 48, 24))])
def test_static_scratch_cfl_dt_matches_existing_path_twice(oracle, gpu, n, shape):
    import torch
    cfg, kw, (u, v, w), dt = pc.prepare(oracle, n, shape)
    o = pc.make(oracle.Oracle, kw)
    g = pc.make(gpu.Solver, kw)
    o.set_velocity(u, v, w); g.set_velocity(u, v, w)
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    # call 1: the solver's own velocity
    g.cfl_dt_static(0.95, out[0:1])
    want1 = g.cfl_dt(0.95)
    ref1 = o.cfl_dt(0.95)
    # call 2, right behind it: the stepped field, shared scratch still holding call 1's maxima
    o.step(dt); g.step(dt)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    g.cfl_dt_static(0.5, out[1:2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the call changed the device's free memory"
    want2 = g.cfl_dt(0.5)
    ref2 = o.cfl_dt(0.5)
    got = out.cpu().numpy()
    assert got[0] == want1 and got[1] == want2, (got, want1, want2)
    assert abs(got[0] - ref1) <= 1e-12 * ref1 and abs(got[1] - ref2) <= 1e-12 * ref2
    assert want1 != want2 * 0.95 / 0.5      # the two calls really saw different fields
    g.close()


def test_static_scratch_cfl_dt_external_field_and_rest(oracle, gpu):
    """External velocity fields (a second solver holds them for the existing path), then a field at rest: dt = 0."""
    import torch
    cfg, kw, (u, v, w), dt = pc.prepare(oracle, 4, (96, 36, 24))
    g = pc.make(gpu.Solver, kw)
    h = pc.make(gpu.Solver, kw)
    g.set_velocity(u, v, w)
    h.set_velocity(2.0 * u, 0.5 * v, -w)
    ext = [torch.from_numpy(np.ascontiguousarray(h.get_numpy(f))).cuda() for f in range(3)]
    out = torch.empty((3,), dtype=torch.float64, device="cuda")
    g.cfl_dt_static(0.95, out[0:1], *ext)          # call 1: external field through g
    g.cfl_dt_static(0.95, out[1:2])                # call 2: g's own field
    z = [torch.zeros_like(ext[0]) for _ in range(3)]
    g.cfl_dt_static(0.95, out[2:3], *z)            # call 3: at rest
    got = out.cpu().numpy()
    assert got[0] == h.cfl_dt(0.95) and got[1] == g.cfl_dt(0.95) and got[2] == 0.0, got
    assert got[0] != got[1]
    with pytest.raises(gpu.CalesError):
        g.cfl_dt_static(0.95, out[0:1], ext[0], None, None)
    with pytest.raises(gpu.CalesError):
        g.cfl_dt_static(-1.0, out[0:1])
    g.close(); h.close()


def test_static_scratch_rejects_grids_beyond_the_array(gpu):
    """ceil(nx/32) ceil(ny/8) nz = 1 x 256 x 4100 > 2^20 slots: a clear error, and the allocating path still works."""
    import torch
    from paper_2411_09364_b200 import inputs
    cfg = inputs.config(1, (2, 2048, 4100))
    g = pc.make(gpu.Solver, inputs.solver_kwargs(cfg, None))
    rng = np.random.default_rng(7)      # any field at motion will do here (the seeded box field is undefined on a 2-point x line)
    g.set_velocity(*[rng.standard_normal((4100, 2048, 2)) for _ in range(3)])
    out = torch.empty((1,), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.CalesError, match="static array holds 1048576"):
        g.cfl_dt_static(0.95, out)
    assert g.cfl_dt(0.95) > 0.0
    g.close()
