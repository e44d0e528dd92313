"""Full-size parity: the GPU path against the CPU oracle at BASELINE.json's sizes for configs 3, 4 and 5, in the launch
geometry bench.py times (rt_chunk, TI, L, 64-bit offsets), element by element, at north_star's one-step bound 1e-11.

Config 3 (256x256x192) and config 4 (1024x256x256) run the oracle on the whole grid (seconds to minutes on the box's host
cores).  Config 5 (1536x1024x512, 805 M points) is beyond the oracle's reach in a test, so it is covered by x-y periodic
tiling: the oracle steps a 192x128x512 box of the same dx, dy and z grid; the GPU steps that field tiled 8x8 in x-y.  Every
stencil, the plane-averaged dynamic coefficient, the wall model and the bulk-velocity forcing are invariant under the tiling
(the plane sums are 64 x the small ones, their ratio unchanged up to round-off), so every tile of the GPU result must equal
the oracle's field.
"""
import numpy as np
import pytest

from tests import parity_cases as pc

pytestmark = pytest.mark.gpu

TOL_1STEP = 1e-11


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2411_09364_b200 import binding
    binding.lib()
    return binding


def _need(host_bytes, dev_bytes):
    import psutil
    import torch
    torch.cuda.empty_cache()          # blocks cached by earlier tests are not free memory to mem_get_info
    free, _ = torch.cuda.mem_get_info()
    if free < dev_bytes or psutil.virtual_memory().available < host_bytes:
        pytest.skip("not enough device / host memory (need %.0f / %.0f GB)" % (dev_bytes / 1e9, host_bytes / 1e9))


@pytest.mark.parametrize("n,steps", [(3, 2), (4, 1)])
def test_full_size_oracle_parity(oracle, gpu, n, steps):
    from paper_2411_09364_b200 import inputs
    p = inputs.config(n)["params"]
    npts = p["nx"] * p["ny"] * p["nz"]
    _need(90 * npts * 8, 20 * npts * 8)
    cfg, kw, (u, v, w), dt = pc.prepare(oracle, n, None)
    o = pc.make(oracle.Oracle, kw)
    g = pc.make(gpu.Solver, kw)
    o.set_velocity(u, v, w); g.set_velocity(u, v, w)
    del u, v, w
    for s in range(steps):
        o.step(dt); g.step(dt)
        err = pc.field_errors([g.get_numpy(f) for f in range(5)], [o.get(f) for f in range(5)], o.dzf, kw["nu"])
        assert max(err.values()) <= TOL_1STEP * (1 if s == 0 else 10 * (s + 1)), (n, s, err)
    d = g.diagnostics()
    assert d["nan_count"] == 0
    assert abs(d["u_bulk"] - kw["u_bulk"]) <= 1e-13 * abs(kw["u_bulk"])
    g.close()


def test_config5_full_size_by_xy_tiling(oracle, gpu):
    import torch
    from paper_2411_09364_b200 import inputs
    TX, TY = 8, 8
    full = inputs.config(5)["params"]
    nx, ny, nz = full["nx"] // TX, full["ny"] // TY, full["nz"]
    npts = full["nx"] * full["ny"] * full["nz"]
    _need(100 * nx * ny * nz * 8, 17 * npts * 8)
    # the small box: same dx, dy, z grid and options as config 5
    cfg = inputs.config(5, (nx, ny, nz))
    cfg["params"]["lx"] = full["lx"] / TX; cfg["params"]["ly"] = full["ly"] / TY
    u, v, w, ub = inputs.initial_fields(cfg)
    kw = inputs.solver_kwargs(cfg, ub)
    o = pc.make(oracle.Oracle, kw)
    o.set_velocity(u, v, w); o.project()
    u, v, w = o.velocity()
    kw["u_bulk"] = float(np.sum(u * o.dzf[:, None, None]) / (nx * ny * kw["lz"]))
    dt = inputs.time_step(cfg, u, v, w)
    o = pc.make(oracle.Oracle, kw)
    o.set_velocity(u, v, w)
    kwg = dict(kw, nx=full["nx"], ny=full["ny"], lx=full["lx"], ly=full["ly"])
    g = pc.make(gpu.Solver, kwg)
    for f, a in enumerate((u, v, w)):
        t = torch.from_numpy(a).cuda().repeat(1, TY, TX).contiguous()
        g.set_field(f, t)
        del t
    o.step(dt); g.step(dt)
    torch.cuda.synchronize()
    errs = {}
    for f, name in enumerate(("u", "v", "w", "p", "nut")):
        ref = o.get(f)
        if name == "p":
            ref = pc.weighted_mean_removed(ref, o.dzf)
        big = g.get_field(f)
        if name == "p":
            big -= (big.sum(dim=(1, 2)) * torch.from_numpy(o.dzf).cuda()).sum() / (full["nx"] * full["ny"] * kw["lz"])
        r = torch.from_numpy(ref).cuda()
        big = big.view(nz, TY, ny, TX, nx)
        big -= r[:, None, :, None, :]
        scale = max(float(np.max(np.abs(ref))), kw["nu"] if name == "nut" else 1e-300)
        errs[name] = float(big.abs().max()) / scale
        del big, r
    assert max(errs.values()) <= TOL_1STEP, errs
    d = g.diagnostics()
    assert d["nan_count"] == 0 and abs(d["u_bulk"] - kw["u_bulk"]) <= 1e-13 * abs(kw["u_bulk"])
    assert 3 <= d["wm_max_iters"] <= 9
    g.close()
