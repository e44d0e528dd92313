"""CPU-only checks of the boundary: libcales.so builds for sm_100a, loads, exports every symbol include/cales.h declares,
and its host-side logic (validation, workspace sizing, defaults) behaves as the header states.  No kernel is launched."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2411_09364_b200 import binding as b
    b.lib()
    return b


def test_every_declared_symbol_is_exported(binding):
    hdr = open(os.path.join(ROOT, "include", "cales.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cales_[a-z_0-9]+)\s*\(", hdr))
    assert {"cales_create", "cales_step", "cales_poisson_solve", "cales_eddy_viscosity"} <= declared   # north_star's list
    L = C.CDLL(os.path.join(ROOT, "paper_2411_09364_b200", "libcales.so"))
    for name in sorted(declared):
        getattr(L, name)                       # AttributeError if missing
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)


def test_library_is_sm100a_sass(binding):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", os.path.join(ROOT, "paper_2411_09364_b200", "libcales.so")],
                         capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_defaults_and_workspace_size(binding):
    P = binding.make_params(64, 32, 16, 1.0, 1.0, 1.0)
    assert (P.kappa, P.B, P.aplus, P.cs, P.wm_tol, P.wm_maxit, P.dsm_avg_xy_plane) == (0.41, 5.2, 25.0, 0.17, 1e-4, 50, 1)
    n = 64 * 32 * 16
    need = binding.workspace_bytes(64, 32, 16, 1.0, 1.0, 1.0)
    assert 13 * n * 8 <= need <= 14 * n * 8 + (1 << 20)         # 12 fields + Thomas scratch + small tables
    per = binding.workspace_bytes(64, 32, 16, 1.0, 1.0, 1.0, sgs_model=2, bc_z=1)
    assert per > need                                            # + |S| and the dynamic-model partial sums
    # config 5 fits 180 GB with room to spare
    big = binding.workspace_bytes(1536, 1024, 512, 1.0, 1.0, 1.0, sgs_model=2, bc_z=1, wall_model=1)
    assert 85e9 < big < 100e9


@pytest.mark.parametrize("kw,msg", [
    (dict(nx=30, ny=14), "factor into 2 and 3"),
    (dict(nx=31), "even"),
    (dict(nz=3), "too small"),
    (dict(bc_z=0, zstretch=1), "uniform"),
    (dict(wall_model=1, bc_z=0), "wall model needs z walls"),
    (dict(implicit_z=1, bc_z=0), "implicit z needs z walls"),
    (dict(van_driest=1, bc_z=0), "van Driest"),
    (dict(nu=0.0), "nu must be positive"),
    (dict(dsm_filter3d=1, sgs_model=1), "dsm_filter3d needs the dynamic model"),
    (dict(wall_model_y=1, bc_y=0), "wall model on y walls needs y walls"),
    (dict(lx=-1.0), "positive"),
])
def test_argument_errors_are_reported_at_create_time(binding, kw, msg):
    g = dict(nx=32, ny=16, nz=8, lx=1.0, ly=1.0, lz=1.0)
    opts = {}
    for k, v in kw.items():
        (g if k in g else opts)[k] = v
    assert binding.workspace_bytes(g["nx"], g["ny"], g["nz"], g["lx"], g["ly"], g["lz"], **opts) == 0
    assert msg in binding.lib().cales_last_error().decode()


def test_null_arguments_do_not_crash(binding):
    L = binding.lib()
    assert L.cales_step(None, 1.0) == 1
    assert L.cales_destroy(None) == 0
    assert L.cales_create(None, None) == 1
    h = C.c_void_p()
    P = binding.make_params(32, 16, 8, 1.0, 1.0, 1.0)          # null workspace
    assert L.cales_create(C.byref(P), C.byref(h)) == 1 and not h.value


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.CalesError):
        binding.Solver(32, 16, 8, 1.0, 1.0, 1.0)
