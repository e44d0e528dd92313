"""Mutation check of the oracle pins: every plausible single-line mistake listed below is injected into a COPY of
oracle/cales_oracle.cpp, the copy is built, and tests/test_oracle_pins.py is run against it; at least the pin named
beside the mutant must turn red.  M1-M6 are the mistakes the round-1 review found already caught, M7-M12 the six it
found surviving (config-3 and config-4 arithmetic: Eq. 22, tanh-grid metrics, x-line averaging, total-viscosity clip);
the pins that kill those were added in round 2; M13-M16 are mistakes in the fully implicit scheme (Eq. 17-19) added in round 2.  Test infrastructure only; nothing here touches the CUDA path.
"""
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "cales_oracle.cpp")

# (id, text in the source, replacement, pin that must fail)
MUTANTS = [
    ("M1_rk_alpha", "const double al[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};", "const double al[3] = {8.0 / 15.0, 5.0 / 13.0, 3.0 / 4.0};",
     "test_rk3_coefficients_and_third_order"),
    ("M2_advection_doubled", "au[S.id(i, j, k)] = -((uxp * uxp", "au[S.id(i, j, k)] = -2.0 * ((uxp * uxp",
     "test_advection_vs_numpy_stencil"),
    ("M3_alpha_grad_p", "be * S.Ru[n] - ga * gpx", "be * S.Ru[n] - al * gpx", "test_taylor_green_decay"),
    ("M4_two_point_edge_viscosity", "double ne = 0.25 * (nt(i, j, k) + nt(i + 1, j, k) + nt(i, j + 1, k) + nt(i + 1, j + 1, k));",
     "double ne = 0.5 * (nt(i, j, k) + nt(i + 1, j + 1, k));", "test_sgs_fluxes_telescope"),
    ("M5_two_point_wall_model_interpolation",
     "b = 0.25 * (at(S.v, i, j) + at(S.v, i + 1, j) + at(S.v, i, j - 1) + at(S.v, i + 1, j - 1)); }\n        else { a = at(S.v, i, j);",
     "b = 0.5 * (at(S.v, i, j) + at(S.v, i + 1, j - 1)); }\n        else { a = at(S.v, i, j);",
     "test_wall_model_on_y_walls_is_the_z_wall_model_rotated"),
    ("M6_alpha_not_reduced_on_y_wall_rows", "if (!(S.P.bc_y == BC_WALL && (j == 0 || j == ny - 1))) ++nf;", "++nf;",
     "test_3d_filter_first_layer_rule_and_filter_ratio"),
    ("M7_eq22_term_dropped", "S.p(i, j, k) += ph(i, j, k) - (imp ? cimp * lzz : 0.0) -", "S.p(i, j, k) += ph(i, j, k) -",
     "test_pressure_update_eq22_on_tanh_grid"),
    ("M8_diffusion_z_metrics_swapped",
     "lz = ((u(i, j, k + 1) - u(i, j, k)) / S.dzc(k) - (u(i, j, k) - u(i, j, k - 1)) / S.dzc(k - 1)) / S.dzf(k);\n    du[n]",
     "lz = ((u(i, j, k + 1) - u(i, j, k)) / S.dzc(k - 1) - (u(i, j, k) - u(i, j, k - 1)) / S.dzc(k)) / S.dzf(k);\n    du[n]",
     "test_diffusion_vs_numpy_stencil"),
    ("M9_cn_matrix_uv_metrics_swapped", "double ak = 1.0 / (S.dzf(k) * S.dzc(k - 1)), ck = 1.0 / (S.dzf(k) * S.dzc(k));\n            a[k] = -cimp * ak;",
     "double ak = 1.0 / (S.dzf(k) * S.dzc(k)), ck = 1.0 / (S.dzf(k) * S.dzc(k - 1));\n            a[k] = -cimp * ak;",
     "test_crank_nicolson_dense_matrix_on_tanh_grid"),
    ("M10_cn_matrix_w_metrics_swapped", "double ak = 1.0 / (S.dzc(k) * S.dzf(k)), ck = 1.0 / (S.dzc(k) * S.dzf(k + 1));",
     "double ak = 1.0 / (S.dzc(k) * S.dzf(k + 1)), ck = 1.0 / (S.dzc(k) * S.dzf(k));", "test_crank_nicolson_dense_matrix_on_tanh_grid"),
    ("M11_x_line_coefficient_mirrored_row", "if (!per_plane) S.cs[(size_t)k * ny + j] = (mm > 0.0) ? ll / mm : 0.0;",
     "if (!per_plane) S.cs[(size_t)k * ny + (ny - 1 - j)] = (mm > 0.0) ? ll / mm : 0.0;", "test_dynamic_coefficient_per_x_line_vs_dense_bruteforce"),
    ("M13_eq19_xy_part_dropped", "- (imp3 ? cimp * (lxy + lzz) : 0.0);", "- (imp3 ? cimp * lzz : 0.0);", "test_pressure_update_eq19"),
    ("M14_helmholtz_wall_closure_sign", "double sg = S.P.wall_model ? -1.0 : 1.0;", "double sg = S.P.wall_model ? 1.0 : -1.0;", "test_helmholtz_manufactured_discrete"),
    ("M15_eq17_diffusion_counted_in_R", "double Ru = au[n] + su[n] + (imp3 ? 0.0 : dxu[n])", "double Ru = au[n] + su[n] + dxu[n]", "test_fully_implicit_ustar_is_the_helmholtz_solution"),
    ("M16_helmholtz_w_metrics_swapped", "else { ak = 1.0 / (S.dzc(k) * S.dzf(k)); ck = 1.0 / (S.dzc(k) * S.dzf(k + 1)); }", "else { ak = 1.0 / (S.dzc(k) * S.dzf(k + 1)); ck = 1.0 / (S.dzc(k) * S.dzf(k)); }", "test_helmholtz_manufactured_discrete"),
    ("M12_total_clip_floor_halved", "nut[n] = (t < -nu) ? -nu : t;", "nut[n] = (t < -0.5 * nu) ? -0.5 * nu : t;", "test_total_viscosity_clip_floor_binds"),
]


def _run_mutant(args):
    mid, old, new, pin, tmp = args
    src = open(SRC).read()
    if src.count(old) != 1:
        return mid, "source text not found exactly once", ""
    msrc = os.path.join(tmp, mid + ".cpp")
    lib = os.path.join(tmp, mid + ".so")
    with open(msrc, "w") as f:
        f.write(src.replace(old, new))
    cmd = ["g++", "-std=c++17", "-O1", "-fopenmp", "-fPIC", "-shared", "-I", os.path.join(ROOT, "oracle"), "-o", lib, msrc]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        return mid, "mutant does not compile: " + r.stderr[-400:], ""
    env = dict(os.environ, CALES_ORACLE_LIB=lib, OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-q", "-k", pin,
                        "-p", "no:cacheprovider"], capture_output=True, text=True, env=env, cwd=ROOT)
    return mid, None, r.stdout[-1500:] if r.returncode == 0 else "KILLED"


def test_every_listed_mutant_is_killed_by_its_pin():
    with tempfile.TemporaryDirectory() as tmp:
        with ThreadPoolExecutor(max_workers=4) as ex:
            results = list(ex.map(_run_mutant, [m + (tmp,) for m in MUTANTS]))
    survivors = []
    for mid, err, out in results:
        assert err is None, (mid, err)
        if out != "KILLED":
            survivors.append((mid, out))
    assert not survivors, survivors


def test_mutation_harness_would_notice_a_green_run():
    """The harness reports a mutant that changes nothing (a comment) as a survivor."""
    with tempfile.TemporaryDirectory() as tmp:
        mid, err, out = _run_mutant(("M0_noop", "// O-step 7b: Eq. 12", "// O-step 7b: Eq. 12 ", "test_thomas_vs_dense", tmp))
    assert err is None and out != "KILLED"
