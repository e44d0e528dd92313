"""Parity cases shared by the host-emulator tests (CPU) and the GPU tests: reduced replicas of the five
BASELINE.json configurations with the same option sets, sized so that the oracle finishes in seconds while the
grids still span several CUDA tiles and a ragged tail (nx not a multiple of 32, ny not a multiple of 8).

Holds no arithmetic of the method: it only draws the seeded inputs (paper_2411_09364_b200.inputs), runs ONE side
and compares arrays.  The initial field is made solenoidal by the oracle's own projection.
"""
import numpy as np

from paper_2411_09364_b200 import inputs

# name -> (config number, replica shape (nx, ny, nz), steps)
SMALL = {
    "cfg1_dit": (1, (24, 16, 12), 2),
    "cfg2_wmles": (2, (48, 24, 16), 2),
    "cfg3_wrles_cn": (3, (36, 24, 20), 2),
    "cfg4_duct_dsm": (4, (48, 36, 16), 2),            # wall-row tiles + column-marching kernel
    "cfg4_duct_dsm_narrow": (4, (48, 4, 16), 1),      # ny < 6: tile kernel on every row
    "cfg5_wmles_dsm": (5, (36, 24, 16), 2),
    "duct_static_smag": (4, (24, 12, 12), 2, dict(sgs_model=1, cs=0.1)),   # static model next to y walls
    "cfg5_hwm_interp": (5, (24, 12, 16), 2, dict(h_wm=0.1)),               # wall model sampled between centres
    "cfg2_wm_implicit": (2, (24, 12, 16), 2, dict(implicit_z=1)),
    "duct_wmles_dsm": (4, (48, 24, 16), 2, dict(wall_model=1, wall_model_y=1, nu=1.0 / 40000)),   # duct WMLES: wall model on all four walls
    "duct_wmles_smag_y_only": (4, (24, 12, 12), 2, dict(wall_model_y=1, sgs_model=1, cs=0.1, nu=1.0 / 40000)),          # wall model on the y walls only, no-slip z walls
    "duct_wmles_hwm_interp": (4, (24, 12, 12), 2, dict(wall_model=1, wall_model_y=1, sgs_model=1, cs=0.1, nu=1.0 / 40000, h_wm=0.12)),   # sampled between centres on all four walls
    # 3-D box test filter (8(f) item 2): WMLES channel, no-slip duct, duct WMLES, triply periodic box
    "cfg5_dsm_filter3d": (5, (36, 24, 16), 2, dict(dsm_filter3d=1)),
    "cfg4_duct_dsm_filter3d": (4, (48, 18, 12), 2, dict(dsm_filter3d=1)),
    "duct_wmles_dsm_filter3d": (4, (36, 12, 12), 1, dict(wall_model=1, wall_model_y=1, nu=1.0 / 40000, dsm_filter3d=1)),
    "cfg1_dsm_filter3d": (1, (24, 16, 12), 2, dict(sgs_model=2, dsm_filter3d=1)),
    # nx >= 66: the register-window march with staged rows (k_dsm3_col_tma), two x blocks, periodic wrap in x and in z / walls
    "cfg5_dsm_filter3d_wide": (5, (72, 12, 12), 1, dict(dsm_filter3d=1)),
    "cfg1_dsm_filter3d_wide": (1, (72, 8, 8), 1, dict(sgs_model=2, dsm_filter3d=1)),
}
# the sizes the GPU parity tests use: several tiles in every direction plus ragged tails
GPU_CASES = {
    "cfg1_dit32": (1, None, 10),                     # BASELINE config 1 at full size, 10 steps
    "cfg2_wmles": (2, (96, 48, 32), 3),
    "cfg3_wrles_cn": (3, (96, 72, 48), 3),
    "cfg4_duct_dsm": (4, (192, 54, 48), 3),
    "cfg5_wmles_dsm": (5, (192, 128, 64), 3),        # the replica SURVEY.md 8(d) names for config 5
    "duct_static_smag": (4, (96, 36, 24), 2, dict(sgs_model=1, cs=0.1)),
    "cfg5_hwm_interp": (5, (96, 48, 32), 2, dict(h_wm=0.1)),
    "cfg4_duct_dsm_narrow": (4, (72, 4, 16), 2),
    "cfg2_wm_implicit": (2, (96, 48, 32), 3, dict(implicit_z=1)),
    "cfg5_wm_implicit_dsm": (5, (96, 48, 32), 2, dict(implicit_z=1, h_wm=0.1)),
    "duct_wmles_dsm": (4, (192, 54, 48), 3, dict(wall_model=1, wall_model_y=1, nu=1.0 / 40000)),
    "duct_wmles_smag_implicit": (4, (96, 36, 24), 2, dict(wall_model=1, wall_model_y=1, sgs_model=1, cs=0.1, implicit_z=1, nu=1.0 / 40000)),
    "duct_wmles_hwm_interp": (4, (96, 36, 24), 2, dict(wall_model=1, wall_model_y=1, nu=1.0 / 40000, h_wm=0.12)),
    "cfg5_dsm_filter3d": (5, (96, 54, 32), 3, dict(dsm_filter3d=1)),
    "cfg4_duct_dsm_filter3d": (4, (72, 36, 24), 2, dict(dsm_filter3d=1)),
    "duct_wmles_dsm_filter3d": (4, (72, 36, 24), 2, dict(wall_model=1, wall_model_y=1, nu=1.0 / 40000, dsm_filter3d=1)),
    "cfg1_dsm_filter3d": (1, None, 3, dict(sgs_model=2, dsm_filter3d=1)),
    # fully implicit Crank-Nicolson (8(f) item 3, Eq. 17-19): triply periodic box, tanh channel with van Driest + forcing,
    # wall-modelled channel (wall model restricted to the z walls)
    "cfg1_implicit_xyz": (1, None, 3, dict(implicit_xyz=1)),
    "cfg3_implicit_xyz": (3, (96, 72, 48), 3, dict(implicit_z=0, implicit_xyz=1)),
    "cfg2_wm_implicit_xyz": (2, (96, 48, 32), 2, dict(implicit_xyz=1)),
    "cfg5_dsm_implicit_xyz": (5, (96, 48, 32), 2, dict(implicit_xyz=1, h_wm=0.1)),
}


def prepare(oracle, n, shape, overrides=None):
    """(cfg, kwargs, (u, v, w), dt): seeded field, projected by the oracle, with its time step."""
    cfg = inputs.config(n, shape)
    u, v, w, ub = inputs.initial_fields(cfg)
    kw = inputs.solver_kwargs(cfg, ub)
    kw.update(overrides or {})
    g = {k: kw[k] for k in ("nx", "ny", "nz", "lx", "ly", "lz")}
    o = oracle.Oracle(g["nx"], g["ny"], g["nz"], g["lx"], g["ly"], g["lz"],
                      **{k: v_ for k, v_ in kw.items() if k not in g})
    o.set_velocity(u, v, w)
    o.project()
    u, v, w = o.velocity()
    if kw["const_flow_rate"]:
        # the projection leaves the bulk velocity unchanged in periodic x; keep the imposed value consistent
        kw["u_bulk"] = float(np.sum(u * o.dzf[:, None, None]) / (g["nx"] * g["ny"] * g["lz"]))
    dt = inputs.time_step(cfg, u, v, w)
    return cfg, kw, (u, v, w), dt


def make(cls, kw):
    g = {k: kw[k] for k in ("nx", "ny", "nz", "lx", "ly", "lz")}
    return cls(g["nx"], g["ny"], g["nz"], g["lx"], g["ly"], g["lz"], **{k: v for k, v in kw.items() if k not in g})


def weighted_mean_removed(p, dzf):
    m = np.sum(p * dzf[:, None, None]) / (np.sum(dzf) * p.shape[1] * p.shape[2])
    return p - m


def field_errors(got, ref, dzf, nu):
    """max|delta| / max|field| for u, v, w, p (weighted mean removed), nu_t (scale max(nu_t) or nu)."""
    out = {}
    for name, a, b in zip("uvw", got[:3], ref[:3]):
        out[name] = float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))
    pa, pb = weighted_mean_removed(got[3], dzf), weighted_mean_removed(ref[3], dzf)
    out["p"] = float(np.max(np.abs(pa - pb)) / max(np.max(np.abs(pb)), 1e-300))
    sc = max(float(np.max(np.abs(ref[4]))), nu)
    out["nut"] = float(np.max(np.abs(got[4] - ref[4])) / sc)
    return out
