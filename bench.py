#!/usr/bin/env python
"""bench.py -- throughput of the CaLES hot path (one full RK3 step = all rows of SURVEY.md 8(a)) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

Prints ONE JSON line (rank 0).  metric = fp64 grid-point RK3 steps per second (Gpts*step/s).
  value     : N_points * K / t with the state resident in HBM (CUDA events on the launching stream, max over ranks)
  e2e       : same metric through the C ABI with HOST buffers: every step copies u, v, w host->device
              (cales_set_field), steps, and copies u, v, w, p device->host (cales_get_field)
  roofline  : the dominant kernel of the step, algorithmic bytes / its mean launch duration (events recorded by the
              library after every launch inside the timed region) against MEASURED_PEAKS.json's HBM copy rate
  kernels   : the same figure for every kernel of the step
  cpu_baseline : the CPU oracle as it stands on the host cores, on a bounded replica of the same option set
Multi-GPU: replicas only: every rank steps its own simulation, no collective on the data path.
`--impl reference` times the oracle (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 grid-point RK3 steps/sec (Gpts*step/s)"
UNIT = "Gpts*step/s"
L2_BYTES = 126 * 1024 * 1024

# Algorithmic bytes per grid point per LAUNCH (fp64; every field a kernel needs read once, every result written once;
# DESIGN.md "Kernels and their rooflines").  k_rhs: substeps read 5 (+3 R^{k-1}) fields and write
# 3 (+3 R^k): 88 / 112 / 88 B/pt, mean 96.
ALGO_BYTES = {
    "k_rhs": 96.0, "k_cn_z": 48.0, "k_fft_x_fwd": 32.0, "k_fft_y_fwd": 16.0, "k_poisson_z": 16.0, "k_fft_y_inv": 16.0,
    "k_fft_x_inv": 16.0, "k_correct": 72.0, "k_smag": 32.0, "k_dsm_col": 32.0, "k_dsm_nut": 16.0, "k_fill": 8.0,
    "k_dsm3_pass1": 32.0,
}


# fp64 operations per grid point of the one kernel that is bound by the plain fp64 ALUs rather than by HBM (ncu instruction counts of
# round 2, profiles/r2_ncu_dsm.md: 95 DFMA + 69 DADD + 55 DMUL = 219 fp64 instructions per point; an FMA counts 2).
ALGO_FLOPS = {"k_dsm_col": 314.0}
# Algorithmic bytes per grid point and RK3 step of SURVEY.md 8(d)'s pass structure (296 B/pt per substep with the static model and
# explicit diffusion; +16 per substep for the two-pass dynamic model; +48 per substep for the Crank-Nicolson z solves): the yardstick
# the whole step is measured with, whatever passes this implementation fuses away.
SURVEY_STEP_BYTES = {1: 888.0, 2: 888.0, 3: 1032.0, 4: 936.0, 5: 936.0}
SPLIT_KERNELS = {"k_dsm_col"}      # names whose launches of one substep share the grid between them
# fallback if the in-process measurement (cales_fp64_peak) fails: 148 SMs x 64 FMA lanes x 2 flop x 1.965 GHz
FP64_PEAK_TFLOPS_DERIVED = 148 * 64 * 2 * 1.965e9 / 1e12
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_ncu_traffic.csv")


def ncu_traffic():
    """{(config, kernel): (dram bytes per launch, source)} from the committed ncu --set full capture (profiles/r2_ncu_traffic.csv,
    made by the command in profiles/r2b_ncu_full.md): dram__bytes_read.sum + dram__bytes_write.sum, averaged over the launches
    of that kernel in the capture."""
    out = {}
    try:
        with open(TRAFFIC_CSV) as f:
            for line in f:
                if line.startswith("#") or not line.strip() or line.startswith("config,"):
                    continue
                c, k, rd, wr = line.strip().split(",")[:4]
                out[(int(c), k)] = (float(rd) + float(wr), "profiles/r2_ncu_traffic.csv (ncu --set full, see profiles/r2b_ncu_full.md)")
    except OSError:
        pass
    return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True); self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


REPLICA = {1: None, 2: None, 3: (128, 128, 96), 4: (256, 64, 64), 5: (192, 128, 128)}   # bounded oracle samples (seconds each)


def oracle_leg(cfg_no, steps, warmup, overrides=None):
    """Time the CPU oracle as it stands (never tuned for this) on a bounded replica of config cfg_no's option set."""
    import numpy as np
    import oracle
    from paper_2411_09364_b200 import inputs
    shape = REPLICA[cfg_no]
    cfg = inputs.config(cfg_no, shape)
    u, v, w, ub = inputs.initial_fields(cfg)
    kw = inputs.solver_kwargs(cfg, ub)
    kw.update(overrides or {})
    g = {k: kw.pop(k) for k in ("nx", "ny", "nz", "lx", "ly", "lz")}
    o = oracle.Oracle(g["nx"], g["ny"], g["nz"], g["lx"], g["ly"], g["lz"], **kw)
    o.set_velocity(u, v, w); o.project()
    dt = inputs.time_step(cfg, *o.velocity())
    for _ in range(warmup):
        o.step(dt)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(dt)
    t = time.perf_counter() - t0
    npts = g["nx"] * g["ny"] * g["nz"]
    assert np.isfinite(o.get(0)).all()
    return {"value": npts * steps / t / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "config %d option set on a %dx%dx%d grid (%s), %d steps after %d warm-up" %
                      (cfg_no, g["nx"], g["ny"], g["nz"], "full size" if shape is None else "reduced replica", steps, warmup),
            "ms_per_step": 1e3 * t / steps, "workload": cfg["name"]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg_no = args.config or 5
    steps, warmup = args.steps, args.warmup
    if REPLICA[cfg_no] is not None:            # keep the whole run within a few minutes on a small host
        steps, warmup = min(steps, 5), min(warmup, 1)
    r = oracle_leg(cfg_no, steps, warmup, {"dsm_filter3d": 1} if args.dsm_filter3d else None)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": r["workload"], "sample": r["sample"]},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def pick_config(torch, requested, ranks_on_node=1):
    """Config 5 (the largest single-GPU workload) when the device and the host have room for it, else config 4."""
    if requested:
        return requested
    import psutil
    free, _ = torch.cuda.mem_get_info()
    host = psutil.virtual_memory().available
    # config 5: 15 resident fields x 6.44 GB on the device; per rank 4 pinned host fields + generation temporaries (~50 GB)
    if free >= 110e9 and host >= 60e9 * ranks_on_node + 30e9:
        return 5
    return 4


def host_register(torch, a):
    """Pin an existing numpy array in place (no copy) so the e2e copies run from pinned host memory."""
    rc = torch.cuda.cudart().cudaHostRegister(a.ctypes.data, a.nbytes, 0)
    return int(rc) == 0


def max_over_ranks(x, device):
    """MAX of a python float over the ranks of the default process group (identity when there is none).  The only
    collective of the multi-GPU bench: replicas share no data."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(npts_per_rank, steps, world, max_ms):
    """Whole-job Gpts*step/s of `world` replicas that each advanced npts_per_rank points by `steps` steps."""
    return world * npts_per_rank * steps / (max_ms * 1e-3) / 1e9


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2411_09364_b200 import binding, inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CaLES hot path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()
    cfg_no = pick_config(torch, args.config, int(os.environ.get("LOCAL_WORLD_SIZE", str(world))))
    if world > 1:                    # every replica runs the same workload: rank 0 decides
        box = [cfg_no]
        dist.broadcast_object_list(box, src=0)
        cfg_no = int(box[0])
    K, W = args.steps, max(args.warmup, 3)

    # ---- seeded synthetic workload (inputs.py), every rank its own replica (seed + rank)
    cfg = inputs.config(cfg_no)
    cfg["seed"] += rank
    t_gen = time.perf_counter()
    u, v, w, ub = inputs.initial_fields(cfg)
    dt = inputs.time_step(cfg, u, v, w)
    kw = inputs.solver_kwargs(cfg, ub)
    if args.dsm_filter3d:
        if kw["sgs_model"] != 2:
            raise SystemExit("--dsm-filter3d needs a dynamic-model workload (config 4 or 5)")
        kw["dsm_filter3d"] = 1
        cfg["name"] += " + 3-D box test filter"
    g = {k: kw.pop(k) for k in ("nx", "ny", "nz", "lx", "ly", "lz")}
    npts = g["nx"] * g["ny"] * g["nz"]
    p_host = np.zeros_like(u)
    pinned = all(host_register(torch, a) for a in (u, v, w, p_host))
    t_gen = time.perf_counter() - t_gen
    # a dedicated (non-default) stream: everything below -- the solver's kernels, torch's L2 flush, the CUDA events -- is
    # issued on it, and cales_step can capture its substeps into a CUDA graph (the legacy default stream cannot be captured)
    stream = torch.cuda.Stream(device=local)
    torch.cuda.set_stream(stream)
    s = binding.Solver(g["nx"], g["ny"], g["nz"], g["lx"], g["ly"], g["lz"], device=local, stream=stream, **kw)
    for kv in args.option:
        key, val = kv.split("=")
        s.set_option(key, int(val))
    s.set_velocity(u, v, w)
    s.project()                      # discretely solenoidal start, by the GPU solver itself
    for f, a in zip(range(3), (u, v, w)):
        s.get_field(f, torch.from_numpy(a))       # the host copies now hold the projected field
    flush = None
    small = s.workspace_bytes < 2 * L2_BYTES
    if small:
        flush = torch.empty(2 * L2_BYTES // 8, dtype=torch.float64, device="cuda")
    big = npts >= 4_000_000
    for _ in range(W):
        s.step(dt)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()

    # ---- timed region: K steps, CUDA events on the launching stream (the solver runs on torch's current stream)
    ktot = {}
    def add_kernel_times():
        for name, (ms, n) in s.kernel_times().items():
            a = ktot.setdefault(name, [0.0, 0]); a[0] += ms; a[1] += n
    sampler = ClockSampler(local); sampler.start()
    try:
        fp64_peak, fp64_src = s.fp64_peak(), "measured in this process (cales_fp64_peak: register-resident DFMA loop, best of 3)"
    except Exception as e:       # keep the line
        fp64_peak, fp64_src = FP64_PEAK_TFLOPS_DERIVED, "derived 148 x 64 x 2 x 1.965 GHz (measurement failed: %r)" % (e,)
    s.set_timing(big)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for k in range(K):
        if flush is not None:
            flush.fill_(float(k))    # L2 flush between timed iterations (small configs only)
        ev[k][0].record()
        s.step(dt)
        ev[k][1].record()
        if big:
            add_kernel_times()       # per-launch events of this step -> per-kernel totals (syncs, outside the event pair)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    if not big:                      # launch-bound sizes: per-launch events would perturb the timed region; second pass
        s.set_timing(True)
        for k in range(K):
            if flush is not None:
                flush.fill_(float(k))
            s.step(dt); add_kernel_times()
    s.set_timing(False)
    diag = s.diagnostics()
    launches = s.launches_per_step() * K
    ms = max_over_ranks(ms, "cuda")
    value = aggregate_value(npts, K, world, ms)

    # ---- e2e: the same metric with HOST buffers: every step uploads that step's input velocity (3 fields) from pinned host memory and
    # downloads the step's result (u, v, w, p); both copies are inside the timed region.  The three stages are pipelined the way a
    # user streaming fields through the solver would: H2D of step n+1 (copy stream) and D2H of step n-1 (second copy stream) run
    # while step n computes; device staging tensors decouple them from the solver state, which is read and written through the
    # C ABI (cales_set_field / cales_step / cales_get_field with device pointers).  PCIe is full duplex, so the steady state is
    # max(H2D, D2H, compute + 7 field copies on the device).
    Ke = max(1, min(K, 8)) if not args.no_e2e else 0
    e2e = None
    if Ke:
        free, _ = torch.cuda.mem_get_info()
        staged = free > 8 * npts * 8 + (2 << 30)
        hosts = [torch.from_numpy(a) for a in (u, v, w, p_host)]
        if staged:
            st_in = [torch.empty(s.shape, dtype=torch.float64, device="cuda") for _ in range(3)]
            st_out = [torch.empty(s.shape, dtype=torch.float64, device="cuda") for _ in range(4)]
            h2d, d2h = torch.cuda.Stream(device=local), torch.cuda.Stream(device=local)
            in_ready, in_free = torch.cuda.Event(), torch.cuda.Event()
            out_ready, out_free = torch.cuda.Event(), torch.cuda.Event()
            in_free.record(stream); out_free.record(stream)
            def upload():
                with torch.cuda.stream(h2d):
                    h2d.wait_event(in_free)
                    for f in range(3):
                        st_in[f].copy_(hosts[f], non_blocking=True)
                    in_ready.record(h2d)
            def e2e_step(last):
                stream.wait_event(in_ready)
                for f in range(3):
                    s.set_field(f, st_in[f])
                in_free.record(stream)
                if not last:
                    upload()                        # the next step's input travels while this step computes
                s.step(dt)
                stream.wait_event(out_free)
                for f in range(4):
                    s.get_field(f, st_out[f])
                out_ready.record(stream)
                with torch.cuda.stream(d2h):
                    d2h.wait_event(out_ready)
                    for f in range(4):
                        hosts[f].copy_(st_out[f], non_blocking=True)
                    out_free.record(d2h)
            def e2e_run(n):
                upload()
                for q in range(n):
                    e2e_step(q == n - 1)
                torch.cuda.synchronize()
        else:
            def e2e_run(n):
                for _ in range(n):
                    for f in range(3):
                        s.set_field(f, hosts[f])        # H2D, synchronous (cales_set_field with a host pointer)
                    s.step(dt)
                    for f in range(4):
                        s.get_field(f, hosts[f])        # D2H of the step's result
                torch.cuda.synchronize()
        e2e_run(1)                              # warm-up
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        e2e_run(Ke)
        te = time.perf_counter() - t0
        te = max_over_ranks(te, "cuda")
        e2e = {"value": aggregate_value(npts, Ke, world, te * 1e3), "unit": UNIT, "h2d_bytes_per_step": 3 * npts * 8, "d2h_bytes_per_step": 4 * npts * 8,
               "steps": Ke, "ms_per_step": 1e3 * te / Ke, "host_memory": "pinned (cudaHostRegister)" if pinned else "pageable",
               "pipeline": "H2D / compute / D2H overlapped on three streams through device staging tensors" if staged else "sequential (no room for staging)",
               "note": "each step: upload u,v,w from host, cales_set_field x3, cales_step, cales_get_field x4, download u,v,w,p to host; a new "
                       "velocity makes the library re-evaluate the wall stress and nu_t first; wall time over the Ke steps including the "
                       "pipeline fill and drain"}
        if staged:
            del st_in, st_out
        del hosts

    # ---- per-kernel roofline table (algorithmic bytes / mean launch duration) and the dominant kernel
    peak, peak_src = measured_peaks()
    traffic = ncu_traffic()
    kernels = {}
    step_ms = sum(a[0] for a in ktot.values()) / K
    for name, (tot, n) in sorted(ktot.items(), key=lambda kv: -kv[1][0]):
        per = tot / n
        row = {"ms_per_launch": per, "launches_per_step": n // K, "share_of_step": (tot / K) / step_ms if step_ms else None}
        # a kernel name launched more than once per substep (k_dsm_col: the staged march on the inner planes + the direct-load march on
        # the two wall planes) covers the grid ONCE per substep with all its launches together: its per-launch share of the work
        cover = 3.0 / max(n // K, 1) if (name in SPLIT_KERNELS and (n // K) > 3) else 1.0
        row["grid_fraction_per_launch"] = cover
        if name in ALGO_BYTES:
            gbs = ALGO_BYTES[name] * cover * npts / (per * 1e-3) / 1e9
            row.update({"algo_bytes_per_pt": ALGO_BYTES[name], "achieved_gbs": gbs, "frac": gbs / peak})
        if name in ALGO_FLOPS:       # the kernel bound by the plain fp64 ALUs: also against the fp64 peak measured in this process
            tf = ALGO_FLOPS[name] * cover * npts / (per * 1e-3) / 1e12
            row.update({"algo_flops_per_pt": ALGO_FLOPS[name], "achieved_tflops": tf, "fp64_frac": tf / fp64_peak})
        if (cfg_no, name) in traffic:
            row["ncu_dram_bytes_per_launch"] = traffic[(cfg_no, name)][0]
        kernels[name] = row
    # the dominant kernel = the largest total time per step among the kernels of the byte model (a kernel launched twice per
    # substep, like k_dsm_col with its wall planes, counts with both launches)
    top = next((n for n in kernels if n in ALGO_BYTES), None)
    roofline = None
    if top:
        r = kernels[top]
        tr = traffic.get((cfg_no, top))
        roofline = {"kernel": top, "bound": "hbm", "achieved": r["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": r["frac"],
                    "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None, "peak_source": peak_src,
                    "algo_bytes_per_launch": ALGO_BYTES[top] * r["grid_fraction_per_launch"] * npts, "ms_per_launch": r["ms_per_launch"],
                    "share_of_step": r["share_of_step"]}
        if top in ALGO_FLOPS:        # bound by the plain fp64 ALUs, not by HBM: report it against that peak
            roofline.update({"bound": "alu", "achieved": r["achieved_tflops"], "peak": fp64_peak, "unit": "TFLOP/s", "frac": r["fp64_frac"],
                             "peak_source": fp64_src, "algo_flops_per_launch": ALGO_FLOPS[top] * r["grid_fraction_per_launch"] * npts, "hbm_frac_of_measured_peak": r["frac"]})
    # whole-step algorithmic traffic: the sum over the step's launches of the table above
    step_bytes = sum(ALGO_BYTES.get(n, 0.0) * (a[1] // K) * kernels[n]["grid_fraction_per_launch"] for n, a in ktot.items()) * npts
    step_gbs = step_bytes / (ms / K * 1e-3) / 1e9
    survey_gbs = SURVEY_STEP_BYTES[cfg_no] * npts / (ms / K * 1e-3) / 1e9

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config %d: %s %dx%dx%d" % (cfg_no, cfg["name"], g["nx"], g["ny"], g["nz"]), "points": npts,
                       "dt": dt, "parallelism": "replicas x%d (no data-path collective)" % world,
                       "launch": "cales_step replays one CUDA graph per step" if not big else "plain stream launches (per-kernel events on)",
                       "l2": "L2 flushed between timed steps" if small else "state (%.1f GB) larger than L2" % (s.workspace_bytes / 1e9),
                       "options": {k: kw[k] for k in ("bc_y", "bc_z", "zstretch", "sgs_model", "wall_model", "implicit_z", "const_flow_rate",
                                                      "dsm_avg_xy_plane", "dsm_clip_total", "van_driest")},
                       "kernel_options": args.option or "defaults"},
            "step_hbm": {"algo_bytes_per_pt_step": SURVEY_STEP_BYTES[cfg_no], "achieved_gbs": survey_gbs, "frac_of_measured_peak": survey_gbs / peak,
                         "frac_of_8TBs": survey_gbs / 8000.0, "model": "SURVEY.md 8(d) bytes per point and step x points / measured step time",
                         "own_passes_bytes_per_pt_step": step_bytes / npts, "own_passes_frac_of_measured_peak": step_gbs / peak},
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "kernels": kernels,
            "fp64_peak": {"tflops": fp64_peak, "source": fp64_src, "derived_for_comparison": FP64_PEAK_TFLOPS_DERIVED},
            "diagnostics": {k: diag[k] for k in ("max_div", "u_bulk", "kinetic_energy", "wm_max_iters", "nan_count")},
            "input_generation_s": t_gen}
    s.close()
    del s
    torch.cuda.empty_cache()
    if world > 1:
        dist.destroy_process_group()
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            r = oracle_leg(cfg_no, 2, 1, {"dsm_filter3d": 1} if args.dsm_filter3d else None)
            line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        if not args.no_other_configs and world == 1:
            # north_star: all five workloads at 1 GPU.  The other four run as short child processes of this same script
            # (device-resident timing only) after this process has released its device memory.
            for a in (u, v, w, p_host):
                torch.cuda.cudart().cudaHostUnregister(a.ctypes.data)
            del u, v, w, p_host
            others = {}
            for cno in (1, 2, 3, 4, 5):
                if cno == cfg_no:
                    continue
                cmd = [sys.executable, os.path.abspath(__file__), "--config", str(cno), "--steps", "5", "--warmup", "3",
                       "--no-cpu-baseline", "--no-other-configs", "--no-e2e"]
                try:
                    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
                    d = json.loads(out.stdout.strip().splitlines()[-1])
                    others["config %d" % cno] = {"workload": d["config"]["workload"], "value": d["value"], "unit": UNIT,
                                                 "ms_per_step": d["ms_per_step"], "launch": d["config"]["launch"], "l2": d["config"]["l2"],
                                                 "step_hbm_frac_of_measured_peak": d["step_hbm"]["frac_of_measured_peak"],
                                                 "top_kernels": {k: round(v["share_of_step"], 3) for k, v in list(d["kernels"].items())[:3]}}
                except Exception as e:      # a failed side run must not lose the main line
                    others["config %d" % cno] = {"error": repr(e)[:200]}
                if not args.no_cpu_baseline:      # the oracle timed on every workload (bounded replicas, two steps)
                    try:
                        r = oracle_leg(cno, 2, 1)
                        others["config %d" % cno]["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
                    except Exception as e:
                        others["config %d" % cno]["cpu_baseline"] = {"error": repr(e)[:200]}
            line["other_configs"] = others
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=0, help="BASELINE.json config 1..5 (default: 5 if it fits, else 4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short side runs of the other four workloads")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=VALUE",
                    help="cales_set_option knob for A/B timing (e.g. dsm_col_variant=2, rhs_variant=0, lazy_nut=0); repeatable")
    ap.add_argument("--dsm-filter3d", action="store_true", help="configs 4, 5 with the 3-D box test filter of PAPER.md:128 (SURVEY.md 8(f) item 2); "
                    "not a BASELINE.json workload: the line is labelled and is for the widening table of DESIGN.md only")
    args = ap.parse_args()
    if args.impl == "reference":
        if not args.config:
            try:
                import torch
                args.config = pick_config(torch, 0) if torch.cuda.is_available() else 5
            except Exception:
                args.config = 5
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
