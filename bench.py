#!/usr/bin/env python
"""bench.py - price evaluations per second of the VMAT beamlet-price path on B200.

One "step" = one whole price evaluation (d = D x -> F, g -> p = D^T g -> leaf-row openings -> best
control point) on a fresh fluence vector x, through the C ABI
(`vmat_price_eval`).  Inputs are synthetic (synth/), shaped like BASELINE.json `configs`.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config {0,1,2,3,4}] [--scale S] [--impl reference]

Prints ONE JSON line (rank 0).  Multi-GPU: the path does not need a second GPU (BASELINE.json
north_star), so N > 1 runs N independent replicas, one process per GPU ("replicas only", weak scaling).
`--impl reference` times the CPU oracle (oracle/) on the host cores: the whole matrix when K + W evaluations fit the time
budget (the all-cores variant for config 3), else an evenly spaced sample of control points (angle blocks).
"""
from __future__ import annotations

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

import numpy as np
import torch

import synth

METRIC = "beamlet-price evaluations/sec"
UNIT = "evals/s"


# ----------------------------------------------------------------------------- helpers
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.proc, self.lines = gpu_index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


NCU_CAPTURES = ["r3_ncu_full_cfg2.csv", "r2_ncu_full_cfg3_sm_affine.csv", "r2_ncu_full_cfg3.csv", "r1_ncu_full_cfg3_v6.csv",
                "r1_ncu_full_cfg3_v4.csv"]                                           # newest first


def ncu_traffic(kernel_prefix: str, grid: int, algorithmic_bytes: int):
    """dram bytes (read + write) per launch of the dominant kernel from a committed `ncu --set full` capture under
    profiles/ - but only from a capture of THIS launch: its grid size must equal the running handle's and its bytes
    must lie within [0.9, 1.3] x the algorithmic bytes.  Returns (bytes or None, source or the reason for None)."""
    import csv
    why = "no committed ncu capture of this kernel"
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for name in NCU_CAPTURES:
        path = os.path.join(ROOT, "profiles", name)
        if not os.path.exists(path):
            continue
        try:
            rows = [r for r in csv.reader(open(path)) if len(r) > 3]
            hdr, units = rows[0], rows[1]
            for r in rows[2:]:
                if kernel_prefix not in r[hdr.index("Kernel Name")]:
                    continue
                g = int(r[hdr.index("Grid Size")].strip("() ").split(",")[0])
                if g != grid:
                    why = f"profiles/{name}: captured grid {g} != this launch's {grid} (another layout or workload)"
                    continue
                tot = 0.0
                for col in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    i = hdr.index(col)
                    tot += float(r[i]) * mult[units[i]]
                if not 0.9 * algorithmic_bytes <= tot <= 1.3 * algorithmic_bytes:
                    why = f"profiles/{name}: captured {tot:.4g} B is not this launch ({algorithmic_bytes} algorithmic bytes)"
                    continue
                return tot, f"profiles/{name} (ncu --set full, one launch; grid {g} matches this run)"
        except Exception as e:                                # a malformed file is a reason, not a crash
            why = f"profiles/{name}: {e}"
    return None, why


def rank_eval_index(rank: int, k: int) -> int:
    """Fluence draw index of step k on `rank`: every replica prices its own sequence of x vectors."""
    return rank * 100000 + k


def reduce_max(values, dist, device):
    """Max over ranks of per-rank device times (dist = torch.distributed or None for one rank)."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def aggregate(world: int, steps: int, elapsed_ms: float) -> dict:
    """Whole-job throughput: all ranks' evaluations over the slowest rank's time."""
    return {"value": world * steps / (elapsed_ms * 1e-3), "ms_per_step": elapsed_ms / steps}


def phantom_arrays_host(ph):
    return dict(vox=ph.coo_voxel.cpu().numpy(), beam=ph.coo_beamlet.cpu().numpy(), val=ph.coo_val.cpu().numpy(),
                n_v=ph.n_voxels, n_b=ph.n_beamlets, sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(),
                wo=ph.struct_w_over.numpy(), wu=ph.struct_w_under.numpy(), lco=ph.leafrow_col_offset.numpy(),
                aro=ph.angle_row_offset.numpy())


# ----------------------------------------------------------------------------- the CPU oracle, timed
ORACLE_KINDS = {
    "oracle": "oracle (oracle/vmat_oracle.c, plain single-thread FP64 loops over the COO triplets)",
    "oracle_mt": "oracle_mt (oracle/vmat_oracle_mt.c: the same C functions, every thread on its share of the triplets / "
                 "voxels / leaf rows, PAPER.md L191)",
}


def host_ram_available() -> int:
    try:
        import psutil
        return int(psutil.virtual_memory().available)
    except Exception:
        return 0


def oracle_probe(spec, gen_device):
    """Seconds of the single-thread oracle per control point, and non-zeros per control point (one control point timed)."""
    import oracle
    probe = synth.generate(spec, device=gen_device, angles=[spec.n_angles // 3])
    A = phantom_arrays_host(probe)
    x = synth.draw_x(probe.n_beamlets, 0).numpy()
    t0 = time.perf_counter()
    oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"], A["wu"],
                      A["lco"], A["aro"])
    return time.perf_counter() - t0, probe.nnz


def oracle_workload(spec, gen_device, budget_s: float, t_cp: float, nnz_cp: int, coo_host=None):
    """The data one oracle step evaluates: the WHOLE matrix when one single-thread evaluation fits `budget_s` and the
    triplets fit the host's memory, else an evenly spaced sample of control points (angle blocks: the
    evaluation is additive over them) sized to the budget.  Returns (arrays, description dict)."""
    n_a = spec.n_angles
    full_ok = t_cp * n_a <= budget_s and 12.0 * nnz_cp * n_a * 1.6 <= max(host_ram_available(), 8e9)
    if full_ok:
        A = coo_host if coo_host is not None else phantom_arrays_host(synth.generate(spec, device=gen_device))
        return A, {"control_points": n_a, "of": n_a, "nnz": int(A["val"].size), "fraction": 1.0}
    ram_cap = max(4e8, 0.4 * host_ram_available() / 12.0)                             # triplets the host can hold (>= 5 GB worth)
    k = int(max(1, min(n_a, budget_s / max(t_cp, 1e-4), ram_cap / max(nnz_cp, 1))))
    angles = sorted(set(int(round(i * n_a / k)) % n_a for i in range(k)))
    smp = synth.generate(spec, device=gen_device, angles=angles)
    return phantom_arrays_host(smp), {"control_points": len(angles), "of": n_a, "nnz": int(smp.nnz),
                                      "fraction": len(angles) / n_a}


def oracle_step(A, k: int, kind: str, cores: int):
    """One whole price evaluation O1-O5 on x draw k; returns seconds."""
    import oracle
    x = synth.draw_x(A["n_b"], k).numpy()
    args = (A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"], A["wu"], A["lco"], A["aro"])
    t0 = time.perf_counter()
    if kind == "oracle":
        oracle.price_eval(*args)
    else:
        oracle.price_eval_mt(*args, n_threads=cores)
    return time.perf_counter() - t0


def oracle_leg(A, desc, spec, kind: str, cores: int, reps: int, budget_s: float, warm: int = 0) -> dict:
    """Times `reps` evaluations (stops early beyond `budget_s`); the reported value is what was MEASURED on the data
    evaluated; when that is a sample of the control points, the full-matrix figure by additivity sits in its own key."""
    times = []
    for r in range(warm + reps):
        t = oracle_step(A, r, kind, cores)
        if r >= warm:
            times.append(t)
        if r >= warm and sum(times) > budget_s:
            break
    t_med = float(np.median(times))
    frac = desc["fraction"]
    what = "the whole matrix" if frac == 1.0 else \
        f"{desc['control_points']} of {desc['of']} control points (every {1 / frac:.1f}th angle block)"
    leg = {"value": 1.0 / t_med, "unit": UNIT, "cores": cores, "kind": "oracle", "variant": ORACLE_KINDS[kind],
           "ms_per_step": 1e3 * t_med,
           "reps": len(times), "sample_nnz": desc["nnz"],
           "sample": f"{what} of {spec.name}, {desc['nnz']} nnz; one whole evaluation O1-O5 per rep, {len(times)} reps, "
                     f"median; measured, not extrapolated"}
    if frac < 1.0:
        leg["full_matrix"] = {"value": frac / t_med, "unit": UNIT, "ms_per_step": 1e3 * t_med / frac, "extrapolated": True,
                              "factor": 1.0 / frac, "how": "angle-block additivity of the evaluation (PAPER.md L119, pin P6)"}
    return leg


def cpu_baseline(spec, gen_device, coo_host=None) -> dict:
    """bench.py's `cpu_baseline`: the plain oracle on one core (about 20 s of CPU work) and the all-cores variant on the
    same data."""
    import oracle
    t_cp, nnz_cp = oracle_probe(spec, gen_device)
    A, desc = oracle_workload(spec, gen_device, 25.0, t_cp, nnz_cp, coo_host)
    one = oracle_leg(A, desc, spec, "oracle", 1, 5, 20.0)
    cores = oracle.available_cores()
    one["all_cores"] = oracle_leg(A, desc, spec, "oracle_mt", cores, 7, 10.0, warm=1)
    return one


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (rank 0 only), K timed steps after W warm-up steps, every step
    one whole evaluation.  The plain single-thread oracle on the whole matrix when K + W such steps fit the time budget
    (configs 0-2); else the all-cores variant on the whole matrix (config 3 on a 16-core box); else an angle-block
    sample.  `value` and `ms_per_step` are what was measured on the data evaluated."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    spec = synth.config_spec(args.config, args.scale)
    gen_dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    total_budget = 150.0                                     # seconds for the whole --steps/--warmup run
    n_steps = max(1, args.steps + args.warmup)
    per_step = total_budget / n_steps
    t_cp, nnz_cp = oracle_probe(spec, gen_dev)
    cores = oracle.available_cores()
    t_full = t_cp * spec.n_angles
    if t_full <= per_step or cores == 1:
        kind, n_thr = "oracle", 1
        A, desc = oracle_workload(spec, gen_dev, per_step, t_cp, nnz_cp)
    else:
        kind, n_thr = "oracle_mt", cores
        A, desc = oracle_workload(spec, gen_dev, per_step * 0.5 * cores, t_cp, nnz_cp)   # threads scale ~0.5 x cores
    times = [oracle_step(A, k, kind, n_thr) for k in range(n_steps)]
    timed = times[args.warmup:] if len(times) > args.warmup else times
    t_med = float(np.median(timed))
    frac = desc["fraction"]
    what = "the whole matrix" if frac == 1.0 else f"{desc['control_points']} of {desc['of']} control points"
    line = {
        "impl": "reference", "metric": METRIC, "value": 1.0 / t_med, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_med, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": spec.name, "n_voxels": int(A["n_v"]), "n_beamlets": int(A["n_b"]), "nnz": int(desc["nnz"]),
                   "n_angles": int(desc["control_points"]), "n_leaf_rows": int(len(A["lco"]) - 1),
                   "evaluated": what, "sample_nnz": desc["nnz"], "fraction_of_matrix": frac},
        "cpu_baseline": {"value": 1.0 / t_med, "unit": UNIT, "cores": n_thr, "kind": "oracle", "variant": ORACLE_KINDS[kind],
                         "sample": f"{what} of {spec.name}, {desc['nnz']} nnz; every step one whole evaluation O1-O5, "
                                   f"median of the {len(timed)} timed steps; measured, not extrapolated"},
        "e2e": {"value": 1.0 / t_med, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    if frac < 1.0:
        line["full_matrix"] = {"value": frac / t_med, "unit": UNIT, "ms_per_step": 1e3 * t_med / frac, "extrapolated": True,
                               "factor": 1.0 / frac, "how": "angle-block additivity of the evaluation (PAPER.md L119)"}
    print(json.dumps(line))


# ----------------------------------------------------------------------------- NEXT-2: the master problem, timed
def bench_master_problem(vm, h, obj, out, dev, m: int) -> dict:
    """BB iterations of the master problem (vmat_mp_solve, Eq. (6)-(10)) on `m` apertures of the bench
    phantom: one aperture at each of m evenly spaced control points, every leaf row opened over a seeded random
    contiguous range, dose vectors by vmat_aperture_dose (Eq. (5)).  One iteration = one pass over the dense
    voxel-major aperture dose matrix (the rows of the voxels some aperture reaches: 4 m n_reached bytes) + the one-CTA step kernel; the time per iteration is
    the whole synchronous solve (host looks at the stop flag every 8 iterations) divided by its iterations."""
    n_v, n_a, n_rows = h.n_voxels, h.n_angles, h.n_leaf_rows
    m = max(1, min(m, n_a, 384))
    ph_lco = h.leafrow_col_offset_host
    g = torch.Generator().manual_seed(20150301)
    lens = (ph_lco[1:] - ph_lco[:-1]).to(torch.float64)
    a = torch.rand(n_rows, generator=g, dtype=torch.float64)
    b = torch.rand(n_rows, generator=g, dtype=torch.float64)
    L = (torch.minimum(a, b) * lens).floor().to(torch.int32).to(dev)
    R = (torch.maximum(a, b) * lens).ceil().to(torch.int32).to(dev)
    mp = vm.MasterProblem(n_v, m, dev)
    xs = torch.empty(h.n_beamlets, dtype=torch.float32, device=dev)
    DA = torch.empty(n_v, dtype=torch.float32, device=dev)
    t0 = time.time()
    for k in range(m):
        vm.vmat_aperture_dose(h, (k * n_a) // m, L, R, xs, DA)
        mp.add_aperture(DA, 0.0, 0.0, 50.0)
    torch.cuda.synchronize()
    t_build = time.time() - t0
    z = torch.empty(n_v, dtype=torch.float32, device=dev)
    mp.solve(obj, max_iter=16, eps_F=0.0, eps_y=0.0, z=z)                    # warm-up
    mp.set_fluence(torch.zeros(m, dtype=torch.float64))
    # five identical solves of 96 iterations from y = 0, each between its own pair of events; the median is reported (a
    # solve is ~10 ms: one alone is at the mercy of the clock the 200 price evaluations before it left behind)
    reps, runs = 5, []
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    for _ in range(reps):
        mp.set_fluence(torch.zeros(m, dtype=torch.float64))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        sol = mp.solve(obj, max_iter=96, eps_F=0.0, eps_y=0.0, z=z)
        e1.record()
        torch.cuda.synchronize()
        runs.append(1e3 * e0.elapsed_time(e1) / max(sol.n_iter, 1))
    clocks = sampler.stop()
    us = float(np.median(runs))
    Fh, _ = mp.history()
    n_reached = mp.n_reached_voxels                                           # only these rows of DA are read
    bytes_it = 4 * m * n_reached
    res = {"apertures": m, "iterations": sol.n_iter, "stop_reason": sol.reason, "us_per_iteration": us,
           "us_per_iteration_runs": [round(r, 2) for r in runs], "solves_timed": reps,
           "algorithmic_bytes_per_iteration": bytes_it, "reached_voxels": n_reached, "gbs": bytes_it / (us * 1e-6) / 1e9,
           "F_start": float(Fh[0]), "F_end": sol.F, "dtype": "f32 storage, f64 sums", "build_s": round(t_build, 2),
           "clocks": clocks,
           "workload": f"{m} apertures (random contiguous openings, one per control point), {n_v} voxels"}
    mp.close()
    return res


def bench_constrained_selection(vm, h, ph, obj, dev) -> dict:
    """NEXT-3: vmat_select_apertures_constrained (interdigitation) on the bench phantom's fields with
    the prices of a mixed-sign evaluation (x scaled so that rows open partially); ms per call, CUDA events."""
    vm.vmat_ddc_set_leaf_geometry(h, ph.leafrow_pos0)
    out = h.alloc_outputs()
    res = {}
    for scale in (0.6, 0.45, 0.35, 0.27, 0.2, 0.15, 0.1):       # a fluence level at which the prices have both signs
        vm.vmat_price_eval(h, synth.draw_x(h.n_beamlets, 424242, device=dev, scale=scale), obj, out)
        neg = float((out.p < 0).float().mean())
        res["x_scale"], res["negative_price_fraction"] = scale, neg
        if 0.25 <= neg:
            break
    o2 = h.alloc_outputs()
    for name, inter in (("interdigitation", True), ("windows_only_path", False)):
        for _ in range(3):
            vm.vmat_select_apertures_constrained(h, out.p, None, inter, o2.L, o2.R, o2.row_price, o2.angle_price, o2.best_angle)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(20):
            vm.vmat_select_apertures_constrained(h, out.p, None, inter, o2.L, o2.R, o2.row_price, o2.angle_price, o2.best_angle)
        e1.record()
        torch.cuda.synchronize()
        res[name + "_ms"] = e0.elapsed_time(e1) / 20
        if inter:
            res["rows_changed_by_constraint"] = int(((o2.L != out.L) | (o2.R != out.R)).logical_and(out.R > out.L).sum())
            res["price_ratio_constrained_over_free"] = float(o2.angle_price.min() / out.angle_price.min()) \
                if float(out.angle_price.min()) < 0 else None
    res["gpu_launches_per_call"] = vm.last_launch_count()
    res["workload"] = f"{h.n_angles} control points, {h.n_leaf_rows} leaf rows, longest row {h.info['max_leaf_row_len']} beamlets"
    return res


def bench_plan(vm, h, obj, dev, constrained=None) -> dict:
    """One whole plan optimisation by column generation (vmat_column_generation, PAPER.md L56 / Figure 1(a)): one
    aperture per control point until every control point is occupied or no aperture improves F; master problems
    with eps_F = 1e-6, at most 200 BB iterations each, fluence rates in [0, 100].  Wall clock of the synchronous call
    (the paper's headline is this loop: ~1 minute per H&N case on 4 GPUs; context, other constraints)."""
    n_a = h.n_angles
    cap = min(n_a, 384)
    mp = vm.MasterProblem(h.n_voxels, cap, dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    kw = constrained or {}
    plan = vm.vmat_column_generation(h, mp, obj, cap, 0.0, 100.0, mp_max_iter=200, eps_F=1e-6, eps_y=1e-9, **kw)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    res = {"seconds": dt, "apertures": int(plan.angles.numel()), "control_points": n_a, "stop": plan.stop,
           "F_start": float(plan.F_hist[0]), "F_end": float(plan.F_hist[-1]),
           "mp_iterations_total": int(plan.mp_iters.sum()), "gpu_launches": vm.last_launch_count(),
           "settings": "y in [0, 100], MP: eps_F 1e-6, eps_y 1e-9, <= 200 BB iterations"
                       + (", interdigitation, leaf travel <= %d beamlet widths per control point" % kw["max_leaf_travel"]
                          if kw else "")}
    mp.close()
    return res


# ----------------------------------------------------------------------------- NEXT-4: angle shards, timed
def run_sharded(args):
    """--parallelism angle-shards: ONE matrix split by control point over the N ranks (sharded.py);
    every step is one evaluation of the whole matrix: dose on every block, all-reduce of d (NCCL), objective on every
    rank, price + selection on every block, all-gather of the best control points.  Strong scaling: value = K / t."""
    import paper_1503_01721_b200 as vm
    from paper_1503_01721_b200 import sharded
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the product path has no CPU fallback")
    vm.load_library()
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    spec = synth.config_spec(args.config, args.scale)
    n_a = spec.n_angles
    from synth import phantom as P
    _, _, aco, aro, lco = P._fields(spec)
    # balance by beamlets (the non-zeros per beamlet are even); every rank generates its block only
    offs = sharded.partition_angles((aco[1:] - aco[:-1]).tolist(), world)
    ph = synth.generate(spec, device=dev, angles=list(range(offs[rank], offs[rank + 1])))
    sh = sharded.ShardedDDC.create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                                   ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, offs[rank],
                                   offs[rank + 1], device=dev, index_bits=args.index_bits)
    ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
    torch.cuda.empty_cache()
    obj = vm.Objective(ph.voxel_struct.to(dev), ph.struct_T.to(dev), ph.struct_w_over.to(dev), ph.struct_w_under.to(dev))
    out = sh.h.alloc_outputs()
    K, W = args.steps, args.warmup
    b0, b1 = sh.block.beamlet_lo, sh.block.beamlet_hi
    xs = [synth.draw_x(ph.n_beamlets, k, device=dev)[b0:b1].contiguous() for k in range(K + W)]   # same x on every rank

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(W):
        best = sh.price_eval(xs[k], obj, out)
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    launches = 0
    start.record()
    for k in range(K):
        best = sh.price_eval(xs[W + k], obj, out)
        launches += sh.last_launches   # counted by the library: vmat_last_launch_count() after each of its five calls
    stop.record()
    barrier()
    best = sharded.best_to_host(best)                            # the only read of the merged result on the host
    clocks = sampler.stop() if rank == 0 else None
    elapsed_ms, nnz_total, bytes_total = reduce_max([start.elapsed_time(stop), 0.0, 0.0], dist, dev)
    tot = torch.tensor([float(sh.h.nnz), float(sh.h.info["bytes_stream_d"] + sh.h.info["bytes_stream_dt"])],
                       dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tot)
    if rank == 0:
        peak, peak_src = measured_peaks()
        ms = elapsed_ms / K
        gbs = float(tot[1]) / (ms * 1e-3) / 1e9
        print(json.dumps({
            "metric": METRIC, "value": K / (elapsed_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": spec.name, "parallelism": f"angle-shards x{world}", "n_angles": n_a,
                       "angle_offsets": offs, "nnz": int(tot[0]), "bytes_streamed_per_step_all_ranks": int(tot[1]),
                       "exchange": f"all-reduce of d ({4 * ph.n_voxels} bytes) + all-gather of {world} (price, control point) pairs per step",
                       "x": "re-drawn per step, seeded Uniform[0,1)"},
            "hbm_gbs": gbs, "hbm_frac_of_measured_per_gpu": gbs / world / peak, "clocks": clocks,
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": "whole step incl. the exchange (no per-kernel events on this path)",
                         "achieved": gbs / world, "peak": peak, "unit": "GB/s", "frac": gbs / world / peak,
                         "peak_source": peak_src, "traffic": None},
            "result_check": {"best_angle_last": best[0], "best_price_last": best[1], "F_last": float(out.F.item())},
        }))
    sh.close()
    if dist is not None:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------- configs[4]: the roofline sweep
SWEEP_SCALES = [(1e7, 3.74), (1e8, 1.546), (1e9, 0.667), (4e9, 0.4097)]      # target nnz -> scale of the config 1 generator


def run_sweep(args):
    """--config 4 (BASELINE.json configs[4]): the config 1 generator with voxel and beamlet size scaled so that nnz spans
    1e7, 1e8, 1e9 and 4e9; at each size K consecutive price evaluations with x re-drawn every time; GB/s and fraction of
    the HBM peak for the D x and the D^T g kernels separately and for the whole fused step.  One JSON line, `sweep` = one
    entry per size; the headline value is the largest size's."""
    import paper_1503_01721_b200 as vm
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the product path has no CPU fallback")
    vm.load_library()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py --config 4 runs on one GPU")
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    peak, peak_src = measured_peaks()
    K, W = args.steps, args.warmup
    points = []
    for target, scale in SWEEP_SCALES:
        if args.sweep_max_nnz and target > args.sweep_max_nnz:
            continue
        spec = synth.config_spec(1, scale)
        pt = {"target_nnz": target, "scale": scale, "workload": spec.name}
        try:
            t0 = time.time()
            ph = synth.generate(spec, device=dev)
            torch.cuda.synchronize()
            pt["gen_s"] = round(time.time() - t0, 2)
            t0 = time.time()
            try:
                h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                                       ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=dev,
                                       index_bits=args.index_bits)
                pt["ingest"] = "COO on the device"
            except vm.VmatError as e:
                if e.status != -4:
                    raise
                # the device cannot hold the triplets next to the build's scratch: stream them from the host
                hv, hb, hw = ph.coo_voxel.cpu(), ph.coo_beamlet.cpu(), ph.coo_val.cpu()
                ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
                torch.cuda.empty_cache()
                h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, hv, hb, hw, ph.angle_col_offset, ph.angle_row_offset,
                                       ph.leafrow_col_offset, device=dev, index_bits=args.index_bits)
                del hv, hb, hw
                pt["ingest"] = "COO streamed from host memory (the device build ran out of memory with the triplets resident)"
            pt["ingest_s"] = round(time.time() - t0, 2)
            h.set_schedule({"auto": None, "sm-affine": True, "static": False}[args.schedule])
            pt["sm_affine"] = [bool(h.info["sm_affine_dose"]), bool(h.info["sm_affine_price"])]
            ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
            torch.cuda.empty_cache()
            obj = vm.Objective(ph.voxel_struct.to(dev), ph.struct_T.to(dev), ph.struct_w_over.to(dev), ph.struct_w_under.to(dev))
            out = h.alloc_outputs()
            n_b, n_v, nnz, n_rows = h.n_beamlets, h.n_voxels, h.nnz, h.n_leaf_rows
            xs = [synth.draw_x(n_b, k, device=dev) for k in range(K + W)]
            for k in range(W):
                vm.vmat_price_eval(h, xs[k], obj, out)
            ev_k = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
            for evs in ev_k:
                for e in evs:
                    e.record()
            start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            sampler = ClockSampler(local)
            sampler.start()
            time.sleep(0.25)
            start.record()
            for k in range(K):
                h.set_profile_events(ev_k[k])
                vm.vmat_price_eval(h, xs[W + k], obj, out)
            stop.record()
            torch.cuda.synchronize()
            clocks = sampler.stop()
            h.set_profile_events(None)
            ms = start.elapsed_time(stop) / K
            t_dose = float(np.mean([e[0].elapsed_time(e[1]) for e in ev_k]))
            t_price = float(np.mean([e[2].elapsed_time(e[3]) for e in ev_k]))
            info = h.info
            B_dose = info["bytes_stream_d"] + 4 * n_b + 4 * n_v + 5 * n_v
            B_price = info["bytes_stream_dt"] + 4 * n_v + 4 * n_b + 4 * (n_rows + 1) + 16 * n_rows
            l2 = (B_dose + B_price) <= 4 * 126e6
            gb = lambda b, t: b / (t * 1e-3) / 1e9
            pt.update({"nnz": nnz, "n_voxels": n_v, "n_beamlets": n_b, "evals_per_s": 1e3 / ms, "ms_per_eval": ms,
                       "index_bits": [info["index_bits_d"], info["index_bits_dt"]],
                       "dose": {"ms": t_dose, "bytes": B_dose, "gbs": gb(B_dose, t_dose), "gbs_8B_csr_equiv": gb(8 * nnz, t_dose)},
                       "price": {"ms": t_price, "bytes": B_price, "gbs": gb(B_price, t_price), "gbs_8B_csr_equiv": gb(8 * nnz, t_price)},
                       "fused_step": {"ms": ms, "bytes": B_dose + B_price, "gbs": gb(B_dose + B_price, ms),
                                      "gbs_8B_csr_equiv": gb(16 * nnz, ms)},
                       "l2_resident": l2, "clocks": clocks, "F_last": float(out.F.item())})
            if not l2:                                       # an HBM fraction only where the streams come from HBM
                for k in ("dose", "price", "fused_step"):
                    pt[k]["frac_of_measured"] = pt[k]["gbs"] / peak
                    pt[k]["frac_of_8TBs"] = pt[k]["gbs"] / 8000.0
            else:
                pt["note"] = "L2-resident: both layouts fit the 126 MB L2; no HBM fraction is claimed"
            h.close()
            del out, xs, obj, ph
        except Exception as e:                               # a size the box cannot hold is reported, not hidden
            pt["failed"] = f"{type(e).__name__}: {e}"[:400]
        torch.cuda.empty_cache()
        points.append(pt)
    ok = [p for p in points if "failed" not in p]
    top = ok[-1] if ok else None
    line = {"metric": METRIC, "value": top["evals_per_s"] if top else None, "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W,
            "ms_per_step": top["ms_per_eval"] if top else None, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "cfg4-roofline-sweep (config 1 generator, scaled)", "headline_point": top["workload"] if top else None,
                       "x": "re-drawn per evaluation, seeded Uniform[0,1)", "evaluations_per_size": K},
            "roofline": ({"bound": "hbm", "kernel": "fused step at the largest size", "achieved": top["fused_step"]["gbs"],
                          "peak": peak, "unit": "GB/s", "frac": top["fused_step"]["gbs"] / peak, "peak_source": peak_src,
                          "traffic": None} if top else None),
            "sweep": points}
    print(json.dumps(line))


# ----------------------------------------------------------------------------- the CUDA path, timed
def run_ours(args):
    import paper_1503_01721_b200 as vm
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    vm.load_library()
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    use_dist = world > 1
    if use_dist:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    spec = synth.config_spec(args.config, args.scale)
    t0 = time.time()
    ph = synth.generate(spec, device=dev)
    torch.cuda.synchronize()
    t_gen = time.time() - t0
    t0 = time.time()
    h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                           ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=dev,
                           index_bits=args.index_bits)
    t_ingest = time.time() - t0
    h.set_schedule({"auto": None, "sm-affine": True, "static": False}[args.schedule])
    stats = ph.stats()
    h.leafrow_col_offset_host = ph.leafrow_col_offset.to(torch.int64).cpu()
    # the CPU baseline evaluates the very same triplets: keep a host copy when they fit the host's memory
    coo_host = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and 12.0 * ph.nnz * 1.6 <= max(host_ram_available(), 8e9):
        coo_host = phantom_arrays_host(ph)
    ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None      # the handle holds its own layouts
    torch.cuda.empty_cache()
    obj = vm.Objective(ph.voxel_struct.to(dev), ph.struct_T.to(dev), ph.struct_w_over.to(dev),
                       ph.struct_w_under.to(dev))
    out = h.alloc_outputs()
    K, W = args.steps, args.warmup
    n_b, n_v, nnz = h.n_beamlets, h.n_voxels, h.nnz
    n_rows, n_a = h.n_leaf_rows, h.n_angles
    # x re-drawn for every evaluation (configs[4]); each rank draws its own sequence
    xs = [synth.draw_x(n_b, rank_eval_index(rank, k), device=dev) for k in range(K + W)]

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K evaluations between two events, nothing else on the stream (this is `value`)
    for k in range(W):
        vm.vmat_price_eval(h, xs[k], obj, out)
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    launches = 0
    start.record()
    for k in range(K):
        vm.vmat_price_eval(h, xs[W + k], obj, out)
        launches += vm.last_launch_count()
    stop.record()
    barrier()
    elapsed_ms = start.elapsed_time(stop)
    best_last = int(out.best_angle.item())
    F_last = float(out.F.item())

    # ---- the same K evaluations once more with four events per step around the two streaming kernels (the roofline's
    # per-launch durations; kept out of the loop above, where the event records cost 1-3 % on the small configs)
    def kernel_pass(n, x_of):
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(n)]
        for evs in ev:
            for e in evs:
                e.record()                                   # creates the underlying cudaEvent_t handles
        for k in range(n):
            h.set_profile_events(ev[k])
            vm.vmat_price_eval(h, x_of(k), obj, out)
        h.set_profile_events(None)
        torch.cuda.synchronize()
        return (np.array([e[0].elapsed_time(e[1]) for e in ev]), np.array([e[2].elapsed_time(e[3]) for e in ev]))

    t_dose, t_price = kernel_pass(K, lambda k: xs[W + k])
    clocks = sampler.stop() if rank == 0 else None

    # ---- sustained leg ("200 consecutive evaluations"): evaluations back to back for at least
    # --sustained-seconds of device time, so that the GPU reaches the state it runs this path in for a whole plan (on
    # B200 the power cap, not the full clock of a 0.1-s burst); then, without a pause, a short pass with kernel events
    sustained = None
    if args.sustained_seconds > 0:
        n_sus = min(max(K, int(np.ceil(args.sustained_seconds * 1e3 / max(elapsed_ms / K, 1e-3)))), 100000)
        s_sampler = ClockSampler(local)
        barrier()
        if rank == 0:
            s_sampler.start()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        for k in range(n_sus):
            vm.vmat_price_eval(h, xs[k % len(xs)], obj, out)
        s1.record()
        n_kp = min(max(K, 20), 50)
        sd, sp = kernel_pass(n_kp, lambda k: xs[k % len(xs)])
        s_clocks = s_sampler.stop() if rank == 0 else None
        sustained = {"steps": n_sus, "ms": s0.elapsed_time(s1), "t_dose": sd, "t_price": sp, "clocks": s_clocks,
                     "kernel_pass_steps": n_kp}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    # (vmat_price_eval_host_submit / _wait: two slots, so the copies of one evaluation overlap the kernels of the other;
    # every step still copies its own x in and its own results out inside the timed region)
    xh = [x.cpu().pin_memory() for x in xs]
    pin = lambda n, dt: torch.empty(n, dtype=dt).pin_memory()
    hb = [dict(F=pin(1, torch.float64), L=pin(n_rows, torch.int32), R=pin(n_rows, torch.int32), rp=pin(n_rows, torch.float64),
               ap=pin(n_a, torch.float64), b=pin(1, torch.int32)) for _ in range(2)]

    def e2e_run(k0, n):
        for k in range(n):
            s_ = k % 2
            if k >= 2:
                vm.vmat_price_eval_host_wait(h, s_)
            o = hb[s_]
            vm.vmat_price_eval_host_submit(h, s_, xh[k0 + k], obj, o["F"], o["L"], o["R"], o["rp"], o["ap"], o["b"])
        vm.vmat_price_eval_host_wait(h, 0)
        vm.vmat_price_eval_host_wait(h, 1)

    e2e_run(0, min(W, 4))
    barrier()
    s2, e2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s2.record()
    e2e_run(W, K)
    e2.record()
    barrier()
    e2e_ms = s2.elapsed_time(e2)
    e2e_check = {"F_last": float(hb[(K - 1) % 2]["F"][0]), "best_angle_last": int(hb[(K - 1) % 2]["b"][0])}
    # the synchronous call, for comparison (one evaluation at a time, copies not overlapped)
    o = hb[0]
    for k in range(min(W, 3)):
        vm.vmat_price_eval_host(h, xh[k], obj, o["F"], o["L"], o["R"], o["rp"], o["ap"], o["b"])
    s3, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s3.record()
    for k in range(K):
        vm.vmat_price_eval_host(h, xh[W + k], obj, o["F"], o["L"], o["R"], o["rp"], o["ap"], o["b"])
    e3.record()
    barrier()
    e2e_sync_ms = s3.elapsed_time(e3)
    h2d = 4 * n_b
    d2h = 4 * n_rows * 2 + 8 * n_rows + 8 * n_a + 4 + 8

    # ---- NEXT-2: the master problem on the same phantom, rank 0 at N = 1 only
    mp_line = plan_line = None
    if world == 1 and not args.no_mp:
        mp_line = bench_master_problem(vm, h, obj, out, dev, args.mp_apertures)
    if world == 1 and not args.no_plan:
        plan_line = bench_plan(vm, h, obj, dev)
    cs_line = cplan_line = None
    if world == 1 and not args.no_constrained and ph.leafrow_pos0 is not None:
        cs_line = bench_constrained_selection(vm, h, ph, obj, dev)
        if not args.no_plan:
            cplan_line = bench_plan(vm, h, obj, dev, dict(interdigitation=True, max_leaf_travel=4,
                                                          arc_angle_offset=ph.arc_angle_offset))

    # ---- what a read-only stream reaches on this device right now (context for the roofline: the measured peak is a
    # copy, read + write; the matrix streams are read-only): 4 GiB, 40 passes back to back, rank 0 at N = 1 only
    read_probe = None
    if world == 1:
        try:
            s_ = ClockSampler(local)
            s_.start()
            from paper_1503_01721_b200 import probe
            gbs_ro, _ = probe.hbm_read_probe(4 << 30, 40)
            read_probe = {"gbs": gbs_ro, "bytes": 4 << 30, "passes": 40, "clocks": s_.stop(),
                          "kernel": "vmat_hbm_read_probe (libvmat_probe.so, a bench aid outside the product library): "
                                    "256-bit L1::no_allocate loads, four per thread, nothing else"}
        except Exception as e:
            read_probe = {"failed": f"{type(e).__name__}: {e}"[:200]}

    # ---- max over ranks
    elapsed_ms, e2e_ms = reduce_max([elapsed_ms, e2e_ms], dist if use_dist else None, dev)
    if sustained is not None:
        sustained["ms"] = reduce_max([sustained["ms"]], dist if use_dist else None, dev)[0]

    if rank == 0:
        peak, peak_src = measured_peaks()
        # algorithmic bytes per launch: the matrix streams AS STORED
        # (8 B per entry with int32 indices, 6.125 B with u16 offsets + group bases, pads included) + the
        # vectors once.  `*_8B` is the same launch counted in the paper's 8 B/nnz CSR (Table 2), for context.
        info = h.info
        vec_dose = 4 * n_b + 4 * n_v + (1 * n_v + 4 * n_v)                               # x, d, struct id, g (fused A2)
        vec_price = 4 * n_v + 4 * n_b + 4 * (n_rows + 1) + 16 * n_rows                   # g, p, leaf-row offsets, L/R/price
        B_dose = info["bytes_stream_d"] + vec_dose
        B_price = info["bytes_stream_dt"] + vec_price
        B_dose_8B = 8 * nnz + 8 * (n_v + 1) + vec_dose
        B_price_8B = 8 * nnz + 8 * (n_b + 1) + vec_price
        B_eval = B_dose + B_price
        B_eval_8B = B_dose_8B + B_price_8B
        k_dose = {"name": "k_dose<true> (dose + fused objective/gradient)", "ncu": "k_dose<1", "grid": info["grid_dose"],
                  "ms": float(t_dose.mean()), "ms_min": float(t_dose.min()),
                  "bytes": B_dose, "gbs": B_dose / (t_dose.mean() * 1e-3) / 1e9,
                  "gbs_8B_csr_equiv": B_dose_8B / (t_dose.mean() * 1e-3) / 1e9, "index_bits": info["index_bits_d"],
                  "padded_over_nnz": info["padded_d"] / max(nnz, 1),
                  "tiles_one_base_frac": info["tiles_uniform_d"] / max(info["tiles_d"], 1)}
        k_price = {"name": "k_price<true> (price + fused leaf-row selection)", "ncu": "k_price<1", "grid": info["grid_price"],
                   "ms": float(t_price.mean()), "ms_min": float(t_price.min()),
                   "bytes": B_price, "gbs": B_price / (t_price.mean() * 1e-3) / 1e9,
                   "gbs_8B_csr_equiv": B_price_8B / (t_price.mean() * 1e-3) / 1e9, "index_bits": info["index_bits_dt"],
                   "padded_over_nnz": info["padded_dt"] / max(nnz, 1),
                   "tiles_one_base_frac": info["tiles_uniform_dt"] / max(info["tiles_dt"], 1)}
        dom = k_price if k_price["ms"] >= k_dose["ms"] else k_dose
        traffic, traffic_src = ncu_traffic(dom["ncu"], dom["grid"], dom["bytes"])
        agg = aggregate(world, K, elapsed_ms)
        ms_per_step, value = agg["ms_per_step"], agg["value"]
        eval_gbs = B_eval / (ms_per_step * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": spec.name, "n_voxels": n_v, "n_beamlets": n_b, "nnz": nnz, "n_angles": n_a,
                       "n_leaf_rows": n_rows, "bytes_layout_d": info["bytes_stream_d"],
                       "bytes_layout_dt": info["bytes_stream_dt"], "index_bits": [info["index_bits_d"], info["index_bits_dt"]],
                       "parallelism": "replicas only" if world > 1 else "1 gpu",
                       "l2": f"inputs larger than L2: {B_eval / 1e9:.2f} GB streamed per step vs 126 MB L2"
                             if B_eval > 4 * 126e6 else "L2-resident: matrix fits the 126 MB L2, no HBM fraction claimed",
                       "x": "re-drawn per step, seeded Uniform[0,1)", "gen_s": round(t_gen, 2),
                       "ingest_s": round(t_ingest, 2), "schedule": args.schedule,
                       "sm_affine": [bool(info["sm_affine_dose"]), bool(info["sm_affine_price"])],
                       "grid": [info["grid_dose"], info["grid_price"]]},
            "hbm_gbs": eval_gbs, "hbm_frac_of_8TBs": eval_gbs / 8000.0, "hbm_frac_of_measured": eval_gbs / peak,
            "hbm_gbs_8B_csr_equiv": B_eval_8B / (ms_per_step * 1e-3) / 1e9,
            "clocks": clocks,
            "e2e": {"value": aggregate(world, K, e2e_ms)["value"], "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / K,
                    "api": "vmat_price_eval_host_submit / _wait (two slots: copies overlap the other slot's kernels)",
                    "copied_in": "x (pinned host, 4 n_beamlets bytes)",
                    "copied_back": "F, L, R, row_price, angle_price, best_angle (what the consumer of the path reads); "
                                   "d, g and p stay on the device",
                    "result_check": e2e_check,
                    "synchronous_call": {"value": world * K / (e2e_sync_ms * 1e-3), "ms_per_step": e2e_sync_ms / K,
                                         "api": "vmat_price_eval_host"}},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": dom["name"], "achieved": dom["gbs"], "peak": peak,
                         "unit": "GB/s", "frac": dom["gbs"] / peak, "frac_of_8TBs": dom["gbs"] / 8000.0,
                         "peak_source": peak_src, "traffic": traffic, "traffic_source": traffic_src,
                         "algorithmic_bytes": dom["bytes"],
                         "ms": dom["ms"], "read_only_stream": read_probe},
            "kernels": [k_dose, k_price],
            "result_check": {"F_last": F_last, "best_angle_last": best_last},
        }
        if sustained is not None:
            s_ms = sustained["ms"] / sustained["steps"]
            sd, sp = float(sustained["t_dose"].mean()), float(sustained["t_price"].mean())
            line["sustained"] = {
                "evals_per_s": world * sustained["steps"] / (sustained["ms"] * 1e-3), "ms_per_step": s_ms,
                "seconds": sustained["ms"] * 1e-3, "steps": sustained["steps"],
                "hbm_gbs": B_eval / (s_ms * 1e-3) / 1e9, "hbm_frac_of_measured": B_eval / (s_ms * 1e-3) / 1e9 / peak,
                "kernels": [{"name": k_dose["name"], "ms": sd, "gbs": B_dose / (sd * 1e-3) / 1e9,
                             "frac": B_dose / (sd * 1e-3) / 1e9 / peak},
                            {"name": k_price["name"], "ms": sp, "gbs": B_price / (sp * 1e-3) / 1e9,
                             "frac": B_price / (sp * 1e-3) / 1e9 / peak}],
                "kernel_pass": f"{sustained['kernel_pass_steps']} evaluations with kernel events, enqueued right behind the "
                               "sustained loop (same thermal / power state)",
                "x": "the K + W seeded draws, cycled", "clocks": sustained["clocks"]}
        if mp_line is not None:
            mp_line["frac_of_measured"] = mp_line["gbs"] / peak
            line["master_problem"] = mp_line
        if plan_line is not None:
            line["plan_optimisation"] = plan_line
        if cs_line is not None:
            line["constrained_selection"] = cs_line
        if cplan_line is not None:
            line["plan_optimisation_constrained"] = cplan_line
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(spec, dev, coo_host)
        print(json.dumps(line))
    h.close()
    if use_dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3, 4],
                    help="BASELINE.json config (default 3: the largest DDC; 4: the roofline sweep, one line with a `sweep` array)")
    ap.add_argument("--sweep-max-nnz", type=float, default=0.0, help="--config 4: skip the sizes beyond this many non-zeros")
    ap.add_argument("--scale", type=float, default=1.0, help="config 4 sweep: coarsen voxels/beamlets by this factor")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--index-bits", type=int, default=0, choices=[0, 16, 32],
                    help="index encoding of the layouts (vmat_ddc_create_ex): 0 = chosen per layout")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "angle-shards"],
                    help="N > 1: independent replicas (default; the path needs one GPU) or ONE matrix split by control "
                         "point over the ranks (NEXT-4)")
    ap.add_argument("--schedule", default="auto", choices=["auto", "sm-affine", "static"],
                    help="work distribution of the dose and price kernels (vmat_ddc_set_schedule)")
    ap.add_argument("--sustained-seconds", type=float, default=3.0,
                    help="after the K timed steps, run evaluations back to back for this long (device time) and report "
                         "them as `sustained` (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-mp", action="store_true", help="skip the master-problem measurement")
    ap.add_argument("--mp-apertures", type=int, default=128)
    ap.add_argument("--no-plan", action="store_true", help="skip the whole-plan (column generation) measurements")
    ap.add_argument("--no-constrained", action="store_true", help="skip the constrained-selection (NEXT-3) measurements")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        if args.config == 4:
            args.config, args.scale = 1, SWEEP_SCALES[-1][1]
        run_reference(args)
    elif args.config == 4:
        run_sweep(args)
    elif args.parallelism == "angle-shards":
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
