#!/usr/bin/env python
"""bench.py -- grid-point.steps/s of the fused forward+adjoint gradient sweep (BASELINE.json metric).

A "step" = one pass of the whole hot path (forward sweep + trajectory
store, misfit / background / overlap terms, adjoint sweep) over every subdomain of the workload.
Default workload: BASELINE.json configs[3], the 0.25 deg 1440x720 grid, 256 steps, 16x16x8
decomposition, overlap 2 (the config the roofline target is quoted on).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

`--impl reference` times the CPU oracle (oracle/), as it stands, on the host cores on a bounded
sample of the same workload.  N > 1: one process per GPU (torchrun), each rank runs an independent
replica of the workload ("replicas only"): weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2205_06649_b200 import synth  # noqa: E402

METRIC = "grid-point.steps/s of fused forward+adjoint gradient sweep"
UNIT = "grid-point.steps/s"


def peaks():
    """Measured HBM copy bandwidth (GB/s) from MEASURED_PEAKS.json, else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def algorithmic_bytes(subs, q_time, nobs_binned, with_gw=False):
    """per sweep, forward and adjoint kernels separately.
    subs: list of dicts from subdomain_info; nobs_binned: total binned observations."""
    fwd = adj = 0
    pts = 0
    for s in subs:
        nc = s["ex"] * s["ey"]
        px = s["ex"] + 2 * s["gx"]; py = s["ey"] + s["gys"] + s["gyn"]
        nring = px * py - nc
        W = s["e"] - s["s"]
        pts += nc * W
        fixed_f = 24 * nc * 2            # control, u^b(s_j)
        if s["jw"] > 0:
            fixed_f += 24 * nc           # predecessor end state
        if s["jw"] < q_time - 1:
            fixed_f += 24 * nc           # successor control
        fwd += fixed_f + 24 * W * nring + 24 * W * nc          # ghost read, trajectory write
        fixed_a = 24 * nc * 3            # level W (end forcing), control + u^b (gradient terms)
        if s["jw"] > 0:
            fixed_a += 24 * nc
        if s["jw"] < q_time - 1:
            fixed_a += 24 * nc
        adj += fixed_a + 24 * W * nring + 24 * W * nc + 24 * nc * (2 if with_gw else 1)
    fwd += 20 * nobs_binned
    adj += 20 * nobs_binned
    return fwd, adj, pts


def survey_bytes(subs, nobs_binned):
    """SURVEY.md 8(d)'s accounting, per sweep and kernel: what the METHOD has to move, not what this implementation
    moves -- 48 B per processed point-step (state read + write), the ghost ring, 0.2 B of observations and 126 B per
    control cell of fixed traffic (control, u^b, neighbour data, gradient), split evenly between the two sweeps (about
    61 B per processed point-step on config 3; algorithmic_bytes() above counts 64.5 B because it includes ck_cost's
    re-reads).  The 0.60 target of north_star is read against THIS count (roofline.frac_survey_bytes)."""
    fwd = adj = 0
    for s in subs:
        nc = s["ex"] * s["ey"]
        nring = (s["ex"] + 2 * s["gx"]) * (s["ey"] + s["gys"] + s["gyn"]) - nc
        W = s["e"] - s["s"]
        fwd += 24 * W * nc + 24 * W * nring + 63 * nc
        adj += 24 * W * nc + 24 * W * nring + 63 * nc
    return fwd + 10 * nobs_binned, adj + 10 * nobs_binned


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill(); out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def csrc_hash():
    """sha256 over the CUDA sources: ties profiles/traffic.json to the kernels it was captured from."""
    import hashlib
    d = os.path.join(ROOT, "paper_2205_06649_b200", "csrc")
    hh = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        hh.update(f.encode()); hh.update(open(os.path.join(d, f), "rb").read())
    return hh.hexdigest()[:16]


def measured_traffic(kernel, cfg):
    """DRAM bytes per launch of `kernel` (dram__bytes_read.sum + dram__bytes_write.sum of one
    `ncu --set full` capture, committed as profiles/traffic.json).  None unless the capture was
    taken on config 3 from exactly the CUDA sources of this build (csrc hash recorded in the file)."""
    try:
        if cfg != 3:
            return None
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        if t.get("csrc_sha16") != csrc_hash():
            return None
        return int(t["kernels"][kernel])
    except Exception:
        return None


PATH_NAMES = {1: "generic (block-tiled step kernels)", 2: "row-marching fused kernels", 3: "per-stage generic kernels",
              4: "wavefront forward (wk_forward) + row-marching adjoint (fk_adjoint2)",
              5: "wavefront forward (wk_forward) + control-level terms (ck_cost) + wavefront adjoint (wk_adjoint)"}


def max_over_ranks(values, device=None):
    """Element-wise MAX over all ranks of a list of floats (identity without a process group).
    This is the only cross-rank step of the benchmark: replicas share no data."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_value(units_per_rank, world, seconds):
    """Weak scaling: every rank processes `units_per_rank`; the job takes the slowest rank's time."""
    return world * units_per_rank / seconds


LAYOUT = None          # --layout p_lon,p_lat,q_time,overlap: another decomposition of the chosen config's problem (config 4)


def workload(cfg):
    if cfg in synth.CONFIGS:
        w = synth.CONFIGS[cfg]
        if LAYOUT:
            import dataclasses
            w = dataclasses.replace(w.with_layout(*LAYOUT), name=w.name.rsplit(" ", 2)[0] + " %dx%dx%d o%d" % tuple(LAYOUT))
        return w
    raise SystemExit(f"unknown config {cfg}")


def oracle_sweep_sample(w, budget_pts=1.5e8):
    """The oracle's gradient sweep on the first subdomains of the SAME workload (bounded sample)."""
    from oracle import Oracle
    o = Oracle.from_workload(w)
    prob = synth.make_problem(w, o.forecast)
    o.set_background(prob.xb, prob.sigma_b)
    o.set_observations(prob.obs)
    k1 = 0; pts = 0
    while k1 < o.nsub and pts < budget_pts:
        s = o.subs[k1]; pts += s["ex"] * s["ey"] * (s["e"] - s["s"]); k1 += 1
    tot = sum(s["ex"] * s["ey"] * (s["e"] - s["s"]) for s in o.subs)
    o.useful_ratio = w.nlon * w.nlat * w.nsteps / tot      # useful / processed point-steps
    return o, k1


def cpu_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def _omp_threads(n):
    """Thread count of the OpenMP runtime the oracle library uses (libgomp); the oracle is untouched."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except Exception:
        return False


def cpu_baseline(w):
    """The correctness oracle as it stands (gcc -O2, -ffp-contract=off, long-double sums; never tuned
    as a baseline), timed on a bounded sample: one warm-up sweep, then the median of 3 sweeps with
    OpenMP over subdomains on all cores, and the median of 3 single-thread sweeps on a smaller sample."""
    t0 = time.perf_counter()
    o, k1 = oracle_sweep_sample(w)
    t1 = time.perf_counter()
    cores = cpu_cores()
    o.sweep_range(0, k1)                                   # warm-up
    ts = []
    for _ in range(3):
        a = time.perf_counter(); p, _ = o.sweep_range(0, k1); ts.append(time.perf_counter() - a)
    tm = float(np.median(ts))
    out = {"value": o.useful_ratio * p / tm, "unit": UNIT, "cores": cores, "kind": "oracle",
           "note": "untuned correctness oracle (gcc -O2 -ffp-contract=off), OpenMP over subdomains; a reported baseline, not a target",
           "sample": f"gradient sweep of subdomains 0..{k1 - 1} of {o.nsub} ({int(p)} processed point-steps), "
                     f"median of 3 after 1 warm-up: {tm:.2f} s (oracle setup {t1 - t0:.1f} s not timed)"}
    k1s = max(1, k1 // max(cores, 1))
    if _omp_threads(1):
        o.sweep_range(0, k1s)
        ts1 = []
        for _ in range(3):
            a = time.perf_counter(); p1, _ = o.sweep_range(0, k1s); ts1.append(time.perf_counter() - a)
        _omp_threads(cores)
        out["single_thread"] = {"value": o.useful_ratio * p1 / float(np.median(ts1)), "unit": UNIT, "cores": 1,
                                "sample": f"subdomains 0..{k1s - 1}, median of 3 after 1 warm-up: {float(np.median(ts1)):.2f} s"}
    return out


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    o, k1 = oracle_sweep_sample(w)
    for _ in range(max(args.warmup, 0) and 1):
        o.sweep_range(0, k1)
    t0 = time.perf_counter(); pts = 0.0
    for _ in range(args.steps):
        p, _ = o.sweep_range(0, k1); pts += p
    dt = time.perf_counter() - t0
    val = o.useful_ratio * pts / dt
    sample = (f"subdomains 0..{k1 - 1} of {o.nsub} ({int(pts / args.steps)} processed point-steps per step; "
              f"value scaled by the workload's useful/processed ratio {o.useful_ratio:.4f})")
    line = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": w.name, "counted": "useful = nlon*nlat*nsteps per sweep"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_cores(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_driver(args):
    """Time to analysis of Algorithm 1 on one config: run(outer_iters), cost history, RMSE vs truth."""
    import torch
    from paper_2205_06649_b200.binding import DD4DVar
    w = workload(args.config)
    g = DD4DVar.from_workload(w, path=args.path)
    prob = synth.make_problem(w, g.forecast)
    g.set_background(prob.xb, prob.sigma_b); g.set_observations(prob.obs)
    outer = args.outer if args.outer is not None else w.outer_iters
    extra = {}
    if args.gn:
        # the paper's own local minimiser (Alg 5-7): Gauss-Newton + CG; one CG iteration = TLM sweep + adjoint sweep
        xs = g.get_controls(); pw = torch.ones_like(xs)
        g.gn_hessvec(xs, pw); torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record(); g.sweep_async(0); ev[1].record(); g.gn_hessvec(xs, pw); ev[2].record(); torch.cuda.synchronize()
        fwd_ms = ev[0].elapsed_time(ev[1]); hv_ms = ev[1].elapsed_time(ev[2]) - fwd_ms
        extra = {"local_solver": f"Gauss-Newton n_gn={args.n_gn} n_cg={args.n_cg}", "forward_sweep_ms": fwd_ms,
                 "hessvec_ms": hv_ms, "hessvec": "one product with H_GN on every subdomain = TLM sweep (tk_step, one launch "
                 "per step) + ck_gn + adjoint sweep (wk_adjoint); gn_hessvec call minus its forward sweep"}
    torch.cuda.synchronize(); t0 = time.perf_counter()
    an, hist = g.run_gn(outer, args.n_gn, args.n_cg) if args.gn else g.run(outer)
    torch.cuda.synchronize(); dt = time.perf_counter() - t0
    an = an.cpu().numpy()
    rm = lambda a, b: float(np.sqrt(np.mean((a - b) ** 2)))
    print(json.dumps({"config": args.config, "workload": w.name, "outer_iters": outer, "time_to_analysis_s": dt,
                      "launches": int(g.launch_count), "J_global": [float(x) for x in hist[:, 0]],
                      "sumJ_local": [float(x) for x in hist[:, 1]], "delta": [float(x) for x in hist[:, 2]],
                      "rmse_background_h_u_v": [rm(prob.xb[f], prob.truth0[f]) for f in range(3)],
                      "rmse_analysis_h_u_v": [rm(an[f], prob.truth0[f]) for f in range(3)], **extra}))
    g.close()


def run_sharded(args):
    """Algorithm 1 with the time windows sharded over the ranks (paper_2205_06649_b200/parallel.py): time per outer
    iteration, total work fixed ("strong").  One process per GPU under torchrun; N = 1 runs the same driver."""
    import torch
    import torch.distributed as dist
    from paper_2205_06649_b200.parallel import ShardedDD4DVar
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    w = workload(args.config)
    sh = ShardedDD4DVar(w, device=f"cuda:{local_rank}", path=args.path)
    prob = synth.make_problem(w, sh.g.forecast)
    sh.set_background(prob.xb, prob.sigma_b); sh.set_observations(prob.obs)
    outer = args.outer if args.outer is not None else 3
    sh.run(1)                                           # warm-up iteration
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev); t0 = time.perf_counter()
    an, hist = sh.run(outer)
    torch.cuda.synchronize(dev); dt = time.perf_counter() - t0
    (dt,) = max_over_ranks([dt], dev)
    if rank == 0:
        print(json.dumps({"metric": "outer iterations of Algorithm 1 per second, windows sharded over the GPUs", "value": outer / dt,
                          "unit": "outer iterations/s", "n_gpus": world, "scaling": "strong", "ms_per_outer_iteration": 1e3 * dt / outer,
                          "config": {"workload": w.name, "windows_per_rank": [b[1] - b[0] for b in
                                     __import__("paper_2205_06649_b200.parallel", fromlist=["x"]).window_blocks(w.q_time, world)],
                                     "exchange_bytes_per_iteration": int(2 * 8 * sh.g.ctot)},
                          "sumJ_local": [float(x) for x in hist[:, 0]], "delta": [float(x) for x in hist[:, 1]]}))
    sh.close()
    if world > 1:
        dist.barrier(); dist.destroy_process_group()


def run_table3(args):
    """The shape of the paper's weak-scaling experiment (Table 3; eq (57)): local problems of
    fixed size n_loc = 32 (owned 32x32 cells, overlap 2, 16-step windows), QP = 2 ... 4096 subdomains, here all on ONE
    GPU: time of one gradient sweep of all QP local problems and the software scale-up QP * T(one local problem) / T(QP),
    with T(one local problem) taken from the QP = 2 run (its two subdomains run side by side on two SMs)."""
    import dataclasses
    import torch
    from paper_2205_06649_b200.binding import DD4DVar
    dev = torch.device("cuda", 0)
    layouts = [(2, 1, 1), (2, 2, 1), (2, 2, 2), (4, 2, 2), (4, 4, 2), (4, 4, 4), (8, 4, 4), (8, 8, 4), (8, 8, 8), (16, 8, 8),
               (16, 16, 8), (32, 16, 8)]
    t1 = None
    for (p1, p2, q) in layouts:
        nlon, nlat, nsteps = 32 * p1, 32 * p2, 16 * q
        deg = 360.0 / nlon
        w = synth.Workload(90, nlon, nlat, min(600.0, 300.0 * deg), nsteps, 5, 0.05, 4, p1, p2, q, 2, 1,
                           name=f"table3 n_loc=32 {p1}x{p2}x{q}")
        g = DD4DVar.from_workload(w, device="cuda:0", path=args.path)
        prob = synth.make_problem(w, g.forecast)
        g.set_background(prob.xb, prob.sigma_b); g.set_observations(prob.obs)
        for _ in range(3):
            g.sweep_async(1)
        torch.cuda.synchronize(dev)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        n = 10
        ev[0].record()
        for _ in range(n):
            g.sweep_async(1)
        ev[1].record(); torch.cuda.synchronize(dev)
        ms = ev[0].elapsed_time(ev[1]) / n
        if t1 is None:
            t1 = ms
        qp = p1 * p2 * q
        print(json.dumps({"table": 3, "QP": qp, "layout": f"{p1}x{p2}x{q}", "grid": f"{nlon}x{nlat}", "steps": nsteps,
                          "problem_size": 3 * 32 * 32 * qp, "path": PATH_NAMES.get(g.active_path, str(g.active_path)).split("(")[0].strip(),
                          "sweep_ms": ms, "scale_up": qp * t1 / ms,
                          "useful_point_steps_per_s": nlon * nlat * nsteps / (ms * 1e-3)}), flush=True)
        g.close()


def run_sweep(args):
    """BASELINE.json configs[4]: time-to-analysis and grid-point.steps/s per layout on the fixed
    0.5 deg / 128-step problem (one JSON line per layout; the paper's time-complexity analysis)."""
    import torch
    from paper_2205_06649_b200.binding import DD4DVar
    dev = torch.device("cuda", 0)
    base = synth.CONFIGS[2]
    g0 = DD4DVar.from_workload(base.with_layout(1, 1, 1, 0), device="cuda:0")
    prob = synth.make_problem(base, g0.forecast)
    g0.close()
    for w in synth.sweep_workloads():
        if (w.p_lon, w.p_lat, w.q_time) == (1, 1, 1):
            w = w.with_layout(1, 1, 1, 0)
            if any(l.get("layout") == "1x1x1" for l in getattr(run_sweep, "done", [])):
                continue
        g = DD4DVar.from_workload(w, device="cuda:0")
        g.set_background(prob.xb, prob.sigma_b)
        g.set_observations(prob.obs)
        for _ in range(3):
            g.sweep_async(1)
        torch.cuda.synchronize(dev)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev[0].record(); n = 5
        for _ in range(n):
            g.sweep_async(1)
        ev[1].record(); torch.cuda.synchronize(dev)
        ms = ev[0].elapsed_time(ev[1]) / n
        outer = args.outer if args.outer is not None else w.outer_iters
        t0 = time.perf_counter()
        an, hist = g.run(outer)
        torch.cuda.synchronize(dev)
        tta = time.perf_counter() - t0
        line = {"config": 4, "layout": f"{w.p_lon}x{w.p_lat}x{w.q_time}", "overlap": w.overlap, "subdomains": g.nsub,
                "path": PATH_NAMES.get(g.active_path, str(g.active_path)), "sweep_ms": ms,
                "useful_point_steps_per_s": w.nlon * w.nlat * w.nsteps / (ms * 1e-3), "outer_iters": outer,
                "time_to_analysis_s": tta, "J_first": float(hist[0, 0]), "J_last": float(hist[-1, 0]),
                "delta_last": float(hist[-1, 2])}
        g.close()
        if args.oracle_outer > 0:
            # the CPU oracle beside it (BASELINE.json configs[4]: "against the oracle"): the same layout and inputs, one
            # gradient sweep of every subdomain (median of 2 after a warm-up) and `oracle_outer` outer iterations of
            # Algorithm 1, on this box's host cores; the 20-iteration time is that per-iteration time scaled up
            from oracle import Oracle
            o = Oracle.from_workload(w)
            o.set_background(prob.xb, prob.sigma_b); o.set_observations(prob.obs)
            o.sweep_range(0, o.nsub)
            ts = []
            for _ in range(2):
                a = time.perf_counter(); o.sweep_range(0, o.nsub); ts.append(time.perf_counter() - a)
            osw = float(np.median(ts))
            a = time.perf_counter(); _, oh = o.run(args.oracle_outer); orun = time.perf_counter() - a
            # (this is the cpu_baseline leg of the config-4 mode: the oracle timed beside the GPU, never on the product path)
            line["cpu_baseline"] = {
                "kind": "oracle", "cores": cpu_cores(), "unit": UNIT,
                "value": w.nlon * w.nlat * w.nsteps / osw, "sweep_ms": 1e3 * osw,
                "sample": f"one gradient sweep of all {o.nsub} subdomains (median of 2 after 1 warm-up) and {args.oracle_outer} outer iterations of Algorithm 1",
                "outer_iters": args.oracle_outer, "s_per_outer_iteration": orun / args.oracle_outer,
                "time_to_analysis_s_scaled": orun / args.oracle_outer * outer,
                "J_after": float(oh[-1, 0])}
            line["gpu_J_after_same_iters"] = float(hist[min(args.oracle_outer, outer), 0])
            line["sweep_speedup_vs_oracle"] = osw / (ms * 1e-3)
            line["time_to_analysis_speedup_vs_oracle"] = orun / args.oracle_outer * outer / tta
            del o
        run_sweep.done = getattr(run_sweep, "done", []) + [line]
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 generic, 2 row-marching, 3 per-stage, 4 wavefront fwd + row-marching adj, 5 wavefront")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--run", action="store_true", help="time the whole driver: run(outer_iters) on --config")
    ap.add_argument("--table3", action="store_true", help="the paper's weak-scaling shape (Table 3): n_loc = 32, QP = 2 ... 4096 local problems on one GPU")
    ap.add_argument("--shard", action="store_true", help="Algorithm 1 with the time windows sharded over the ranks (torchrun, one per GPU)")
    ap.add_argument("--gn", action="store_true", help="with --run: Gauss-Newton + CG local minimiser (dd4dvar_run_gn)")
    ap.add_argument("--n-gn", type=int, default=2)
    ap.add_argument("--n-cg", type=int, default=5)
    ap.add_argument("--sweep", action="store_true", help="config 4: decomposition sweep on the 0.5 deg problem")
    ap.add_argument("--oracle-outer", type=int, default=0, help="with --sweep: also time the CPU oracle on every layout (one sweep + this many outer iterations)")
    ap.add_argument("--outer", type=int, default=None, help="outer iterations for --sweep (default: the config's)")
    ap.add_argument("--peaks", action="store_true", help="run the library's fp64 / shared-memory / shuffle microbenchmarks")
    ap.add_argument("--csrc-hash", action="store_true", help="print the hash of the CUDA sources (for profiles/traffic.json)")
    ap.add_argument("--overlap-levels", action="store_true", help="spatial overlap penalty on every level of the window (needs --path 1)")
    ap.add_argument("--layout", default=None, help="p_lon,p_lat,q_time,overlap: decomposition override (config 4 layouts on --config 2)")
    args = ap.parse_args()
    if args.layout:
        global LAYOUT
        LAYOUT = [int(x) for x in args.layout.split(",")]
    if args.csrc_hash:
        print(csrc_hash())
        return
    if args.peaks:
        from paper_2205_06649_b200 import binding
        print(json.dumps(binding.measure_peaks("cuda:0")))
        return
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.sweep:
        run_sweep(args)
        return
    if args.table3:
        run_table3(args)
        return
    if args.shard:
        run_sharded(args)
        return
    if args.run:
        run_driver(args)
        return
    w = workload(args.config)
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    from paper_2205_06649_b200.binding import DD4DVar

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # ---- build the replica of the workload on this rank (seeded synthetic inputs)
    g = DD4DVar.from_workload(w, path=args.path, device=f"cuda:{local_rank}")
    if args.overlap_levels:
        g.set_overlap_levels(True)                    # (25c) on every level of the window (generic kernels: --path 1)
    prob = synth.make_problem(w, g.forecast)          # truth trajectory from the library's own model
    g.set_background(prob.xb, prob.sigma_b)
    g.set_observations(prob.obs)
    nobs_binned = 0
    lv = set(int(x) for x in prob.obs.levels)
    n_per_level = int(prob.obs.offsets[1] - prob.obs.offsets[0]) if len(prob.obs.levels) else 0
    # binned observation count: every observation lands in every (window, tile) that holds it
    cell = prob.obs.index[:n_per_level] % (w.nlon * w.nlat)
    gi = cell % w.nlon; gj = cell // w.nlon
    colmult = np.zeros(w.nlon, dtype=np.int64); rowmult = np.zeros(w.nlat, dtype=np.int64)
    seen_a, seen_b = set(), set()
    for s in g.subs:
        if s["jw"] == 0 and s["b"] == 0:
            colmult[(s["ei0"] + np.arange(s["ex"])) % w.nlon] += 1
        if s["jw"] == 0 and s["a"] == 0:
            rowmult[s["ej0"] + np.arange(s["ey"])] += 1
    per_level = int(np.sum(colmult[gi] * rowmult[gj]))
    wins = sorted(set((s["s"], s["e"]) for s in g.subs))
    for lev in lv:
        nobs_binned += per_level * sum(1 for (s0, e0) in wins if s0 <= lev <= e0)
    fwd_b, adj_b, pts = algorithmic_bytes(g.subs, w.q_time, nobs_binned)
    sv_fwd, sv_adj = survey_bytes(g.subs, nobs_binned)
    useful = w.nlon * w.nlat * w.nsteps

    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing: K gradient sweeps (inputs far larger than L2, no flush needed)
    for _ in range(args.warmup):
        g.sweep_async(1)
    barrier()
    l0 = g.launch_count
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    barrier()
    ev[0].record(stream)
    for _ in range(args.steps):
        g.sweep_async(1)
    ev[1].record(stream)
    barrier()
    ms = ev[0].elapsed_time(ev[1])
    launches = g.launch_count - l0
    clocks = sampler.stop() if sampler else None
    # per-kernel split (forward+cost vs adjoint), same stream, same events
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    t_f = t_a = 0.0
    nsplit = max(3, min(args.steps, 10))
    for _ in range(nsplit):
        evs[0].record(stream); g.sweep_async(0); evs[1].record(stream); g.sweep_async(2); evs[2].record(stream)
        torch.cuda.synchronize(dev)
        t_f += evs[0].elapsed_time(evs[1]); t_a += evs[1].elapsed_time(evs[2])
    t_f /= nsplit; t_a /= nsplit

    # ---- end to end through the C-ABI with host buffers (pinned), copies inside the timed region
    h_ctrl = g.get_controls().cpu().pin_memory()
    h_grad = torch.empty_like(h_ctrl).pin_memory()
    h_cost = np.zeros(g.nsub)
    e2e_steps = max(3, min(args.steps, 5))
    g.eval_local_host(h_ctrl, h_cost, h_grad)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        g.eval_local_host(h_ctrl, h_cost, h_grad)
    torch.cuda.synchronize(dev)
    e2e_s = (time.perf_counter() - t0) / e2e_steps

    # one outer iteration of Algorithm 1 (a5 L-BFGS + a6 exchange + the sweeps it needs), reported
    g.run(1)                                         # (untimed: first use of the driver's kernels)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    g.run(1)
    outer_s = time.perf_counter() - t0
    g.set_history_global(False)                     # the same without the J_global diagnostic (one undecomposed forecast)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    g.run(1)
    outer_ng_s = time.perf_counter() - t0
    g.set_history_global(True)
    # the same outer iteration split by phase with CUDA events on the library's stream (dd4dvar_set_phase_timing)
    g.set_phase_timing(True)
    g.run(1)
    phase = g.phase_ms()
    g.set_phase_timing(False)
    ms, e2e_s, outer_s, outer_ng_s = max_over_ranks([ms, e2e_s, outer_s, outer_ng_s], dev)

    if rank == 0:
        ms_step = ms / args.steps
        peak, peak_src = peaks()
        ap = g.active_path
        fused = ap in (2, 4, 5)
        if fused:   # the dominant kernel of the sweep = the adjoint sweep (one launch per gradient sweep)
            kname = "wk_adjoint" if ap == 5 else "fk_adjoint2"
            fname = "fk_forward2" if ap == 2 else "wk_forward"
            kern, kb, kt = kname + " (adjoint sweep, one launch per gradient sweep)", adj_b, t_a
        else:
            kname = fname = None
            kern, kb, kt = "gradient sweep, all per-stage launches of the generic path", fwd_b + adj_b, ms_step
        achieved = kb / (kt * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": whole_job_value(useful, world, ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "counted": "useful = nlon*nlat*nsteps per sweep",
                       "processed_point_steps_per_sweep": pts, "processed_value": world * pts / (ms_step * 1e-3),
                       "subdomains": g.nsub, "path": PATH_NAMES.get(ap, str(ap)), "overlap_levels": bool(args.overlap_levels),
                       "l2": "inputs larger than L2 (trajectory store %.1f GB per sweep)" % (24.0 * pts / 1e9),
                       "parallelism": "replicas" if world > 1 else "single GPU",
                       "outer_iteration_ms": 1e3 * outer_s, "outer_iteration_ms_without_global_history": 1e3 * outer_ng_s,
                       "outer_iteration": "run(1) after one untimed run(1): 5 L-BFGS iterations (a5) + exchange (a6) + J_global, not in the timed region",
                       "sweeps_ms": phase["sweeps"], "lbfgs_ms": phase["lbfgs"], "exchange_ms": phase["exchange"],
                       "jglobal_ms": phase["jglobal"], "gather_ms": phase["gather"],
                       "outer_iteration_split": "CUDA events on the library's stream inside one more run(1): sweeps (a1-a4 of every "
                                                "trial and accepted point), L-BFGS kernels incl. the host round trip of each line-search "
                                                "check (a5), exchange (a6), J_global diagnostic, final gather"},
            "clocks": clocks,
            "e2e": {"value": world * useful / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(g.ctot * 8),
                    "d2h_bytes_per_step": int(g.ctot * 8 + g.nsub * 8), "ms_per_step": 1e3 * e2e_s},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": measured_traffic(kname, args.config) if fused else None,
                         "traffic_source": "profiles/traffic.json (ncu --set full capture of this build's sources; null = no capture of this build)",
                         "kernel": kern, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": kb, "kernel_ms": kt,
                         "sweep_algorithmic_GBps": (fwd_b + adj_b) / (ms_step * 1e-3) / 1e9,
                         "forward_ms": t_f, "adjoint_ms": t_a,
                         "forward_kernel": {"name": fname, "algorithmic_bytes_per_launch": fwd_b,
                                            "achieved": fwd_b / (t_f * 1e-3) / 1e9, "frac": fwd_b / (t_f * 1e-3) / 1e9 / peak,
                                            "traffic": measured_traffic(fname, args.config) if fused else None,
                                            "note": "forward sweep + trajectory store + cost terms (wk_forward and ck_cost, timed together)"},
                         "bytes_per_processed_point_step": (fwd_b + adj_b) / pts,
                         "frac_survey_bytes": (sv_adj if fused else sv_fwd + sv_adj) / (kt * 1e-3) / 1e9 / peak,
                         "sweep_frac_survey_bytes": (sv_fwd + sv_adj) / (ms_step * 1e-3) / 1e9 / peak,
                         "forward_frac_survey_bytes": sv_fwd / (t_f * 1e-3) / 1e9 / peak,
                         "survey_bytes_per_processed_point_step": (sv_fwd + sv_adj) / pts,
                         "target": "north_star's 0.60 is read against frac_survey_bytes / sweep_frac_survey_bytes (SURVEY.md 8(d): "
                                   "~61 B per processed point-step); frac uses this implementation's own count"},
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    g.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
