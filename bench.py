#!/usr/bin/env python
"""bench.py -- throughput of the whole enhanced-sampling hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl psg|reference]

A "step" is one pass of the whole path over one batch: psg_step for all R replicas / walkers / windows
of the workload (gather -> CVs + Jacobians -> deposit if due -> bias + gradient -> force scatter-add).
Default workload: BASELINE.json configs[1] (512-walker well-tempered metadynamics, 50,000 -> 60,240 hills,
deposits every 500 steps), the configuration the metric is quoted on.  Prints ONE JSON line.

  value     replica-bias-steps/s, inputs resident in HBM, L2 flushed between timed steps, CUDA events per step
  e2e       the same through psg_step_host: pinned HOST positions/forces, H2D + D2H inside the timed region
  roofline  the dominant kernel against its bound (ALU for the hill sum, HBM for the large-group kernels)
  cpu_baseline  the fp64 oracle, as it stands, on the box's host cores (a reported baseline, not the target)

--impl reference times the oracle alone (there is no reference implementation to install: /root/reference
holds only the paper).  N > 1 (torchrun): replicas are sharded by rank, weak scaling; see DESIGN.md "Multi-GPU".
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC, UNIT = "replica-bias-steps/sec", "replica-steps/s"
# FP32-pipe lane-instructions the METHOD needs per hill evaluation:
# per dimension sub, scale, fma(exponent), fma(gradient) = 4 (+3 if periodic: scaled rint, two-constant fma back);
# per hill: mul by height, add into V.  The MUFU.EX2 is counted separately.
def hill_eval_instr(n_cv, n_periodic):
    return 4 * n_cv + 3 * n_periodic + 2


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the committed ncu --set full
# captures (profiles/r1b_*_ncu_full.md); bytes
NCU_TRAFFIC = {1: 1.23e6, 2: 8.58e6, 3: 1.2412e9, 4: 5.87e6}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.p:
            return out
        time.sleep(0.12)
        self.p.terminate()
        try:
            txt, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            return out
        sm, mx, reasons = [], [], set()
        for line in txt.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------ workloads
def make_workload(cfg, K, W_):
    if cfg == 1:
        w = W.make(1, steps=K)          # capacity = 50,000 + (K // 500) * 512
    elif cfg == 0:
        w = W.make(0, steps=K)
    elif cfg == 2:
        w = W.make(2, steps=K, variant=os.environ.get("PSG_CFG2_VARIANT", "hit"))
    elif cfg == 3:
        w = W.make(3, steps=K)
    else:
        w = W.make(4, steps=K)
    if w.method == "metad":
        w.params["capacity"] += w.R     # psg_deposit_hill's host-side bound counts +R for a masked (ragged) round
    return w


def algorithmic_hill_evals(w, K):
    """sum over timed steps 1..K of R * n_hills(step) (deposits happen BEFORE the bias of their step)"""
    p = w.params
    n0, stride = p["n_hills"], p["stride"]
    if not stride:
        return float(w.R) * n0 * K
    s = np.arange(1, K + 1)
    return float((w.R * (n0 + (s // stride) * w.R)).sum())


# ------------------------------------------------------------------------------------------ multi-rank plumbing
def max_over_ranks(times_ms, world, device):
    """element-wise MAX over ranks of a list of per-rank times (the slowest rank defines the job's time)"""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_value(units_per_rank, world, ms):
    """replicas are sharded by rank with no data-path collective: weak scaling, the job
    processed world x units_per_rank units in the time of its slowest rank"""
    return float(units_per_rank) * world / (ms * 1e-3)



def per_call_table(ctx, w, frames, fsamp, force, to_dev, hbm_peak, fma_peak, n=20, reps=3):
    """each C-ABI call timed on its own (a CUDA graph of n calls, best of reps), with the roofline
    that bounds it where one applies; the force array keeps accumulating (pure +=), state (hills / grid) is static."""
    import torch
    main = torch.cuda.current_stream()
    s = torch.cuda.Stream()              # graphs are captured on a side stream; the ctx follows it for this table
    s.wait_stream(main)
    ctx.set_stream(s)
    try:
        with torch.cuda.stream(s):
            return _per_call_table(ctx, w, frames, fsamp, force, hbm_peak, fma_peak, n, reps, s)
    finally:
        torch.cuda.synchronize()
        ctx.set_stream(main)


def _per_call_table(ctx, w, frames, fsamp, force, hbm_peak, fma_peak, n, reps, s):
    import torch
    pos = frames[0]
    xi = torch.empty((w.R, w.n_cv), device=pos.device)
    V = torch.empty(w.R, device=pos.device)
    dV = torch.zeros((w.R, w.n_cv), device=pos.device)
    ctx.cv_eval(pos, xi, None)
    calls = {"psg_cv_eval": lambda: ctx.cv_eval(pos, xi, None)}
    if w.method == "abf":
        calls["psg_abf_update"] = lambda: ctx.abf_update(xi, fsamp[0], None, dV)
    else:
        calls["psg_bias_eval"] = lambda: ctx.bias_eval(xi, V, dV)
    calls["psg_apply_bias_forces"] = lambda: ctx.apply_bias_forces(pos, dV, force)
    calls["psg_step"] = lambda: ctx.step(pos, force, None if fsamp is None else fsamp[0], -1)
    out = {}
    for name, fn in calls.items():
        fn(); torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for _ in range(n):
                fn()
        g.replay(); torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); g.replay(); b.record(); torch.cuda.synchronize()
            best = min(best, a.elapsed_time(b) / n * 1e3)
        out[name] = {"us": round(best, 2)}
    n_range_atoms = sum(g[2] for cv in w.cvs for g in cv["groups"] if g[0] == "range")
    if n_range_atoms and not w.shared_array:
        span = w.R * w.N
        out["psg_cv_eval"].update(bound="hbm", frac=round(16.0 * span / (out["psg_cv_eval"]["us"] * 1e-6) / 1e9 / hbm_peak, 3),
                                  algorithmic_bytes=16.0 * span)
        out["psg_apply_bias_forces"].update(bound="hbm", algorithmic_bytes=48.0 * span,
                                            frac=round(48.0 * span / (out["psg_apply_bias_forces"]["us"] * 1e-6) / 1e9 / hbm_peak, 3))
        out["psg_step"].update(bound="hbm", algorithmic_bytes=48.0 * span,
                               frac=round(48.0 * span / (out["psg_step"]["us"] * 1e-6) / 1e9 / hbm_peak, 3))
    if w.method == "metad":
        C = hill_eval_instr(w.n_cv, int((w.period > 0).sum()))
        work = float(w.R) * ctx.n_hills() * C
        for k in ("psg_bias_eval", "psg_step"):
            out[k].update(bound="alu", frac=round(work / (out[k]["us"] * 1e-6) / fma_peak, 3))
    return out


# ------------------------------------------------------------------------------------------ psg arm
def run_psg(args, rank, world):
    import torch
    import torch.distributed as dist
    import paper_2301_04835_b200 as psg

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    K, Wm = args.steps, args.warmup
    w = make_workload(args.config, K, Wm)
    ctx = psg.Context(local)
    psg.configure_from_workload(ctx, w)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    # ---- state: the pre-filled hill list is produced by the product's own deposit path, in the workload's rounds
    hills0 = None
    if w.method == "metad":
        c = w.params["hill_centers"]
        for b, e in w.hill_rounds():
            xi = np.zeros((w.R, w.n_cv), np.float32)
            xi[: e - b] = c[b:e]
            mask = None
            if e - b < w.R:
                mask = np.zeros(w.R, np.uint8); mask[: e - b] = 1
            ctx.deposit_hill(to_dev(xi), None if mask is None else to_dev(mask))
        hills0 = ctx.get_hills()
        assert hills0[1].shape[0] == w.params["n_hills"]
    frames = [to_dev(w.positions(k)) for k in range(w.K)]
    fsamp = [to_dev(w.fsample(k)) for k in range(w.K)] if w.method == "abf" else None
    f0 = w.forces0()
    force = to_dev(f0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # 256 MiB > 126 MB L2

    def step(s):
        ctx.step(frames[s % w.K], force, None if fsamp is None else fsamp[s % w.K], s)

    def reset_state():
        if hills0 is not None:
            ctx.load_hills(hills0[0], hills0[1])
        if w.method == "abf":
            ctx.set_abf(w.params["lower"], w.params["upper"], w.params["shape"], w.params["periodic"],
                        w.params["n_threshold"])
        force.copy_(to_dev(f0))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- timed region 1 (the reported value): per-step CUDA events, L2 flushed between steps
    for s in range(Wm):
        step(-(s + 1))                       # step numbers <= 0 never deposit
    reset_state()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    launches0 = ctx.launch_count()
    clk = ClockSampler(local) if rank == 0 and not args.no_clock_sampler else None
    barrier()
    t_wall = time.perf_counter()
    for s in range(1, K + 1):
        flush.zero_()
        ev0[s - 1].record()
        step(s)
        ev1[s - 1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall
    launches = ctx.launch_count() - launches0
    ctx.sync_check()
    per_step = np.array([a.elapsed_time(b) for a, b in zip(ev0, ev1)])      # ms
    ms_total = float(per_step.sum())

    # ---- timed region 2 (context): the same K steps back to back, no flush, two events
    reset_state()
    barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for s in range(1, K + 1):
        step(s)
    b.record()
    barrier()
    ms_b2b = a.elapsed_time(b)
    clocks = clk.stop() if clk else None

    # ---- e2e: HOST arrays through psg_step_host (H2D positions + forces, D2H forces, every step)
    Ke = min(K, args.e2e_steps)
    h_frames = [torch.from_numpy(w.positions(k)).pin_memory() for k in range(w.K)]
    h_fs = [torch.from_numpy(w.fsample(k)).pin_memory() for k in range(w.K)] if w.method == "abf" else None
    h_force = torch.from_numpy(f0.copy()).pin_memory()
    reset_state()
    for s in range(3):
        ctx.step_host(h_frames[s % w.K], h_force, None if h_fs is None else h_fs[s % w.K], -(s + 1))
    barrier()
    a.record()
    for s in range(1, Ke + 1):
        ctx.step_host(h_frames[s % w.K], h_force, None if h_fs is None else h_fs[s % w.K], s)
    b.record()
    barrier()
    ms_e2e = a.elapsed_time(b)
    h2d = h_frames[0].numel() * 4 + h_force.numel() * 4 + (h_fs[0].numel() * 4 if h_fs else 0)
    d2h = h_force.numel() * 4

    # ---- max over ranks
    ms_total, ms_b2b, ms_e2e = max_over_ranks([ms_total, ms_b2b, ms_e2e], world, dev)

    out = None
    if rank == 0:
        units = float(w.R) * K * world
        value = whole_job_value(float(w.R) * K, world, ms_total)
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
               "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f32", "data": "synthetic",
               "config": {"workload": f"BASELINE.json configs[{args.config}] ({w.name}): R={w.R} replicas x N={w.N} atoms, "
                                      f"{w.n_cv} CVs, method={w.method}", "replicas_per_gpu": w.R, "parallelism": f"replicas x{world}",
                          "l2": "flushed between timed steps (256 MiB memset outside the per-step event pairs)",
                          "position_frames": w.K},
               "e2e": {"value": float(w.R) * Ke * world / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "steps": Ke, "api": "psg_step_host (pinned host buffers)"},
               "gpu_launches": int(launches), "clocks": clocks,
               "back_to_back": {"value": units / (ms_b2b * 1e-3), "unit": UNIT, "ms_per_step": ms_b2b / K,
                                "note": "same K steps, no L2 flush, two events around the whole loop"},
               "wall_s_timed_region": t_wall,
               "per_step_us": {"min": float(per_step.min() * 1e3), "median": float(np.median(per_step) * 1e3),
                               "p99": float(np.percentile(per_step, 99) * 1e3), "max": float(per_step.max() * 1e3)}}
        hbm_peak, which = _peaks()
        if w.method == "metad":
            evals = algorithmic_hill_evals(w, K)
            nper = int((w.period > 0).sum())
            C = hill_eval_instr(w.n_cv, nper)
            fma_peak = psg.measure_alu_peak(0, local)            # FP32 FFMA lane-instructions/s, measured here
            mufu_peak = psg.measure_alu_peak(2, local)
            ffma2_peak = psg.measure_alu_peak(1, local)
            ach = evals * C / (ms_total * 1e-3)
            out["hill_evals_per_s"] = evals * world / (ms_total * 1e-3)
            out["roofline"] = {"bound": "alu", "kernel": "k_hills (fused step)", "achieved": ach / 1e9, "peak": fma_peak / 1e9,
                               "unit": "G FP32 lane-instr/s", "frac": ach / fma_peak, "traffic": NCU_TRAFFIC.get(args.config),
                               "peak_source": "psg_measure_alu_peak(FFMA), measured in this run (burst, kernel timed alone)",
                               "instr_per_hill_eval": C, "mufu_peak_Gops": mufu_peak / 1e9, "ffma2_peak_Glaneops": ffma2_peak / 1e9,
                               "mufu_frac": (evals / (ms_total * 1e-3)) / mufu_peak,
                               "frac_back_to_back": evals * C / (ms_b2b * 1e-3) / fma_peak}
        elif w.method == "harmonic":
            bytes_step = 48.0 * w.R * w.N                          # read pos once + read force + write force (float4)
            ach = bytes_step * K / (ms_total * 1e-3) / 1e9
            out["roofline"] = {"bound": "hbm", "kernel": "k_range_step (fused umbrella step, one launch)", "achieved": ach, "peak": hbm_peak,
                               "unit": "GB/s", "frac": ach / hbm_peak, "traffic": NCU_TRAFFIC.get(args.config),
                               "peak_source": which + " copy bandwidth", "algorithmic_bytes_per_step": bytes_step,
                               "frac_back_to_back": bytes_step * K / (ms_b2b * 1e-3) / 1e9 / hbm_peak}
        else:
            bytes_step = float(w.R) * (8 * 32 + 3 * 32 + 8 * 32 * 2)
            ach = bytes_step * K / (ms_total * 1e-3) / 1e9
            out["roofline"] = {"bound": "hbm", "kernel": "k_abf_step (fused ABF step, one launch; latency-bound)", "achieved": ach,
                               "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": NCU_TRAFFIC.get(args.config),
                               "peak_source": which + " copy bandwidth",
                               "note": "a step moves < 4 MB: launch latency, not HBM, bounds it (DESIGN.md)"}
        if world == 1 and not args.skip_per_call:
            reset_state()
            out["per_call"] = per_call_table(ctx, w, frames, fsamp, force, to_dev, hbm_peak,
                                             psg.measure_alu_peak(0, local) if w.method == "metad" else 1.0)
            out["per_call"]["note"] = "graph replay of 20 calls each, L2 warm; us per call"
        if not args.skip_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(w, budget_s=args.cpu_budget)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return out


# ------------------------------------------------------------------------------------------ oracle legs
def _oracle_setup(w, Rs):
    """oracle structs for the first Rs replicas of workload w (a bounded sample of the same workload)"""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle as orc
    from _parity import oracle_heights, oracle_system
    import copy
    ws = copy.copy(w)
    ws.R = Rs
    if w.slot_atom is not None and w.slot_atom.ndim == 2:
        ws.slot_atom = w.slot_atom[:Rs]
    ws.params = dict(w.params)
    if w.method == "harmonic":
        ws.params["centers"] = w.params["centers"][:Rs]
    sysm = oracle_system(ws)
    return orc, ws, sysm, oracle_heights


def _oracle_step_fn(w, Rs):
    orc, ws, sysm, oracle_heights = _oracle_setup(w, Rs)
    from _parity import oracle_step
    centers = heights = abf = None
    if w.method == "metad":
        centers, heights = w.params["hill_centers"], oracle_heights(w)
    if w.method == "abf":
        nb = int(np.prod(w.params["shape"]))
        abf = (np.zeros(nb, np.int32), np.zeros((nb, w.n_cv), np.float64))
    n_arr = 1 if w.shared_array else Rs
    frames = [w.positions(k)[:n_arr] for k in range(min(w.K, 2))]
    fs = [w.fsample(k)[:Rs] for k in range(min(w.K, 2))] if w.method == "abf" else None
    f0 = w.forces0()[:n_arr]

    def step(s):
        k = s % len(frames)
        return oracle_step(ws, sysm, frames[k], f0, centers, heights, abf, None if fs is None else fs[k])
    return orc, step


def cpu_baseline(w, budget_s=15.0):
    """the oracle as it stands, all host cores (OpenMP over replicas), on a bounded sample: whole steps of the
    full batch, as many as fit the budget (at least 1)."""
    orc, step = _oracle_step_fn(w, w.R)
    t0 = time.perf_counter(); step(0); t1 = time.perf_counter() - t0
    n = int(max(1, min(50, budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    for s in range(n):
        step(s + 1)
    dt = time.perf_counter() - t0
    return {"value": w.R * n / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": f"{n} whole steps of the full batch (R={w.R}), fp64, hill list static, {dt / n * 1e3:.1f} ms/step",
            "host_cores_available": len(os.sched_getaffinity(0))}


def run_reference(args, rank, world):
    if rank != 0:
        return None
    K, Wm = args.steps, args.warmup
    w = make_workload(args.config, K, Wm)
    # bounded sample: the first Rs replicas, Rs chosen so that K + W steps take about args.ref_budget seconds
    orc, step = _oracle_step_fn(w, min(w.R, 8))
    t0 = time.perf_counter(); step(0); t1 = (time.perf_counter() - t0) / min(w.R, 8)
    Rs = int(max(1, min(w.R, args.ref_budget / max(t1 * (K + Wm), 1e-9))))
    orc, step = _oracle_step_fn(w, Rs)
    for s in range(Wm):
        step(s)
    t0 = time.perf_counter()
    for s in range(1, K + 1):
        step(s)
    dt = time.perf_counter() - t0
    v = Rs * K / dt
    sample = f"first {Rs} of {w.R} replicas per step, all hills / atoms of those replicas, fp64 oracle"
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": dt / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config}] ({w.name}): R={w.R} replicas x N={w.N} atoms, "
                                   f"{w.n_cv} CVs, method={w.method}", "sample": sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="psg", choices=["psg", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2000)
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--ref-budget", type=float, default=60.0)
    ap.add_argument("--skip-cpu-baseline", action="store_true")
    ap.add_argument("--skip-per-call", action="store_true")
    ap.add_argument("--no-clock-sampler", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    out = run_reference(args, rank, world) if args.impl == "reference" else run_psg(args, rank, world)
    if rank == 0 and out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
