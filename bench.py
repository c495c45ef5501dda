#!/usr/bin/env python
"""bench.py -- throughput of the whole enhanced-sampling hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl psg|reference] [--no-per-config]

A "step" is one pass of the whole path over one batch: psg_step for all R replicas / walkers / windows
of the workload (gather -> CVs + Jacobians -> deposit if due -> bias + gradient -> force scatter-add).
Headline workload: BASELINE.json configs[4], the largest single-GPU configuration (1,024 walkers on one shared
1,000,000-atom array, 3 CVs, 200,000 hills); BASELINE.json's `metric` names no configuration.  Prints ONE JSON line.

  value     replica-bias-steps/s, inputs resident in HBM, L2 flushed between timed steps, one CUDA-event pair per step
            (= per launch: a step is one launch); rounds of K steps are repeated until >= 50 ms of event time, so the
            number does not depend on --steps being large
  e2e       the same through psg_step_host: pinned HOST positions/forces, H2D + D2H inside the timed region
  roofline  the dominant kernel against its bound (ALU for the hill sum, HBM for the large-group kernels)
  cpu_baseline  the fp64 oracle, as it stands, on the box's host cores (a reported baseline, not the target)
  per_config    the same measurements for every BASELINE.json config 0..4 (N = 1 only)

--impl reference times the oracle alone (there is no reference implementation to install: /root/reference
holds only the paper).  N > 1 (torchrun): replicas are sharded by rank, weak scaling; the shared-state methods run
their one exchange (hill all-gather at a deposit, ABF grid all-reduce per step); see DESIGN.md "Multi-GPU".
"""
from __future__ import annotations

import argparse
import gc
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
MIN_TIMED_MS = 50.0          # event time the timed rounds must add up to
MAX_TIMED_STEPS = 6000       # ... but never more steps than this (config 0: ~10 us per step)
E2E_CAP = {2: 2, 3: 2}       # configs whose step moves GBs over PCIe: a few steps are enough (6.6 GB / 1.2 GB per step)


# FP32-pipe lane-instructions the METHOD needs per hill evaluation:
# per dimension sub, scale, fma(exponent), fma(gradient) = 4 (+3 if periodic: scaled rint, two-constant fma back);
# per hill: mul by height, add into V.  The MUFU.EX2 is counted separately.
def hill_eval_instr(n_cv, n_periodic):
    return 4 * n_cv + 3 * n_periodic + 2


# FP64-pipe lane-instructions per hill evaluation of the binary64-term mode (PSG_HILLS_F64): the same
# C as above plus a software exp(): range reduction 4, degree-11 polynomial 11, scaling 3
def hill_eval_instr_f64(n_cv, n_periodic):
    return hill_eval_instr(n_cv, n_periodic) + 18


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, bytes, NOT measured in this run:
# copied from the committed ncu --set full captures named here
NCU_TRAFFIC = {1: (1.224e6, "profiles/r2_hills_config1_ncu_full.md"), 2: (8.52e6, "profiles/r2b_abf_step_config2_ncu_full.md"),
               3: (1.2412e9, "profiles/r1b_range_step_config3_ncu_full.md"), 4: (5.98e6, "profiles/r2_hills_config4_ncu_full.md")}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json copy bandwidth (driver-written)"
    return 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            time.sleep(0.15)      # let the first sample arrive before the timed region starts
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.p:
            return out
        time.sleep(0.05)
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
def make_workload(cfg, steps, world=1):
    """the BASELINE.json config at full size; metadynamics stores get room for every deposit of `steps` steps on
    `world` ranks (a deposit event appends the walkers of ALL ranks)"""
    if cfg == 2:
        w = W.make(2, steps=steps, variant=os.environ.get("PSG_CFG2_VARIANT", "hit"))
    else:
        w = W.make(cfg, steps=steps)
    if w.method == "metad":
        p = w.params
        n_dep = (steps // p["stride"] + 1) if p["stride"] else 0
        p["capacity"] = p["n_hills"] + n_dep * w.R * world
    return w


def workload_config(cfg, w, world):
    """the `config` object of the JSON line; both arms print the same one"""
    return {"workload": f"BASELINE.json configs[{cfg}] ({w.name}): R={w.R} replicas x N={w.N} atoms, "
                        f"{w.n_cv} CVs, method={w.method}", "replicas_per_gpu": w.R, "parallelism": f"replicas x{world}",
            "l2": "flushed between timed steps (256 MiB memset outside the per-step event pairs)", "position_frames": w.K}


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
    """replicas are sharded by rank: weak scaling, the job processed world x units_per_rank
    units in the time of its slowest rank"""
    return float(units_per_rank) * world / (ms * 1e-3)


class Peaks:
    """roofline denominators measured once per process (psg_measure_alu_peak: register-only loops, burst)"""

    def __init__(self, psg, local):
        self.hbm, self.hbm_source = _peaks()
        self.ffma = psg.measure_alu_peak(0, local)
        self.ffma2 = psg.measure_alu_peak(1, local)
        self.mufu = psg.measure_alu_peak(2, local)
        self.dfma = psg.measure_alu_peak(3, local)
        self.f64_exp = psg.measure_alu_peak(10, local)                     # binary64 exp() per second
        self.t_floor_us = 1e6 / psg.measure_alu_peak(9, local)            # empty kernel node of a replayed graph
        self.t_event_floor_us = 1e6 / psg.measure_alu_peak(11, local)     # empty kernel between two event records after a flush


# ------------------------------------------------------------------------------------------ one config on this rank
class ConfigRun:
    def __init__(self, cfg, args, rank, world, local, psg, torch, dist):
        self.cfg, self.args, self.rank, self.world, self.local = cfg, args, rank, world, local
        self.psg, self.torch, self.dist = psg, torch, dist
        self.dev = torch.device("cuda", local)
        self.max_steps = MAX_TIMED_STEPS
        self.w = w = make_workload(cfg, self.max_steps + 64, world)
        self.ctx = ctx = psg.Context(local)
        psg.configure_from_workload(ctx, w)
        to_dev = self.to_dev
        # the pre-filled hill list is produced by the product's own deposit path, in the workload's rounds
        self.hills0 = None
        if w.method == "metad":
            c = w.params["hill_centers"]
            for b, e in w.hill_rounds():
                xi = np.zeros((w.R, w.n_cv), np.float32)
                xi[: e - b] = c[b:e]
                mask = None
                if e - b < w.R:
                    mask = np.zeros(w.R, np.uint8); mask[: e - b] = 1
                ctx.deposit_hill(to_dev(xi), None if mask is None else to_dev(mask))
            self.hills0 = ctx.get_hills()
            assert self.hills0[1].shape[0] == w.params["n_hills"]
        self.frames = [to_dev(w.positions(k)) for k in range(w.K)]
        self.fsamp = [to_dev(w.fsample(k)) for k in range(w.K)] if w.method == "abf" else None
        self.f0 = w.forces0()
        self.force = to_dev(self.f0)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)      # 256 MiB > 126 MB L2
        self.xi_scratch = torch.empty((w.R, w.n_cv), device=self.dev)
        self.n_periodic = int((w.period > 0).sum())

    def to_dev(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a)).to(self.dev)

    def close(self):
        self.ctx.close()
        for k in ("frames", "fsamp", "force", "flush", "hills0", "xi_scratch"):
            setattr(self, k, None)
        self.w._extra.clear()
        gc.collect()
        self.torch.cuda.empty_cache()

    # ---- one MD step of this rank's replicas; with several ranks the shared-state methods exchange
    def step(self, s):
        w, ctx = self.w, self.ctx
        pos = self.frames[s % w.K]
        fs = None if self.fsamp is None else self.fsamp[s % w.K]
        if self.world > 1 and w.method == "metad" and w.params["stride"] and s > 0 and s % w.params["stride"] == 0:
            from paper_2301_04835_b200 import multiwalker
            ctx.cv_eval(pos, self.xi_scratch, None)
            multiwalker.deposit_hill_all_ranks(ctx, self.xi_scratch)      # all-gather of every rank's new hills
            ctx.step(pos, self.force, None, 0)                            # step numbers <= 0 never deposit
        elif self.world > 1 and w.method == "abf":
            from paper_2301_04835_b200 import multiwalker
            multiwalker.abf_step_all_ranks(ctx, pos, self.force, fs)      # all-reduce of the grid deltas
        else:
            ctx.step(pos, self.force, fs, s)

    def n_hills_at(self, s):
        """hill count the bias of step s sums over (a deposit happens BEFORE the bias of its step)"""
        p = self.w.params
        if not p.get("stride"):
            return p["n_hills"]
        return p["n_hills"] + (s // p["stride"]) * self.w.R * self.world

    def reset_state(self):
        w, ctx = self.w, self.ctx
        if self.hills0 is not None:
            ctx.load_hills(self.hills0[0], self.hills0[1])
        if w.method == "abf":
            ctx.set_abf(w.params["lower"], w.params["upper"], w.params["shape"], w.params["periodic"], w.params["n_threshold"])
        self.force.copy_(self.to_dev(self.f0))

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
            self.torch.cuda.synchronize()

    # ---- timed region: rounds of K steps, one event pair per step, L2 flushed between steps, until >= min_ms
    def timed(self, K, Wm, min_ms=MIN_TIMED_MS):
        torch = self.torch
        for s in range(Wm):
            self.step(-(s + 1))                       # step numbers <= 0 never deposit
        self.reset_state()
        launches0 = self.ctx.launch_count()
        per_step, s, rounds = [], 0, 0
        self.barrier()
        t_wall = time.perf_counter()
        while True:
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
            for a, b in ev:
                s += 1
                self.flush.zero_()
                a.record()
                self.step(s)
                b.record()
            self.barrier()
            rounds += 1
            per_step += [a.elapsed_time(b) for a, b in ev]
            total = max_over_ranks([sum(per_step)], self.world, self.dev)[0]      # every rank takes the same decision
            if total >= min_ms or s + K > self.max_steps:
                break
        t_wall = time.perf_counter() - t_wall
        self.ctx.sync_check()
        per_step = np.array(per_step)                                             # ms, this rank
        per_step_max = np.array(max_over_ranks(per_step, self.world, self.dev))   # ms, slowest rank per step
        return {"per_step_ms": per_step_max, "steps": s, "rounds": rounds, "launches": self.ctx.launch_count() - launches0,
                "wall_s": t_wall}

    def back_to_back(self, K):
        torch = self.torch
        self.reset_state()
        self.barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for s in range(1, K + 1):
            self.step(s)
        b.record()
        self.barrier()
        return max_over_ranks([a.elapsed_time(b)], self.world, self.dev)[0]

    # ---- e2e: HOST arrays through psg_step_host (H2D positions + forces, D2H forces, every step)
    def e2e(self, K):
        torch, w, ctx = self.torch, self.w, self.ctx
        cap = E2E_CAP.get(self.cfg)
        nf = 1 if cap else min(w.K, 2)
        h_frames = [torch.from_numpy(w.positions(k)).pin_memory() for k in range(nf)]
        h_fs = [torch.from_numpy(w.fsample(k)).pin_memory() for k in range(nf)] if w.method == "abf" else None
        h_force = torch.from_numpy(self.f0.copy()).pin_memory()
        self.reset_state()
        call = lambda s, n: ctx.step_host(h_frames[s % nf], h_force, None if h_fs is None else h_fs[s % nf], n)
        for s in range(1 if cap else 3):
            call(s, -(s + 1))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n, ms = 0, 0.0
        while True:
            Ke = cap or K
            self.barrier()
            a.record()
            for s in range(n + 1, n + Ke + 1):
                call(s, s)
            b.record()
            self.barrier()
            n += Ke
            ms += max_over_ranks([a.elapsed_time(b)], self.world, self.dev)[0]
            if cap or ms >= 20.0 or n + K > 2000:
                break
        h2d = h_frames[0].numel() * 4 + h_force.numel() * 4 + (h_fs[0].numel() * 4 if h_fs else 0)
        d2h = h_force.numel() * 4
        del h_frames, h_force, h_fs
        return {"value": whole_job_value(float(w.R) * n, self.world, ms), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": n, "api": "psg_step_host (pinned host buffers)"}

    # ---- graph replay of n identical calls of fn on a side stream: us per call, best of reps
    def graph_us(self, fn, n=20, reps=3):
        torch, ctx = self.torch, self.ctx
        main = torch.cuda.current_stream()
        s = torch.cuda.Stream()
        s.wait_stream(main)
        ctx.set_stream(s)
        try:
            with torch.cuda.stream(s):
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
                return best
        finally:
            torch.cuda.synchronize()
            ctx.set_stream(main)

    def per_call(self, pk):
        """each C-ABI call timed on its own (a CUDA graph of 20 calls, best of 3), with the roofline that
        bounds it where one applies; the force array keeps accumulating (pure +=), state (hills / grid) is static."""
        torch, w, ctx = self.torch, self.w, self.ctx
        self.reset_state()
        pos = self.frames[0]
        xi = torch.empty((w.R, w.n_cv), device=self.dev)
        V = torch.empty(w.R, device=self.dev)
        dV = torch.zeros((w.R, w.n_cv), device=self.dev)
        ctx.cv_eval(pos, xi, None)
        calls = {"psg_cv_eval": lambda: ctx.cv_eval(pos, xi, None)}
        if w.method == "abf":
            calls["psg_abf_update"] = lambda: ctx.abf_update(xi, self.fsamp[0], None, dV)
        else:
            calls["psg_bias_eval"] = lambda: ctx.bias_eval(xi, V, dV)
        calls["psg_apply_bias_forces"] = lambda: ctx.apply_bias_forces(pos, dV, self.force)
        calls["psg_step"] = lambda: ctx.step(pos, self.force, None if self.fsamp is None else self.fsamp[0], -1)
        out = {name: {"us": round(self.graph_us(fn), 2)} for name, fn in calls.items()}
        n_range_atoms = sum(g[2] for cv in w.cvs for g in cv["groups"] if g[0] == "range")
        if n_range_atoms and not w.shared_array:
            span = w.R * w.N
            for k, bpa in (("psg_cv_eval", 16.0), ("psg_apply_bias_forces", 48.0), ("psg_step", 48.0)):
                out[k].update(bound="hbm", algorithmic_bytes=bpa * span,
                              frac=round(bpa * span / (out[k]["us"] * 1e-6) / 1e9 / pk.hbm, 3))
        if w.method == "metad":
            work = float(w.R) * ctx.n_hills() * hill_eval_instr(w.n_cv, self.n_periodic)
            for k in ("psg_bias_eval", "psg_step"):
                out[k].update(bound="alu", frac=round(work / (out[k]["us"] * 1e-6) / pk.ffma, 3))
        out["note"] = "graph replay of 20 calls each, L2 warm; us per call"
        return out

    def hills_f64(self, pk):
        """the binary64-term mode (PSG_HILLS_F64), the one that meets the literal 1e-5 / 1e-6 rule on ill-conditioned
        gradients: the fused step on the same inputs, L2 flushed, per-step events"""
        torch, w, ctx, psg = self.torch, self.w, self.ctx, self.psg
        self.reset_state()
        ctx.set_hill_precision(psg.HILLS_F64)
        try:
            for s in range(3):
                ctx.step(self.frames[s % w.K], self.force, None, -1)
            n = 20 if self.cfg != 4 else 5
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
            for i, (a, b) in enumerate(ev):
                self.flush.zero_()
                a.record()
                ctx.step(self.frames[i % w.K], self.force, None, -1)
                b.record()
            torch.cuda.synchronize()
            t = np.array([a.elapsed_time(b) for a, b in ev])
        finally:
            ctx.set_hill_precision(psg.HILLS_F32)
        evals = float(w.R) * w.params["n_hills"]
        C64 = hill_eval_instr_f64(w.n_cv, self.n_periodic)
        return {"us_per_step": float(t.mean() * 1e3), "us_per_step_median": float(np.median(t) * 1e3), "steps": n,
                "evals_per_s": evals / (t.mean() * 1e-3), "replica_steps_per_s": w.R / (t.mean() * 1e-3),
                "fp64_instr_per_hill_eval": C64, "dfma_peak_Glaneops": pk.dfma / 1e9,
                "frac_vs_measured_DFMA_peak": evals * C64 / (t.mean() * 1e-3) / pk.dfma,
                "note": "binary64 terms on the FP64 pipe; passes the literal tolerance at full size (tests/test_gpu_fullsize.py)"}

    def deposit_event(self):
        """config 1: one forced deposit event inside a timed region: psg_step at a multiple of the stride
        (CVs -> V_old of every walker under the old list -> heights -> append -> fused step) against the plain step"""
        torch, w, ctx = self.torch, self.w, self.ctx
        stride = w.params["stride"]
        out = []
        for dep in (True, False):
            t = []
            for i in range(5):
                self.reset_state()
                ctx.step(self.frames[0], self.force, None, -1)
                self.flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                ctx.step(self.frames[1 % w.K], self.force, None, stride if dep else -1)
                b.record()
                torch.cuda.synchronize()
                t.append(a.elapsed_time(b) * 1e3)
            out.append(float(np.median(t)))
        self.reset_state()
        return {"step_with_deposit_us": out[0], "plain_step_us": out[1], "deposit_event_us": out[0] - out[1],
                "hills_appended": w.R, "amortised_us_per_step": (out[0] - out[1]) / stride,
                "note": "median of 5, L2 flushed; the event = psg_cv_eval + V_old pass of k_hills + k_deposit"}

    def grid_metad(self, pk):
        """SURVEY NEXT-2, the paper's own speed option: the same walkers with the bias STORED ON A GRID
        (psg_set_metad_grid, reading R-GRID): the workload's hill list is deposited onto the grid by the method's own
        deposit, then psg_step interpolates.  The step is latency-bound (reported against the event-pair floor); the
        deposit event is bound by the binary64 exponential (one per node and hill)."""
        torch, w, psg = self.torch, self.w, self.psg
        p = w.params
        if self.cfg == 1:
            lower, upper, shape, periodic = (-np.pi, -np.pi), (np.pi, np.pi), (256, 256), (1, 1)
        else:
            lower, upper, shape, periodic = (-np.pi, -np.pi, 0.2), (np.pi, np.pi, 1.6), (64, 64, 64), (1, 1, 0)
        ctx = psg.Context(self.local)
        psg.configure_from_workload(ctx, w, with_method=False)
        ctx.set_metad_grid(lower, upper, shape, periodic, p["sigma"].astype(np.float64), p["w0"], p["kB_deltaT"], 0)
        c = p["hill_centers"]
        ev_t = []
        for b, e in w.hill_rounds():
            xi = np.zeros((w.R, w.n_cv), np.float32)
            xi[: e - b] = c[b:e]
            mask = None
            if e - b < w.R:
                mask = np.zeros(w.R, np.uint8); mask[: e - b] = 1
            d_xi, d_m = self.to_dev(xi), None if mask is None else self.to_dev(mask)
            a, bb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); ctx.deposit_hill(d_xi, d_m); bb.record()
            ev_t.append((a, bb, e - b))
        torch.cuda.synchronize()
        full = [a.elapsed_time(b) * 1e3 for a, b, n in ev_t if n == w.R]
        dep_us = float(np.median(full))
        nodes = int(np.prod(shape))
        n = 200
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for i in range(5):
            ctx.step(self.frames[i % w.K], self.force, None, -1)
        for i, (a, b) in enumerate(evs):
            self.flush.zero_(); a.record(); ctx.step(self.frames[i % w.K], self.force, None, -1); b.record()
        torch.cuda.synchronize()
        t = np.array([a.elapsed_time(b) for a, b in evs]) * 1e3
        old, self.ctx = self.ctx, ctx
        try:
            g_us = self.graph_us(lambda: ctx.step(self.frames[0], self.force, None, -1))
        finally:
            self.ctx = old
        ctx.close()
        gauss = float(w.R) * nodes / (dep_us * 1e-6)
        return {"grid_shape": list(shape), "nodes": nodes, "hills_on_grid": int(p["n_hills"]),
                "step_us_flushed_median": float(np.median(t)), "step_us_graph_replay": g_us, "launches_per_step": 1,
                "frac_of_event_floor": pk.t_event_floor_us / float(np.median(t)),
                "deposit_event_us": dep_us, "deposit_gaussians_per_s": gauss, "f64_exp_peak_per_s": pk.f64_exp,
                "deposit_frac_of_f64_exp_peak": gauss / pk.f64_exp,
                "note": "step: one launch whatever the number of hills (O(1) per walker); deposit: R hills onto every node, "
                        "one binary64 exp per (hill, node), amortised over `stride` steps"}

    def abf_estimate(self):
        """the instantaneous-force estimator that produces ABF's fsample (psg_abf_estimate), on this config's
        replicas; graph replay of 20 calls (latency-bound: a few KB per replica)"""
        torch, w, ctx = self.torch, self.w, self.ctx
        pos = self.frames[0]
        vel = torch.randn_like(pos) * 0.5
        mass = torch.ones(w.N, device=self.dev)
        fprev = torch.zeros((w.R, w.n_cv), device=self.dev)
        fs = torch.empty((w.R, w.n_cv), device=self.dev)
        us = self.graph_us(lambda: ctx.abf_estimate(pos, vel, mass, 0.002, fprev, fs))
        del vel
        return {"us_per_call_graph_replay": us, "replicas": w.R, "note": "one launch: Jacobians, J J^T solve, second-order backward difference"}

    # ---- the roofline of the dominant kernel from the per-step (= per-launch) event times
    def roofline(self, tr, pk, b2b_ms_per_step):
        w, cfg = self.w, self.cfg
        t = tr["per_step_ms"]
        ms_total, n = float(t.sum()), len(t)
        traffic = NCU_TRAFFIC.get(cfg)
        common = {"traffic": traffic[0] if traffic else None,
                  "traffic_source": (f"from {traffic[1]} (one launch under ncu --set full), not measured in this run" if traffic
                                     else "no capture of this config")}
        if w.method == "metad":
            C = hill_eval_instr(w.n_cv, self.n_periodic)
            evals = float(sum(w.R * self.n_hills_at(s) for s in range(1, n + 1)))
            ach = evals * C / (ms_total * 1e-3)
            r = {"bound": "alu", "kernel": "k_hills (fused step)", "achieved": ach / 1e9, "peak": pk.ffma / 1e9,
                 "unit": "G FP32 lane-instr/s", "frac": ach / pk.ffma,
                 "peak_source": "psg_measure_alu_peak(FFMA), measured in this run (burst, kernel timed alone)",
                 "instr_per_hill_eval": C, "algorithmic_units_per_step": evals / n * C,
                 "algorithmic_units": "FP32 lane-instructions (hill-evals x C)",
                 "mufu_peak_Gops": pk.mufu / 1e9, "ffma2_peak_Glaneops": pk.ffma2 / 1e9,
                 "mufu_frac": (evals / (ms_total * 1e-3)) / pk.mufu,
                 "frac_back_to_back": evals / n * C / (b2b_ms_per_step * 1e-3) / pk.ffma,
                 "hill_evals_per_s": evals / (ms_total * 1e-3)}
            model_us = evals / n * C / pk.ffma * 1e6
        elif w.method == "harmonic":
            bytes_step = 48.0 * w.R * w.N                          # read pos once + read force + write force (float4)
            ach = bytes_step * n / (ms_total * 1e-3) / 1e9
            r = {"bound": "hbm", "kernel": "k_range_step (fused umbrella step, one launch)", "achieved": ach, "peak": pk.hbm,
                 "unit": "GB/s", "frac": ach / pk.hbm, "peak_source": pk.hbm_source, "algorithmic_units_per_step": bytes_step,
                 "algorithmic_units": "bytes (48 B/atom)",
                 "frac_back_to_back": bytes_step / (b2b_ms_per_step * 1e-3) / 1e9 / pk.hbm}
            model_us = bytes_step / (pk.hbm * 1e9) * 1e6
        else:
            bytes_step = float(w.R) * (8 * 32 + 3 * 32 + 8 * 32 * 2)   # sectors: 8 gathered, <= 3 grid RMW, 8 force RMW
            ach = bytes_step * n / (ms_total * 1e-3) / 1e9
            r = {"bound": "hbm", "kernel": "k_abf_step_lean (fused ABF step, one launch; latency-bound)", "achieved": ach,
                 "peak": pk.hbm, "unit": "GB/s", "frac": ach / pk.hbm, "peak_source": pk.hbm_source,
                 "algorithmic_units_per_step": bytes_step, "algorithmic_units": "bytes (32 B sectors touched)"}
            model_us = bytes_step / (pk.hbm * 1e9) * 1e6
        r.update(common)
        # The per-step event pair itself costs t_event_floor (an empty kernel measures that much in this protocol; probe:
        # psg_measure_alu_peak(11)): `frac` above is on the raw event time, as the contract asks; this is the same
        # fraction with the protocol's floor taken off the launch duration
        t_net = ms_total / n * 1e3 - pk.t_event_floor_us
        r["event_pair_floor_us"] = pk.t_event_floor_us
        if t_net > 0:
            r["frac_net_of_event_floor"] = r["frac"] * (ms_total / n * 1e3) / t_net
        if cfg in (0, 2):
            # a step that moves a few KB..MB is bounded by the launch floor, not by a pipe: report
            # t_step against max(work / peak, t_floor), t_floor = an empty kernel node of a replayed graph, measured here
            t_med = float(np.median(t)) * 1e3
            r["launch_floor"] = {"t_floor_us": pk.t_floor_us, "t_event_floor_us": pk.t_event_floor_us, "t_model_us": model_us,
                                 "t_step_us_median": t_med, "t_step_us_graph_replay": b2b_ms_per_step * 1e3,
                                 "frac_of_floor": max(model_us, pk.t_event_floor_us) / t_med,
                                 "note": "60 % of a pipe or of HBM is not meaningful here; the step is latency-bound: "
                                         "frac_of_floor = max(work / peak, event-pair floor) / median event time"}
        return r

    def run(self, K, Wm, pk, headline, cpu_budget):
        w = self.w
        clk = ClockSampler(self.local) if (headline and self.rank == 0 and not self.args.no_clock_sampler) else None
        tr = self.timed(K, Wm)
        b2b_ms = self.back_to_back(K)
        clocks = clk.stop() if clk else None
        e2e = self.e2e(K)
        t = tr["per_step_ms"]
        ms_total, n = float(t.sum()), len(t)
        out = {"config": self.cfg, "workload": workload_config(self.cfg, w, self.world)["workload"],
               "steps": n, "rounds": tr["rounds"], "ms_per_step_mean": ms_total / n, "ms_per_step_median": float(np.median(t)),
               "per_step_us": {"min": float(t.min() * 1e3), "median": float(np.median(t) * 1e3),
                               "p99": float(np.percentile(t, 99) * 1e3), "max": float(t.max() * 1e3)},
               "value": whole_job_value(float(w.R) * n, self.world, ms_total), "unit": UNIT,
               "roofline": self.roofline(tr, pk, b2b_ms / K), "e2e": e2e, "gpu_launches": int(tr["launches"]),
               "back_to_back": {"value": whole_job_value(float(w.R) * K, self.world, b2b_ms), "unit": UNIT,
                                "ms_per_step": b2b_ms / K, "note": "K steps, no L2 flush, two events around the whole loop"},
               "wall_s_timed_region": tr["wall_s"], "clocks": clocks}
        if w.method == "metad" and w.params["stride"]:
            out["deposits_in_timed_region"] = n // w.params["stride"]
        if self.rank == 0 and self.world == 1:
            if w.method == "metad":
                out["hills_f64"] = self.hills_f64(pk)
                if w.params["stride"]:
                    out["deposit_event"] = self.deposit_event()
                if self.cfg in (1, 4):
                    out["grid_metad"] = self.grid_metad(pk)
            if w.method == "abf":
                out["abf_estimate"] = self.abf_estimate()
            if not self.args.skip_per_call:
                out["per_call"] = self.per_call(pk)
        if self.rank == 0 and not self.args.skip_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(w, budget_s=cpu_budget)
        return out


def interface_cv_line(psg, torch, dev, local, pk):
    """DistanceToInterface, the paper's worked CV (Eq. 4-8, App. A), 64 replicas x 50,000 interface
    atoms x 100 bins: evaluation and force application, each bins x atoms binary64 exponentials per replica"""
    R, N, bins = 64, 50000, 100
    rng = np.random.default_rng([W.SEED, 99])
    pos = torch.from_numpy((rng.random((R, N, 4), dtype=np.float32) * np.float32(10.0))).to(dev)
    force = torch.zeros((R, N, 4), device=dev)
    ctx = psg.Context(local)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.interface_cv_set(np.arange(8, dtype=np.int32), None, 8, N - 8, 2, 0.3, (1.0, 9.0), bins, 5.0)
    xi = torch.empty(R, device=dev)
    dV = torch.ones(R, device=dev)
    out = {}
    for name, fn in (("eval", lambda: ctx.interface_cv_eval(pos, xi)), ("apply", lambda: ctx.interface_cv_apply(pos, dV, force))):
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e3)
        us = float(np.median(ts))
        exps = float(R) * (N - 8) * bins / (us * 1e-6)
        out[name] = {"us": us, "f64_exps_per_s": exps, "frac_of_f64_exp_peak": exps / pk.f64_exp}
    ctx.close()
    out["shape"] = {"replicas": R, "interface_atoms": N - 8, "bins": bins}
    out["f64_exp_peak_per_s"] = pk.f64_exp
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
    pk = Peaks(psg, local)

    run = ConfigRun(args.config, args, rank, world, local, psg, torch, dist)
    head = run.run(K, Wm, pk, True, args.cpu_budget)
    cfg_obj = workload_config(args.config, run.w, world)
    run.close()

    per_config = None
    if world == 1 and not args.no_per_config:
        per_config = []
        for cfg in range(5):
            if cfg == args.config:
                per_config.append(head)
                continue
            r = ConfigRun(cfg, args, rank, world, local, psg, torch, dist)
            per_config.append(r.run(K, Wm, pk, False, args.per_config_cpu_budget))
            r.close()

    dti = None
    if world == 1 and not args.no_per_config:
        dti = interface_cv_line(psg, torch, dev, local, pk)

    out = None
    if rank == 0:
        out = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
               "ms_per_step": head["ms_per_step_mean"], "ms_per_step_median": head["ms_per_step_median"],
               "timed_steps": head["steps"], "rounds": head["rounds"],
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
               "config": cfg_obj, "e2e": head["e2e"], "gpu_launches": head["gpu_launches"], "clocks": head["clocks"],
               "roofline": head["roofline"], "back_to_back": head["back_to_back"], "per_step_us": head["per_step_us"],
               "wall_s_timed_region": head["wall_s_timed_region"],
               "timing": f"rounds of --steps={K} steps, one CUDA-event pair per step (= per launch), repeated until >= "
                         f"{MIN_TIMED_MS:.0f} ms of event time; value = R x timed_steps / sum of the event times"}
        if "hill_evals_per_s" in head["roofline"]:
            out["hill_evals_per_s"] = head["roofline"]["hill_evals_per_s"] * world
        for k in ("hills_f64", "deposit_event", "per_call", "cpu_baseline"):
            if k in head:
                out[k] = head[k]
        if per_config is not None:
            out["per_config"] = per_config
        out["peaks_measured_in_run"] = {"ffma_Glaneops": pk.ffma / 1e9, "ffma2_Glaneops": pk.ffma2 / 1e9, "mufu_ex2_Gops": pk.mufu / 1e9,
                                        "dfma_Glaneops": pk.dfma / 1e9, "f64_exp_Gops": pk.f64_exp / 1e9, "hbm_GBs": pk.hbm,
                                        "hbm_source": pk.hbm_source, "graph_node_floor_us": pk.t_floor_us,
                                        "event_pair_floor_us": pk.t_event_floor_us}
        if dti is not None:
            out["interface_cv"] = dti
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
    w = make_workload(args.config, K, world)
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
            "data": "synthetic", "config": workload_config(args.config, w, world), "sample": sample,
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="psg", choices=["psg", "reference"])
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--per-config-cpu-budget", type=float, default=4.0)
    ap.add_argument("--ref-budget", type=float, default=60.0)
    ap.add_argument("--no-per-config", action="store_true", help="headline config only")
    ap.add_argument("--skip-cpu-baseline", action="store_true")
    ap.add_argument("--skip-per-call", action="store_true")
    ap.add_argument("--no-clock-sampler", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    args.steps = max(args.steps, 1)
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    out = run_reference(args, rank, world) if args.impl == "reference" else run_psg(args, rank, world)
    if rank == 0 and out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
