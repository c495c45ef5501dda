"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (psg_step on the whole batch).

The oracle is fast enough to check every replica of one step of configs 0, 1, 3 and 4; config 2 (4,096 replicas x
50,000 atoms, 3.3 GB per array) is checked on every replica too, but its oracle step takes a few seconds.
Hill heights come from the oracle (never from the CUDA path).  Tolerances are the ones of test_gpu_parity.py.

Metadynamics is checked in BOTH hill-sum precisions (SURVEY.md 8(c) "Tolerance reading"):
  PSG_HILLS_F64 through the fused psg_step must meet the LITERAL 1e-5 / 1e-6 rule on dV/dxi at every element, and its
    forces only carry the rounding of the binary32 read-modify-write (R-F32SUM), no conditioning term;
  PSG_HILLS_F32 (the default, benched mode) must meet the literal rule OR |err| <= 2e-7 T, and the literal fail count
    and max |err| / T of every config are written to gpurun_out/parity_fullsize.jsonl (the table of BASELINE.md 4).
"""
import json
import os
import numpy as np
import pytest

import workloads as W
from _parity import assert_close, assert_forces_close, fails, metad_force_extra, oracle_heights, oracle_step, oracle_system

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def psg():
    import paper_2301_04835_b200 as p
    p.load_library()
    return p


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _report(rec):
    """one JSON line per full-size comparison; the directory only exists under gpurun (it is git-ignored scratch)"""
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(d):
        with open(os.path.join(d, "parity_fullsize.jsonl"), "a") as f:
            f.write(json.dumps(rec) + "\n")
    print(json.dumps(rec))


def _lit(gpu, ref, period=None):
    bad = fails(gpu, ref, period)
    return {"literal_fail": int(bad.sum()), "total": int(bad.size)}


def _run_full(torch, psg, cfg, frame=1, precision=None, **kw):
    w = W.make(cfg, **kw)
    ctx = psg.Context(0)
    psg.configure_from_workload(ctx, w)
    f64 = precision is not None and precision == psg.HILLS_F64
    if precision is not None:
        ctx.set_hill_precision(precision)
    rec = {"config": cfg, "workload": w.name, "R": w.R, "method": w.method,
           "mode": ("hills_f64" if f64 else "hills_f32") if w.method == "metad" else "default"}
    sysm = oracle_system(w)
    pos, f0 = w.positions(frame), w.forces0()
    centers = heights = abf = fs = None
    if w.method == "metad":
        centers, heights = w.params["hill_centers"], oracle_heights(w)
        ctx.load_hills(dev(torch, centers), dev(torch, heights))
    if w.method == "abf":
        nb = int(np.prod(w.params["shape"]))
        abf, fs = (np.zeros(nb, np.int32), np.zeros((nb, w.n_cv), np.float64)), w.fsample(frame)
    d_f = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.step(dev(torch, pos), d_f, None if fs is None else dev(torch, fs), 1)
    ctx.sync_check()
    launches = ctx.launch_count() - n0
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    f = d_f.cpu().numpy()
    del d_f
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0, centers, heights, abf, fs)
    assert_close(out["xi"], xi_ref, f"config {cfg} xi", period=w.period)
    rec["xi"] = _lit(out["xi"], xi_ref, w.period)
    if w.method == "abf":
        assert np.array_equal(out["bin"], b["bin"]), "ABF bins must be bit-exact"
        hp, fp, nb = ctx.abf_state()
        from paper_2301_04835_b200.psg import _view
        assert np.array_equal(_view(hp, (nb,), torch.int32, 0).cpu().numpy(), abf[0]), "ABF histogram must be bit-exact"
        assert_close(_view(fp, (nb, w.n_cv), torch.float32, 0).cpu().numpy(), abf[1], "ABF force sums")
        assert_close(out["dVdxi"], b["dVdxi"], f"config {cfg} mean force")
        rec["bin_mismatch"] = 0
        rec["hist_mismatch"] = 0
        rec["dVdxi"] = _lit(out["dVdxi"], b["dVdxi"])
    elif w.method == "metad":
        assert_close(out["V"], b["V"], f"config {cfg} V")
        rec["V"] = _lit(out["V"], b["V"])
        err = np.abs(out["dVdxi"] - b["dVdxi"])
        lit = err > np.maximum(1e-5 * np.abs(b["dVdxi"]), 1e-6)
        rec["dVdxi"] = {"literal_fail": int(lit.sum()), "total": int(lit.size),
                        "max_err_over_T": float(np.max(err / np.maximum(b["T"], 1e-300))),
                        "max_abs_err": float(err.max()), "T_median": float(np.median(b["T"])), "T_max": float(b["T"].max())}
        if f64:
            assert_close(out["dVdxi"], b["dVdxi"], f"config {cfg} dV/dxi (binary64 terms, literal rule)")
        else:
            assert np.all(err <= np.maximum(np.maximum(1e-5 * np.abs(b["dVdxi"]), 1e-6), 2e-7 * b["T"])), "hill-sum gradient"
            assert lit.mean() <= 0.05, f"literal fail fraction {lit.mean():.4f}"
    else:
        assert_close(out["V"], b["V"], f"config {cfg} V")
        assert_close(out["dVdxi"], b["dVdxi"], f"config {cfg} dV/dxi")
        rec["V"] = _lit(out["V"], b["V"])
        rec["dVdxi"] = _lit(out["dVdxi"], b["dVdxi"])
    assert np.array_equal(f[..., 3].view(np.uint32), f0[..., 3].view(np.uint32)), "force w must keep its bits"
    # forces: binary64 hill terms leave only the rounding of the binary32 += (R-F32SUM); binary32 terms add the
    # conditioning bound of their gradient
    extra = metad_force_extra(w, sysm, pos, b["T"]) if (w.method == "metad" and not f64) else None
    lit = assert_forces_close(f[..., :3], f_ref, f0[..., :3], f"config {cfg} forces", extra)
    assert lit.mean() <= 0.02
    # the literal rule on the BIAS force alone (f - f0 against the oracle's, both differences of the same f0): what the
    # path adds, without the engine force's own binary32 rounding
    touched = np.abs(f_ref - f0[..., :3].astype(np.float64)) > 0
    rec["force"] = {"literal_fail": int(lit.sum()), "total": int(lit.size), "cv_atom_elements": int(touched.sum()),
                    "literal_fail_on_cv_atoms": int((lit & touched).sum())}
    rec["launches_per_step"] = int(launches)
    _report(rec)
    ctx.close()
    return launches


def test_full_config0(torch, psg):
    assert _run_full(torch, psg, 0, steps=4) == 1


def test_full_config1_512_walkers_50000_hills(torch, psg):
    assert _run_full(torch, psg, 1, steps=4) == 1


def test_full_config3_256_windows_100000_atoms(torch, psg):
    assert _run_full(torch, psg, 3, steps=2) == 1


def test_full_config4_1024_walkers_200000_hills_shared_million_atom_array(torch, psg):
    assert _run_full(torch, psg, 4, steps=2) == 1


@pytest.mark.parametrize("cfg,kw", [(0, {"steps": 4}), (1, {"steps": 4}), (4, {"steps": 2})])
def test_full_metad_f64_terms_fused_step_literal(torch, psg, cfg, kw):
    """PSG_HILLS_F64 through the fused psg_step at BASELINE.json's full sizes: the literal 1e-5 / 1e-6 rule everywhere"""
    assert _run_full(torch, psg, cfg, precision=psg.HILLS_F64, **kw) == 1


def test_full_config2_4096_replicas_50000_atoms(torch, psg):
    assert _run_full(torch, psg, 2, steps=2) == 1
