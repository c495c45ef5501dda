"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (psg_step on the whole batch).

The oracle is fast enough to check every replica of one step of configs 0, 1, 3 and 4; config 2 (4,096 replicas x
50,000 atoms, 3.3 GB per array) is checked on every replica too, but its oracle step takes a few seconds.
Hill heights come from the oracle (never from the CUDA path).  Tolerances are the ones of test_gpu_parity.py.
"""
import numpy as np
import pytest

import workloads as W
from _parity import assert_close, assert_forces_close, metad_force_extra, oracle_heights, oracle_step, oracle_system

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


def _run_full(torch, psg, cfg, frame=1, **kw):
    w = W.make(cfg, **kw)
    ctx = psg.Context(0)
    psg.configure_from_workload(ctx, w)
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
    if w.method == "abf":
        assert np.array_equal(out["bin"], b["bin"]), "ABF bins must be bit-exact"
        hp, fp, nb = ctx.abf_state()
        from paper_2301_04835_b200.psg import _view
        assert np.array_equal(_view(hp, (nb,), torch.int32, 0).cpu().numpy(), abf[0]), "ABF histogram must be bit-exact"
        assert_close(_view(fp, (nb, w.n_cv), torch.float32, 0).cpu().numpy(), abf[1], "ABF force sums")
        assert_close(out["dVdxi"], b["dVdxi"], f"config {cfg} mean force")
    elif w.method == "metad":
        assert_close(out["V"], b["V"], f"config {cfg} V")
        err = np.abs(out["dVdxi"] - b["dVdxi"])
        lit = err > np.maximum(1e-5 * np.abs(b["dVdxi"]), 1e-6)
        assert np.all(err <= np.maximum(np.maximum(1e-5 * np.abs(b["dVdxi"]), 1e-6), 2e-7 * b["T"])), "hill-sum gradient"
        assert lit.mean() <= 0.05, f"literal fail fraction {lit.mean():.4f}"
        print(f"config {cfg}: hill-sum gradient literal 1e-5/1e-6 fail fraction {lit.mean():.4f} "
              f"(max |err|/T = {np.max(err / np.maximum(b['T'], 1e-300)):.2e})")
    else:
        assert_close(out["V"], b["V"], f"config {cfg} V")
        assert_close(out["dVdxi"], b["dVdxi"], f"config {cfg} dV/dxi")
    assert np.array_equal(f[..., 3].view(np.uint32), f0[..., 3].view(np.uint32)), "force w must keep its bits"
    extra = metad_force_extra(w, sysm, pos, b["T"]) if w.method == "metad" else None
    lit = assert_forces_close(f[..., :3], f_ref, f0[..., :3], f"config {cfg} forces", extra)
    assert lit.mean() <= 0.02
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


def test_full_config2_4096_replicas_50000_atoms(torch, psg):
    assert _run_full(torch, psg, 2, steps=2) == 1
