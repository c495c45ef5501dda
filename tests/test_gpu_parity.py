"""Parity of the CUDA path (through the C ABI) with the fp64 oracle, element by element, on the same
seeded inputs.  Sizes here are reduced so the oracle finishes in seconds but still span several
tiles and a ragged tail; tests/test_gpu_fullsize.py covers BASELINE.json's full sizes.

Bar (BASELINE.json north_star): bit-exact ABF bins and histogram counts; |gpu - ref| <= max(1e-5 |ref|, 1e-6)
on binary32 CVs, bias energies and forces.  The binary32 hill-sum gradient is additionally allowed the
conditioning bound of DESIGN.md ("Hill sum precision"): its literal fail fraction is asserted small and
printed, and the binary64 mode must pass literally.
"""
import math

import numpy as np
import pytest

import oracle as orc
import workloads as W
from _parity import (assert_close, assert_forces_close, fails, metad_force_extra, oracle_bias, oracle_heights, oracle_step,
                     oracle_system, slot_rows, wrap)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def psg():
    import paper_2301_04835_b200 as p
    p.load_library()      # fails loudly if libpsg.so is missing: no fallback
    return p


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_ctx(psg, w, **kw):
    ctx = psg.Context(0)
    psg.configure_from_workload(ctx, w, **kw)
    return ctx


SMALL = {
    0: dict(n_hills=300, steps=10),
    1: dict(R=70, n_hills=2130, steps=10, stride=5),
    2: dict(R=300, N=700, steps=4),
    3: dict(R=3, N=5003, steps=2),
    4: dict(N=6000, R=130, n_hills=2650, steps=3),
}


def small(cfg, **over):
    kw = dict(SMALL[cfg])
    kw.update(over)
    return W.make(cfg, **kw)


# ------------------------------------------------------------------------------------ CVs
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("frame", [0, 1])
def test_cv_eval_matches_oracle(torch, psg, cfg, frame):
    w = small(cfg)
    ctx = make_ctx(psg, w, with_method=False)
    sysm = oracle_system(w)
    pos = w.positions(frame)
    xi_ref, jac_ref = sysm.cv_eval(pos)
    n_slots = ctx.n_slots
    d_xi = torch.full((w.R, w.n_cv), float("nan"), device="cuda")
    d_jac = torch.full((w.R, max(n_slots, 1), 3), float("nan"), device="cuda")
    ctx.cv_eval(dev(torch, pos), d_xi, d_jac if n_slots else None)
    ctx.sync_check()
    assert_close(d_xi.cpu().numpy(), xi_ref, f"xi config {cfg}", period=w.period)
    if n_slots:
        rows = slot_rows(w)
        assert_close(d_jac.cpu().numpy(), jac_ref[:, rows, :], f"jacobian config {cfg}")


def test_cv_zoo_weights_stride3_angle_component(torch, psg):
    """every CV type, weighted explicit groups of several atoms, stride-3 positions, per-replica indices"""
    rng = np.random.default_rng(7)
    R, N = 37, 50
    pos = rng.normal(scale=0.8, size=(R, N, 3)).astype(np.float32)
    slot = np.stack([rng.permutation(N)[:17] for _ in range(R)]).astype(np.int32)
    sw = rng.uniform(1, 16, size=17).astype(np.float32)
    groups = lambda b, sizes: [("slots", b + sum(sizes[:i]), sizes[i]) for i in range(len(sizes))]
    cvs_n = [("angle", groups(0, [2, 1, 3]), 0.0, 0), ("component", groups(6, [4]), 0.0, 1),
             ("distance", groups(10, [1, 2]), 0.0, 0), ("rgyr", groups(13, [4]), 0.0, 0)]
    o_cvs = [{"type": {"angle": orc.ANGLE, "component": orc.COMPONENT, "distance": orc.DISTANCE, "rgyr": orc.RGYR}[k],
              "groups": g, "axis": ax, "period": p} for k, g, p, ax in cvs_n]
    g_cvs = [{"type": {"angle": psg.CV_ANGLE, "component": psg.CV_COM_COMPONENT, "distance": psg.CV_DISTANCE,
                       "rgyr": psg.CV_RGYR}[k], "groups": g, "axis": ax, "period": p} for k, g, p, ax in cvs_n]
    sysm = orc.System(R, N, N, 3, o_cvs, slot, sw, None)
    xi_ref, jac_ref = sysm.cv_eval(pos)
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 3, 3)
    ctx.set_cvs(g_cvs, slot, sw, None)
    d_xi = torch.empty((R, 4), device="cuda")
    d_jac = torch.empty((R, 17, 3), device="cuda")
    d_pos = dev(torch, pos)
    ctx.cv_eval(d_pos, d_xi, d_jac)
    ctx.sync_check()
    assert_close(d_xi.cpu().numpy(), xi_ref, "zoo xi")
    assert_close(d_jac.cpu().numpy(), jac_ref, "zoo jacobian")   # slots listed in oracle row order
    # forces with stride 3, harmonic bias on all four CVs
    ks = np.array([50, 200, 1000, 300], np.float32)
    cen = rng.uniform(0.2, 1.5, size=(R, 4)).astype(np.float32)
    ctx.set_harmonic(ks, cen)
    f0 = (rng.standard_normal((R, N, 3)) * 100).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.step(d_pos, d_f, None, 1)
    ctx.sync_check()
    V, dV = orc.harmonic(xi_ref.astype(np.float32).astype(np.float64), ks, cen, np.zeros(4))
    f_ref = sysm.apply_forces(pos, dV, f0.astype(np.float64))
    assert_forces_close(d_f.cpu().numpy(), f_ref, f0, "zoo forces")
    out = ctx.read_step_outputs()
    assert_close(out["V"].cpu().numpy(), V, "zoo V")


def test_degenerate_geometry_gives_zero_jacobian(torch, psg):
    # replica 0: coincident distance points; replica 1: collinear dihedral; replica 2: regular
    pos = np.zeros((3, 6, 4), np.float32)
    pos[0, :, 0] = [0, 1, 2, 3, 1, 1]        # collinear chain, distance atoms 4,5 coincide
    pos[1] = pos[0]
    pos[2, :, :3] = [[1, 0, 0], [0, 0, 0], [0, 0, 1], [0.5, 0.5, 1], [0, 0, 0], [3, 4, 0]]
    cvs = [{"type": psg.CV_DIHEDRAL, "groups": [("slots", i, 1) for i in range(4)], "period": 2 * math.pi},
           {"type": psg.CV_DISTANCE, "groups": [("slots", 4, 1), ("slots", 5, 1)]}]
    ctx = psg.Context(0)
    ctx.set_layout(3, 6, 6, 4, 4)
    ctx.set_cvs(cvs, np.arange(6, dtype=np.int32))
    d_xi = torch.empty((3, 2), device="cuda")
    d_jac = torch.empty((3, 6, 3), device="cuda")
    ctx.cv_eval(dev(torch, pos), d_xi, d_jac)
    ctx.sync_check()
    j, xi = d_jac.cpu().numpy(), d_xi.cpu().numpy()
    assert np.all(j[0] == 0) and np.all(j[1] == 0) and np.all(np.isfinite(xi))
    assert xi[0, 1] == 0 and abs(xi[2, 1] - 5.0) < 1e-6 and abs(xi[2, 0] - math.pi / 4) < 1e-6
    assert np.allclose(j[2, 5], [0.6, 0.8, 0.0], atol=1e-7)


# ------------------------------------------------------------------------------------ harmonic
def test_harmonic_periodic_matches_oracle(torch, psg):
    w = small(1)
    ctx = make_ctx(psg, w, with_method=False)
    rng = np.random.default_rng(3)
    ks = np.array([100.0, 37.5], np.float32)
    cen = rng.uniform(-math.pi, math.pi, size=(w.R, 2)).astype(np.float32)
    xi = rng.uniform(-math.pi, math.pi, size=(w.R, 2)).astype(np.float32)
    xi[0], cen[0] = (3.0, -3.0), (-3.0, 3.0)
    ctx.set_harmonic(ks, cen)
    d_V, d_dV = torch.empty(w.R, device="cuda"), torch.empty((w.R, 2), device="cuda")
    ctx.bias_eval(dev(torch, xi), d_V, d_dV)
    ctx.sync_check()
    V, dV = orc.harmonic(xi.astype(np.float64), ks, cen, w.period)
    assert_close(d_V.cpu().numpy(), V, "harmonic V")
    assert_close(d_dV.cpu().numpy(), dV, "harmonic dV")
    assert abs(float(d_dV[0, 0]) - 100.0 * (6 - 2 * math.pi)) < 1e-4


# ------------------------------------------------------------------------------------ hill sum
def _hill_case(torch, psg, n_cv, periodic, R, n_h, seed, precision):
    rng = np.random.default_rng([11, seed])
    per = np.array([2 * math.pi if (periodic >> k) & 1 else 0.0 for k in range(n_cv)])
    sigma = np.array([0.35, 0.2, 0.05, 0.5][:n_cv], np.float32)
    lo = np.where(per > 0, -math.pi, 0.3)
    hi = np.where(per > 0, math.pi, 1.5)
    centers = rng.uniform(lo, hi, size=(n_h, n_cv)).astype(np.float32)
    heights = rng.uniform(0.05, 1.2, size=n_h).astype(np.float32)
    xi = rng.uniform(lo, hi, size=(R, n_cv)).astype(np.float32)
    cvs = [{"type": psg.CV_DISTANCE, "groups": [("slots", 2 * k, 1), ("slots", 2 * k + 1, 1)], "period": per[k]}
           for k in range(n_cv)]
    ctx = psg.Context(0)
    ctx.set_layout(R, 2 * n_cv, 2 * n_cv, 4, 4)
    ctx.set_cvs(cvs, np.arange(2 * n_cv, dtype=np.int32))
    ctx.set_metad(sigma, 1.2, 0.0, max(n_h, 1), 0)
    ctx.set_hill_precision(precision)
    if n_h:
        ctx.load_hills(dev(torch, centers), dev(torch, heights))
    d_V = torch.full((R,), float("nan"), device="cuda")
    d_dV = torch.full((R, n_cv), float("nan"), device="cuda")
    ctx.bias_eval(dev(torch, xi), d_V, d_dV)
    ctx.sync_check()
    V, dV, T = orc.metad(xi.astype(np.float64), centers, heights, sigma, per)
    return d_V.cpu().numpy(), d_dV.cpu().numpy(), V, dV, T


@pytest.mark.parametrize("n_cv,periodic", [(1, 0), (1, 1), (2, 3), (2, 1), (3, 3), (3, 0), (4, 5), (4, 0)])
@pytest.mark.parametrize("R,n_h", [(1, 1), (70, 2100), (5, 33), (129, 7000)])
def test_hill_sum_f64_mode_literal(torch, psg, n_cv, periodic, R, n_h):
    gV, gdV, V, dV, T = _hill_case(torch, psg, n_cv, periodic, R, n_h, 1, psg.HILLS_F64)
    assert_close(gV, V, "V (f64 terms)")
    assert_close(gdV, dV, "dV/dxi (f64 terms)")


@pytest.mark.parametrize("n_cv,periodic", [(1, 0), (1, 1), (2, 3), (2, 1), (3, 3), (3, 0), (4, 5), (4, 0)])
@pytest.mark.parametrize("R,n_h", [(1, 1), (70, 2100), (5, 33), (129, 7000)])
def test_hill_sum_f32_mode(torch, psg, n_cv, periodic, R, n_h):
    gV, gdV, V, dV, T = _hill_case(torch, psg, n_cv, periodic, R, n_h, 2, psg.HILLS_F32)
    assert_close(gV, V, "V (f32 terms)")
    bad = fails(gdV, dV)
    # binary32 terms are backward stable: |err| <= 2e-7 * sum_h |term|
    assert np.all(np.abs(gdV - dV) <= np.maximum(np.maximum(1e-5 * np.abs(dV), 1e-6), 2e-7 * T))
    assert bad.mean() <= 0.05, f"literal fail fraction {bad.mean():.4f}"


@pytest.mark.parametrize("n_cv,periodic,R,n_h", [(3, 3, 320, 250000), (4, 5, 130, 410000), (3, 0, 1024, 150000)])
def test_hill_sum_uneven_chunking_on_the_spare_ctas(torch, psg, n_cv, periodic, R, n_h):
    """Long hill lists on a tile count that does not divide the 148 CTAs (5, 3, 16 tiles): the 3- and 4-CV kernels shorten the
    long chunks and let the spare CTAs run one short last chunk per tile (hills_spare_chunking): every hill exactly once."""
    gV, gdV, V, dV, T = _hill_case(torch, psg, n_cv, periodic, R, n_h, 5, psg.HILLS_F32)
    assert_close(gV, V, "V (f32 terms, uneven chunks)")
    assert np.all(np.abs(gdV - dV) <= np.maximum(np.maximum(1e-5 * np.abs(dV), 1e-6), 2e-7 * T))
    # a unit-height list with far-away walkers: V counts the hills that were summed (none twice, none dropped)
    rng = np.random.default_rng(7)
    ctx = psg.Context(0)
    ctx.set_layout(R, 2 * n_cv, 2 * n_cv, 4, 4)
    ctx.set_cvs([{"type": psg.CV_DISTANCE, "groups": [("slots", 2 * k, 1), ("slots", 2 * k + 1, 1)], "period": 0.0}
                 for k in range(n_cv)], np.arange(2 * n_cv, dtype=np.int32))
    ctx.set_metad(np.full(n_cv, 1.0e4, np.float32), 1.0, 0.0, n_h, 0)      # sigma so wide that every Gaussian is 1 to 1e-9
    ctx.load_hills(dev(torch, rng.uniform(0.9, 1.1, size=(n_h, n_cv)).astype(np.float32)), dev(torch, np.ones(n_h, np.float32)))
    d_V = torch.empty(R, device="cuda")
    d_dV = torch.empty((R, n_cv), device="cuda")
    ctx.bias_eval(dev(torch, np.ones((R, n_cv), np.float32)), d_V, d_dV)
    ctx.sync_check()
    assert np.all(np.abs(d_V.cpu().numpy().astype(np.float64) - n_h) <= 1e-5 * n_h), (d_V.min().item(), d_V.max().item(), n_h)
    ctx.close()


def test_hill_sum_empty_store_is_zero(torch, psg):
    gV, gdV, V, dV, T = _hill_case(torch, psg, 2, 3, 9, 0, 3, psg.HILLS_F32)
    assert np.all(gV == 0) and np.all(gdV == 0)


def test_hill_sum_periodic_image(torch, psg):
    """xi = 3.0, s = -3.0: nearest image delta = 6 - 2 pi (closed form, not via the oracle)"""
    ctx = psg.Context(0)
    ctx.set_layout(1, 2, 2, 4, 4)
    ctx.set_cvs([{"type": psg.CV_DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)], "period": 2 * math.pi}],
                np.arange(2, dtype=np.int32))
    ctx.set_metad(np.array([0.35], np.float32), 1.2, 0.0, 4, 0)
    ctx.load_hills(dev(torch, np.array([[-3.0]], np.float32)), dev(torch, np.array([1.2], np.float32)))
    d_V, d_dV = torch.empty(1, device="cuda"), torch.empty((1, 1), device="cuda")
    ctx.bias_eval(dev(torch, np.array([[3.0]], np.float32)), d_V, d_dV)
    ctx.sync_check()
    assert abs(float(d_V[0]) - 0.8650218101534733) < 1e-5 * 0.87
    assert abs(float(d_dV[0, 0]) - 1.9996854451049233) < 2e-5


# ------------------------------------------------------------------------------------ deposition
@pytest.mark.parametrize("cfg", [0, 1, 4])
def test_well_tempered_hill_store_matches_oracle(torch, psg, cfg):
    """build the whole pre-filled hill list by psg_deposit_hill in the workload's rounds (ragged last round
    through the mask) and compare centres (bit-exact) and heights with the oracle's list"""
    w = small(cfg)                       # capacity = exactly the number of hills: a masked (ragged) round needs no padding
    ctx = make_ctx(psg, w)
    c = w.params["hill_centers"]
    for b, e in w.hill_rounds():
        xi = np.zeros((w.R, w.n_cv), np.float32)
        xi[: e - b] = c[b:e]
        mask = None
        if e - b < w.R:
            mask = np.zeros(w.R, np.uint8)
            mask[: e - b] = 1
        ctx.deposit_hill(dev(torch, xi), None if mask is None else dev(torch, mask))
    gc, gh = ctx.get_hills()
    ref_h = oracle_heights(w)
    assert gc.shape[0] == w.params["n_hills"]
    assert np.array_equal(gc.cpu().numpy(), c)
    assert_close(gh.cpu().numpy(), ref_h, f"well-tempered heights config {cfg}")
    assert ref_h[0] == np.float32(1.2) and ref_h.min() < 1.0


def test_deposit_standard_heights_and_capacity(torch, psg):
    w = small(1)
    ctx = make_ctx(psg, w, with_method=False)
    ctx.set_metad(w.params["sigma"], 1.2, 0.0, 2 * w.R + 3, 0)
    xi = W.random_xi(w, 1)
    ctx.deposit_hill(dev(torch, xi))
    ctx.deposit_hill(dev(torch, xi))
    with pytest.raises(psg.PsgError) as ei:
        ctx.deposit_hill(dev(torch, xi))
    assert ei.value.code == -4                      # PSG_ECAPACITY, nothing launched
    gc, gh = ctx.get_hills()
    assert gc.shape[0] == 2 * w.R and np.all(gh.cpu().numpy() == np.float32(1.2))
    assert np.array_equal(gc.cpu().numpy()[w.R:], xi)


# ------------------------------------------------------------------------------------ ABF
def _abf_run(torch, psg, w, xi_list, fs_list, prefill=False, ctx=None):
    p = w.params
    nb = int(np.prod(p["shape"]))
    hist = np.zeros(nb, np.int32)
    fsum = np.zeros((nb, w.n_cv), np.float64)
    if prefill:
        rng = np.random.default_rng(5)
        hist[:] = rng.integers(0, 1000, size=nb)
        fsum[:] = hist[:, None] * rng.normal(loc=(25, -15)[: w.n_cv], scale=1.0, size=(nb, w.n_cv))
        fsum = fsum.astype(np.float32).astype(np.float64)
    d_hist, d_fsum = dev(torch, hist), dev(torch, fsum.astype(np.float32))
    ctx = ctx or make_ctx(psg, w, with_method=False)
    ctx.set_abf(p["lower"], p["upper"], p["shape"], p["periodic"], p["n_threshold"], d_hist, d_fsum)
    for xi, fs in zip(xi_list, fs_list):
        d_bin = torch.full((w.R,), -7, dtype=torch.int32, device="cuda")
        d_dV = torch.full((w.R, w.n_cv), float("nan"), device="cuda")
        ctx.abf_update(dev(torch, xi), dev(torch, fs), d_bin, d_dV)
        ctx.sync_check()
        b_ref, dV_ref = orc.abf_update(xi, fs, p["lower"], p["upper"], p["shape"], p["periodic"], p["n_threshold"],
                                       hist, fsum)
        assert np.array_equal(d_bin.cpu().numpy(), b_ref), "ABF bin indices must be bit-exact"
        assert np.array_equal(d_hist.cpu().numpy(), hist), "ABF histogram must be bit-exact"
        assert_close(d_fsum.cpu().numpy(), fsum, "ABF Fsum")
        assert_close(d_dV.cpu().numpy(), dV_ref, "ABF mean force")
    return hist


@pytest.mark.parametrize("prefill", [False, True])
def test_abf_update_matches_oracle(torch, psg, prefill):
    w = small(2, R=4096 + 37)
    rng = np.random.default_rng(9)
    xis, fss = [], []
    for s in range(4):
        xi = rng.uniform(0.1, 2.1, size=(w.R, 2)).astype(np.float32)
        xi[:70] = rng.uniform(0.95, 1.0, size=(70, 2))            # pile-up: many replicas in few bins
        xis.append(xi)
        fss.append(w.fsample(s))
    hist = _abf_run(torch, psg, w, xis, fss, prefill)
    assert hist.max() > 20


def test_abf_bin_edges_exact(torch, psg):
    """every bin edge of config 2's grid as computed in binary32 and binary64, +-1 ulp, NaN, out of range"""
    w = small(2, R=65 * 6 + 8)
    e32 = (np.float32(0.2) + np.arange(65, dtype=np.float32) * np.float32(1.8 / 64)).astype(np.float32)
    e64 = (0.2 + np.arange(65) * (1.8 / 64)).astype(np.float32)
    vals = np.concatenate([e32, np.nextafter(e32, np.float32(9)), np.nextafter(e32, np.float32(-9)), e64,
                           np.nextafter(e64, np.float32(9)), np.nextafter(e64, np.float32(-9)),
                           np.array([np.nan, -1.0, 0.0, 2.0, 1.99, 0.228125, 1e30, -1e30], np.float32)])[: w.R]
    assert vals.shape[0] == w.R
    xi = np.stack([vals, np.full(w.R, 1.0, np.float32)], axis=1).astype(np.float32)
    _abf_run(torch, psg, w, [xi, xi[:, ::-1].copy()], [w.fsample(0), w.fsample(1)])


def test_abf_periodic_grid(torch, psg):
    w = small(1, R=333)
    w.method = "abf"
    w.params.update(lower=np.array([-math.pi, -math.pi], np.float32), upper=np.array([math.pi, math.pi], np.float32),
                    shape=np.array([24, 17], np.int32), periodic=np.array([1, 1], np.int32), n_threshold=3,
                    fsample_mean=(25.0, -15.0), fsample_std=5.0)
    rng = np.random.default_rng(4)
    xi = rng.uniform(-3 * math.pi, 3 * math.pi, size=(w.R, 2)).astype(np.float32)
    _abf_run(torch, psg, w, [xi, xi], [w.fsample(0), w.fsample(1)])


# ------------------------------------------------------------------------------------ forces, unfused calls
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_five_calls_chain_matches_oracle(torch, psg, cfg):
    """cv_eval -> bias_eval / abf_update -> apply_bias_forces as separate C calls"""
    w = small(cfg)
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    pos, f0 = w.positions(0), w.forces0()
    centers = heights = abf_state = fs = None
    if w.method == "metad":
        centers, heights = w.params["hill_centers"], oracle_heights(w)
        ctx.load_hills(dev(torch, centers), dev(torch, heights))
    if w.method == "abf":
        nb = int(np.prod(w.params["shape"]))
        abf_state = (np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64))
        fs = w.fsample(0)
    d_pos, d_f = dev(torch, pos), dev(torch, f0)
    d_xi = torch.empty((w.R, w.n_cv), device="cuda")
    d_V, d_dV = torch.zeros(w.R, device="cuda"), torch.empty((w.R, w.n_cv), device="cuda")
    ctx.cv_eval(d_pos, d_xi, None)
    if w.method == "abf":
        ctx.abf_update(d_xi, dev(torch, fs), None, d_dV)
    else:
        ctx.bias_eval(d_xi, d_V, d_dV)
    ctx.apply_bias_forces(d_pos, d_dV, d_f)
    ctx.sync_check()
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0, centers, heights, abf_state, fs)
    _check_step(w, sysm, pos, d_xi.cpu().numpy(), d_V.cpu().numpy(), d_dV.cpu().numpy(), d_f.cpu().numpy(), f0, xi_ref, b, f_ref)


def _check_step(w, sysm, pos, xi, V, dV, f, f0, xi_ref, b, f_ref, what=""):
    assert_close(xi, xi_ref, what + "xi", period=w.period)
    if w.method != "abf":
        assert_close(V, b["V"], what + "V")
    if w.method == "metad":
        err = np.abs(dV - b["dVdxi"])
        assert np.all(err <= np.maximum(np.maximum(1e-5 * np.abs(b["dVdxi"]), 1e-6), 2e-7 * b["T"])), what + "dV/dxi"
    else:
        assert_close(dV, b["dVdxi"], what + "dV/dxi")
    # forces: the API's tolerance on the force array; w and untouched atoms keep their bits
    assert np.array_equal(f[..., 3].view(np.uint32), f0[..., 3].view(np.uint32)), "force w must keep its bits"
    touched = np.zeros(f0.shape[:2], bool)
    for cv in w.cvs:
        for g in cv["groups"]:
            if g[0] == "range":
                touched[:, g[1]: g[1] + g[2]] = True
    if w.slot_atom is not None:
        if w.slot_atom.ndim == 1:
            touched[:, w.slot_atom] = True
        else:
            touched[0, w.slot_atom.reshape(-1)] = True
    assert np.array_equal(f[~touched].view(np.uint32), f0[~touched].view(np.uint32)), "non-CV atoms must be untouched"
    # forces inherit the hill-sum gradient's conditioning bound
    extra = metad_force_extra(w, sysm, pos, b["T"]) if w.method == "metad" else None
    lit = assert_forces_close(f[..., :3], f_ref, f0[..., :3], what + "forces", extra)
    assert lit.mean() <= 0.02, f"{what}forces: literal fail fraction {lit.mean():.4f}"


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_fused_step_matches_oracle_over_steps(torch, psg, cfg):
    """psg_step over several steps (frames cycle, forces accumulate, config 1 deposits every 5 steps,
    the ABF grid fills)"""
    w = small(cfg)
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    f0 = w.forces0()
    centers = heights = abf_state = None
    n_h = 0
    if w.method == "metad":
        cap = w.params["capacity"]
        centers = np.zeros((cap, w.n_cv), np.float32)
        heights = np.zeros(cap, np.float32)
        n_h = w.params["n_hills"]
        centers[:n_h], heights[:n_h] = w.params["hill_centers"], oracle_heights(w)
        ctx.load_hills(dev(torch, centers[:n_h]), dev(torch, heights[:n_h]))
    if w.method == "abf":
        nb = int(np.prod(w.params["shape"]))
        abf_state = (np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64))
    d_f = dev(torch, f0)
    f_ref32 = f0.copy()
    frames = [dev(torch, w.positions(k)) for k in range(w.K)]
    for step in range(1, w.steps + 1):
        pos = w.positions(step % w.K)
        fs = w.fsample(step % w.K) if w.method == "abf" else None
        f_before = d_f.cpu().numpy()
        ctx.step(frames[step % w.K], d_f, None if fs is None else dev(torch, fs), step)
        ctx.sync_check()
        out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
        # oracle: xi -> (deposit if due, heights from the OLD list) -> bias with the NEW list -> forces
        xi_ref = sysm.cv_eval(pos, want_jac=False)
        stride = w.params.get("stride", 0) if w.method == "metad" else 0
        if stride and step % stride == 0:
            n_h = orc.deposit_hills(xi_ref.astype(np.float32), None, w.params["w0"], w.params["kB_deltaT"],
                                    w.params["sigma"], w.period, n_h, centers, heights)
        c_now = None if centers is None else centers[:n_h]
        h_now = None if heights is None else heights[:n_h]
        b = oracle_bias(w, xi_ref.astype(np.float32), c_now, h_now, abf_state, fs)
        f_ref = sysm.apply_forces(pos, b["dVdxi"], f_before[..., :3].astype(np.float64))
        _check_step(w, sysm, pos, out["xi"], out["V"], out["dVdxi"], d_f.cpu().numpy(), f_before, xi_ref, b, f_ref,
                    what=f"config {cfg} step {step}: ")
        if w.method == "abf":
            assert np.array_equal(out["bin"], b["bin"])
    if w.method == "metad" and w.params["stride"]:
        gc, gh = ctx.get_hills()
        assert gc.shape[0] == n_h == w.params["capacity"]
        assert_close(gh.cpu().numpy(), heights[:n_h], "hill heights after deposits")
        assert_close(gc.cpu().numpy(), centers[:n_h], "hill centres after deposits", period=w.period)
    if w.method == "abf":
        hp, fp, nb = ctx.abf_state()
        from paper_2301_04835_b200.psg import _view
        assert np.array_equal(_view(hp, (nb,), torch.int32, 0).cpu().numpy(), abf_state[0])
        assert abf_state[0].sum() > 0


def test_fused_step_equals_unfused_calls_bitwise(torch, psg):
    """the fused metadynamics step and the five separate calls give identical bits (same arithmetic, fixed order)"""
    w = small(1, stride=0)
    heights = oracle_heights(w)
    outs = []
    for fused in (True, False):
        ctx = make_ctx(psg, w)
        ctx.load_hills(dev(torch, w.params["hill_centers"]), dev(torch, heights))
        d_pos, d_f = dev(torch, w.positions(1)), torch.zeros((w.R, w.N, 4), device="cuda")
        if fused:
            ctx.step(d_pos, d_f, None, 1)
            o = ctx.read_step_outputs()
            xi, V, dV = o["xi"], o["V"], o["dVdxi"]
        else:
            xi, V, dV = torch.empty((w.R, 2), device="cuda"), torch.empty(w.R, device="cuda"), torch.empty((w.R, 2), device="cuda")
            ctx.cv_eval(d_pos, xi, None)
            ctx.bias_eval(xi, V, dV)
            ctx.apply_bias_forces(d_pos, dV, d_f)
        ctx.sync_check()
        outs.append([t.cpu().numpy() for t in (xi, V, dV)] + [d_f.cpu().numpy()])
    for a, b in zip(outs[0][:3], outs[1][:3]):
        assert np.array_equal(a, b)
    # forces: atoms 6, 8, 14 receive two atomic adds whose order is free -> compare to 1 ulp of the larger term
    assert np.allclose(outs[0][3], outs[1][3], rtol=3e-7, atol=1e-9)


@pytest.mark.parametrize("R,N,weighted", [(3, 5003, False), (2, 2048, False), (5, 6161, True), (1, 100, False), (40, 33000, False)])
def test_fused_range_step_equals_unfused_calls_bitwise(torch, psg, R, N, weighted):
    """config 3 (umbrella windows over large contiguous groups): the one-launch persistent step (TMA-staged slices,
    inter-CTA window reduction) and the separate calls use the same arithmetic in the same order -> same bits;
    several steps in a row check that the window counters re-arm"""
    w = W.make(3, R=R, N=N, steps=3, weighted=weighted)
    f0 = w.forces0()
    res = []
    for fused in (True, False):
        ctx = make_ctx(psg, w)
        d_f = dev(torch, f0)
        launches = []
        for step in (1, 2, 3):
            d_pos = dev(torch, w.positions(step % w.K))
            n0 = ctx.launch_count()
            if fused:
                ctx.step(d_pos, d_f, None, step)
                o = ctx.read_step_outputs()
                xi, V, dV = o["xi"], o["V"], o["dVdxi"]
            else:
                xi, V, dV = (torch.empty((w.R, 2), device="cuda"), torch.empty(w.R, device="cuda"),
                             torch.empty((w.R, 2), device="cuda"))
                ctx.cv_eval(d_pos, xi, None)
                ctx.bias_eval(xi, V, dV)
                ctx.apply_bias_forces(d_pos, dV, d_f)
            launches.append(ctx.launch_count() - n0)
        ctx.sync_check()
        res.append([t.cpu().numpy() for t in (xi, V, dV, d_f)])
        if fused:
            assert launches == [1, 1, 1], f"the umbrella step must be ONE launch, got {launches}"
    for name, a, b in zip(("xi", "V", "dVdxi", "force"), res[0], res[1]):
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), f"{name}: fused and unfused bits differ"


def test_fused_range_step_is_cuda_graph_capturable(torch, psg):
    w = W.make(3, R=4, N=9000, steps=2)
    s = torch.cuda.Stream()
    ctx = psg.Context(0, s)
    psg.configure_from_workload(ctx, w)
    d_pos = dev(torch, w.positions(0))
    d_f = torch.zeros((w.R, w.N, 4), device="cuda")
    ref = torch.zeros_like(d_f)
    with torch.cuda.stream(s):
        ctx.step(d_pos, ref, None, 1)
        ctx.step(d_pos, ref, None, 2)
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        ctx.step(d_pos, d_f, None, 1)
        ctx.step(d_pos, d_f, None, 2)
    d_f.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(d_f.cpu().numpy(), ref.cpu().numpy())


@pytest.mark.parametrize("R,N", [(300, 700), (4100, 64), (1, 30)])
def test_fused_abf_step_equals_unfused_calls(torch, psg, R, N):
    """the one-launch ABF step (CVs -> grid update -> grid barrier -> mean force -> scatter) against the four
    separate calls: xi, bins, dV/dxi inputs and histogram are identical; Fsum and forces differ only by the order
    of the float atomics; R = 4100 makes every warp loop over several replicas"""
    w = W.make(2, R=R, N=N, steps=3)
    f0 = w.forces0()
    res = []
    for fused in (True, False):
        ctx = make_ctx(psg, w)
        d_f = dev(torch, f0)
        for step in (1, 2, 3):
            d_pos, d_fs = dev(torch, w.positions(step % w.K)), dev(torch, w.fsample(step % w.K))
            n0 = ctx.launch_count()
            if fused:
                ctx.step(d_pos, d_f, d_fs, step)
                o = ctx.read_step_outputs()
                xi, b, dV = o["xi"], o["bin"], o["dVdxi"]
                assert ctx.launch_count() - n0 == 1, "the ABF step must be ONE launch"
            else:
                xi, b, dV = (torch.empty((w.R, 2), device="cuda"), torch.empty(w.R, dtype=torch.int32, device="cuda"),
                             torch.empty((w.R, 2), device="cuda"))
                ctx.cv_eval(d_pos, xi, None)
                ctx.abf_update(xi, d_fs, b, dV)
                ctx.apply_bias_forces(d_pos, dV, d_f)
        ctx.sync_check()
        hp, fp, nb = ctx.abf_state()
        from paper_2301_04835_b200.psg import _view
        hist = _view(hp, (nb,), torch.int32, 0).cpu().numpy().copy()
        fsum = _view(fp, (nb, 2), torch.float32, 0).cpu().numpy().copy()
        res.append([xi.cpu().numpy(), b.cpu().numpy(), dV.cpu().numpy(), d_f.cpu().numpy(), hist, fsum])
    a, c = res
    assert np.array_equal(a[0].view(np.uint32), c[0].view(np.uint32)), "xi"
    assert np.array_equal(a[1], c[1]), "bins"
    assert np.array_equal(a[4], c[4]), "histogram"
    assert np.allclose(a[5], c[5], rtol=2e-6, atol=1e-4), "Fsum"
    assert np.allclose(a[2], c[2], rtol=2e-6, atol=1e-6), "dV/dxi"
    assert np.allclose(a[3], c[3], rtol=1e-5, atol=1e-4), "forces"
    assert np.array_equal(a[3][..., 3].view(np.uint32), f0[..., 3].view(np.uint32))


@pytest.mark.parametrize("ps", [3, 4])
def test_fused_abf_step_two_threads_per_cv_kernel_on_weighted_groups(torch, psg, ps):
    """k_abf_step_lean (explicit groups, no box, point-group CVs): weighted groups of 1..3 atoms, per-replica index lists,
    angle + dihedral + component + distance on a 4-D grid, several steps with the grid filling up: xi, bins and histogram
    against the oracle bit for bit, mean forces and forces within the tolerance; and the ctx Jacobian cache it leaves behind"""
    rng = np.random.default_rng(23)
    R, N = 75, 60        # 3 CTAs of 32 replicas, the last one ragged
    groups = lambda b, sizes: [("slots", b + sum(sizes[:i]), sizes[i]) for i in range(len(sizes))]
    cvs_n = [("angle", groups(0, [2, 1, 3]), 0.0, 0), ("dihedral", groups(6, [1, 2, 1, 1]), 2 * math.pi, 0),
             ("component", groups(11, [3]), 0.0, 2), ("distance", groups(14, [1, 2]), 0.0, 0)]
    ok = {"angle": orc.ANGLE, "dihedral": orc.DIHEDRAL, "component": orc.COMPONENT, "distance": orc.DISTANCE}
    gk = {"angle": psg.CV_ANGLE, "dihedral": psg.CV_DIHEDRAL, "component": psg.CV_COM_COMPONENT, "distance": psg.CV_DISTANCE}
    o_cvs = [{"type": ok[k], "groups": g, "axis": ax, "period": p} for k, g, p, ax in cvs_n]
    g_cvs = [{"type": gk[k], "groups": g, "axis": ax, "period": p} for k, g, p, ax in cvs_n]
    slot = np.stack([rng.permutation(N)[:17] for _ in range(R)]).astype(np.int32)
    sw = rng.uniform(1, 16, size=17).astype(np.float32)
    sysm = orc.System(R, N, N, ps, o_cvs, slot, sw, None)
    lower = np.array([0.0, -math.pi, -2.5, 0.0], np.float32)
    upper = np.array([math.pi, math.pi, 2.5, 4.0], np.float32)
    shape, periodic, n_thr = np.array([4, 5, 3, 4], np.int32), np.array([0, 1, 0, 0], np.int32), 2
    nb = int(np.prod(shape))
    hist, fsum = np.zeros(nb, np.int32), np.zeros((nb, 4), np.float64)
    abs_sum = np.zeros((nb, 4))                                   # sum of |f| per bin: what bounds the rounding of the device's Fsum
    slot_cv = np.array([0] * 6 + [1] * 5 + [2] * 3 + [3] * 3)     # CV that owns each of the 17 slots
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, ps, ps)
    ctx.set_cvs(g_cvs, slot, sw, None)
    ctx.set_abf(lower, upper, shape, periodic, n_thr)
    f0 = np.zeros((R, N, ps), np.float32)
    f0[..., :3] = rng.standard_normal((R, N, 3)) * 50
    for step in range(1, 5):
        d_f = dev(torch, f0)      # a fresh force array per step: the tolerance of a binary32 += is relative to ITS operands
        pos = np.zeros((R, N, ps), np.float32)
        pos[..., :3] = rng.normal(scale=0.9, size=(R, N, 3))
        fs = rng.normal(scale=30.0, size=(R, 4)).astype(np.float32)
        n0 = ctx.launch_count()
        ctx.step(dev(torch, pos), d_f, dev(torch, fs), step)
        ctx.sync_check()
        assert ctx.launch_count() - n0 == 1
        out = ctx.read_step_outputs()
        xi_ref, jac_ref = sysm.cv_eval(pos)
        b_ref, dV_ref = orc.abf_update(xi_ref.astype(np.float32), fs, lower, upper, shape, periodic, n_thr, hist, fsum)
        f_ref = sysm.apply_forces(pos, dV_ref, f0[..., :3].astype(np.float64))
        assert_close(out["xi"].cpu().numpy(), xi_ref, f"xi, step {step}", period=np.array([0, 2 * math.pi, 0, 0]))
        assert np.array_equal(out["bin"].cpu().numpy(), b_ref), f"bins, step {step}"
        assert (b_ref >= 0).sum() >= R // 3
        # Fsum is a binary32 sum built by atomics in any order (the oracle's is binary64): the mean force of a bin carries
        # ~ulp32 of sum |f| over the bin's samples, divided by the count, and the forces inherit it through the Jacobian
        inb = b_ref >= 0
        np.add.at(abs_sum, b_ref[inb], np.abs(fs[inb]).astype(np.float64))
        dv_tol = np.zeros((R, 4))
        dv_tol[inb] = 4e-7 * abs_sum[b_ref[inb]] / np.maximum(hist[b_ref[inb]], n_thr)[:, None]
        g = out["dVdxi"].cpu().numpy()
        assert np.all(np.abs(g - dV_ref) <= np.maximum(np.maximum(1e-5 * np.abs(dV_ref), 1e-6), dv_tol)), f"mean force, step {step}"
        extra = np.zeros((R, N, 3))
        for sl in range(17):
            extra[np.arange(R), slot[:, sl]] += dv_tol[:, slot_cv[sl]][:, None] * np.abs(jac_ref[:, sl])
        assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], f"forces, step {step}", extra)
    hp, fp, nbins = ctx.abf_state()
    from paper_2301_04835_b200.psg import _view
    assert np.array_equal(_view(hp, (nb,), torch.int32, 0).cpu().numpy(), hist)
    assert np.allclose(_view(fp, (nb, 4), torch.float32, 0).cpu().numpy(), fsum, rtol=1e-5, atol=1e-3)
    # the estimator on the same layout (k_abf_estimate_lean: one thread per (replica, CV); the weighted groups share no atoms
    # within a replica, the angle and the dihedral of one replica are coupled only through the solve)
    mass = rng.uniform(1.0, 16.0, size=N).astype(np.float32)
    whist = np.zeros((R, 2, 4))
    d_fs = torch.empty((R, 4), device="cuda")
    for est_step in range(3):
        vel = np.zeros((R, N, ps), np.float32)
        vel[..., :3] = rng.normal(scale=0.5, size=(R, N, 3))
        fb = None if est_step == 0 else rng.normal(scale=20.0, size=(R, 4)).astype(np.float32)
        ctx.abf_estimate(dev(torch, pos), dev(torch, vel), dev(torch, mass), 0.002, None if fb is None else dev(torch, fb), d_fs)
        ctx.sync_check()
        ref, Wref = sysm.abf_estimate(pos, vel, mass, 0.002, fb, whist, first=(est_step == 0))
        tol = np.maximum(np.maximum(1e-5 * np.abs(ref), 1e-6), 4e-7 * np.abs(Wref).max(axis=0) / 0.002)
        assert np.all(np.abs(d_fs.cpu().numpy() - ref) <= tol), f"estimator step {est_step}: max err {np.abs(d_fs.cpu().numpy() - ref).max()}"
    # the Jacobian cache the fused step leaves (psg_apply_bias_forces would use it): the oracle's, slot by slot
    d_jac = torch.empty((R, 17, 3), device="cuda")
    d_xi = torch.empty((R, 4), device="cuda")
    ctx.cv_eval(dev(torch, pos), d_xi, d_jac)
    ctx.sync_check()
    assert_close(d_jac.cpu().numpy(), jac_ref, "jacobian of the separate call")
    ctx.close()


def test_abf_shared_grid_split_over_two_contexts(torch, psg):
    """SURVEY 8(e), shared-grid ABF over several GPUs, on one: two contexts hold half of the replicas each, run
    psg_abf_accumulate_delta, exchange by summing the two delta grids (what the all-reduce does), and run
    psg_abf_apply_grid_delta; one context holds all replicas and runs psg_step.  Histograms and bins must agree bit for
    bit (and with the oracle); force sums, mean forces and forces up to the order of the binary32 additions."""
    from paper_2301_04835_b200.psg import _view
    R, N, steps = 600, 90, 4
    w = W.make(2, R=R, N=N, steps=steps)
    h = R // 2
    p = w.params
    f0 = w.forces0()
    nb = int(np.prod(p["shape"]))

    def ctx_for(n):
        c = psg.Context(0)
        c.set_layout(n, N, N, 4, 4)
        cvs = [{"type": psg.CV_DISTANCE, "groups": cv["groups"], "axis": 0, "period": 0.0} for cv in w.cvs]
        c.set_cvs(cvs, w.slot_atom, None, None)
        c.set_abf(p["lower"], p["upper"], p["shape"], p["periodic"], p["n_threshold"])
        return c

    halves, whole = [ctx_for(h), ctx_for(R - h)], ctx_for(R)
    with pytest.raises(psg.PsgError):     # apply without a pending accumulate
        halves[0].abf_apply_grid_delta(torch.zeros(nb, dtype=torch.int32, device="cuda"), torch.zeros(nb * 2, device="cuda"),
                                       dev(torch, w.positions(0)[:h]), dev(torch, f0[:h]))
    d_fw = dev(torch, f0)
    d_fh = [dev(torch, f0[:h]), dev(torch, f0[h:])]
    hist_ref, fsum_ref = np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64)
    for step in range(1, steps + 1):
        pos, fs = w.positions(step % w.K), w.fsample(step % w.K)
        whole.step(dev(torch, pos), d_fw, dev(torch, fs), step)
        parts = [(dev(torch, pos[:h]), dev(torch, fs[:h])), (dev(torch, pos[h:]), dev(torch, fs[h:]))]
        deltas = []
        for c, (dp, dfs) in zip(halves, parts):
            dh = torch.full((nb,), 77, dtype=torch.int32, device="cuda")       # the call must overwrite, not add
            dfm = torch.full((nb * 2,), 7.0, device="cuda")
            c.abf_accumulate_delta(dp, dfs, dh, dfm)
            deltas.append((dh, dfm))
        tot_h, tot_f = deltas[0][0] + deltas[1][0], deltas[0][1] + deltas[1][1]      # the all-reduce
        for c, (dp, _), df in zip(halves, parts, d_fh):
            c.abf_apply_grid_delta(tot_h, tot_f, dp, df)
        for c in halves + [whole]:
            c.sync_check()
        xi = whole.read_step_outputs()["xi"].cpu().numpy()
        b_ref, _ = orc.abf_update(xi, fs, p["lower"], p["upper"], p["shape"], p["periodic"], p["n_threshold"], hist_ref, fsum_ref)
        ow = whole.read_step_outputs()
        oh = [c.read_step_outputs() for c in halves]
        assert np.array_equal(np.concatenate([o["bin"].cpu().numpy() for o in oh]), ow["bin"].cpu().numpy())
        assert np.array_equal(ow["bin"].cpu().numpy(), b_ref)
        assert np.allclose(np.concatenate([o["dVdxi"].cpu().numpy() for o in oh]), ow["dVdxi"].cpu().numpy(), rtol=2e-6, atol=1e-6)
    grids = []
    for c in halves + [whole]:
        hp, fp, n = c.abf_state()
        grids.append((_view(hp, (n,), torch.int32, 0).cpu().numpy().copy(), _view(fp, (n, 2), torch.float32, 0).cpu().numpy().copy()))
    assert np.array_equal(grids[0][0], grids[2][0]) and np.array_equal(grids[1][0], grids[2][0]), "histogram, bit for bit"
    assert np.array_equal(grids[2][0], hist_ref) and hist_ref.sum() > R
    assert np.array_equal(grids[0][1].view(np.uint32), grids[1][1].view(np.uint32)), "both ranks hold the identical grid"
    assert_close(grids[0][1], fsum_ref, "Fsum of the split update")
    assert np.allclose(np.concatenate([d_fh[0].cpu().numpy(), d_fh[1].cpu().numpy()]), d_fw.cpu().numpy(), rtol=1e-5, atol=1e-4)


def test_fused_abf_step_is_cuda_graph_capturable(torch, psg):
    """the cooperative one-launch ABF step replays from a CUDA graph and leaves its grid barrier re-armed"""
    w = W.make(2, R=600, N=100, steps=2)
    s = torch.cuda.Stream()
    outs = []
    for graph in (False, True):
        ctx = psg.Context(0, s)
        psg.configure_from_workload(ctx, w)
        d_pos, d_fs = dev(torch, w.positions(0)), dev(torch, w.fsample(0))
        d_f = torch.zeros((w.R, w.N, 4), device="cuda")
        torch.cuda.synchronize()
        if graph:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                ctx.step(d_pos, d_f, d_fs, 1)
            d_f.zero_()
            ctx.set_abf(w.params["lower"], w.params["upper"], w.params["shape"], w.params["periodic"], w.params["n_threshold"])
            torch.cuda.synchronize()
            for _ in range(3):
                g.replay()
        else:
            with torch.cuda.stream(s):
                for _ in range(3):
                    ctx.step(d_pos, d_f, d_fs, 1)
        torch.cuda.synchronize()
        hp, fp, nb = ctx.abf_state()
        from paper_2301_04835_b200.psg import _view
        outs.append((_view(hp, (nb,), torch.int32, 0).cpu().numpy().copy(), d_f.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and outs[0][0].sum() > 0
    assert np.allclose(outs[0][1], outs[1][1], rtol=1e-5, atol=1e-4)


def test_metad_step_more_tiles_than_ctas(torch, psg):
    """20,000 walkers = 313 replica tiles for ~148 CTAs: every CTA of the persistent k_hills loops over several
    (tile, chunk) items (stage ring, tickets and partial buffers are reused across items); R is not a multiple of 64"""
    w = W.make(1, R=20000, n_hills=2600, steps=2, stride=0)
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    centers, heights = w.params["hill_centers"], oracle_heights(w)
    ctx.load_hills(dev(torch, centers), dev(torch, heights))
    pos, f0 = w.positions(1), w.forces0()
    d_f = dev(torch, f0)
    for _ in range(2):                      # twice: the second launch must find tickets / counters re-armed
        d_f.copy_(dev(torch, f0))
        ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0, centers, heights)
    _check_step(w, sysm, pos, out["xi"], out["V"], out["dVdxi"], d_f.cpu().numpy(), f0, xi_ref, b, f_ref, what="R=20000: ")


def test_abf_step_at_the_replica_limit(torch, psg):
    """65,535 replicas (the ctx maximum): every warp of the cooperative k_abf_step loops over many replicas"""
    w = W.make(2, R=65535, N=40, steps=2)
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    pos, f0, fs = w.positions(0), w.forces0(), w.fsample(0)
    nb = int(np.prod(w.params["shape"]))
    abf = (np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64))
    d_f = dev(torch, f0)
    ctx.step(dev(torch, pos), d_f, dev(torch, fs), 1)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0, None, None, abf, fs)
    assert np.array_equal(out["bin"], b["bin"])
    hp, fp, nbins = ctx.abf_state()
    from paper_2301_04835_b200.psg import _view
    assert np.array_equal(_view(hp, (nbins,), torch.int32, 0).cpu().numpy(), abf[0])
    _check_step(w, sysm, pos, out["xi"], None, out["dVdxi"], d_f.cpu().numpy(), f0, xi_ref, b, f_ref, what="R=65535: ")


def _range_workload(R, N, cvs, weighted=False):
    """config-3 geometry with a custom list of range-group CVs (windows' centres re-cut to the number of CVs)"""
    w = W.make(3, R=R, N=N, steps=2, weighted=weighted)
    w.cvs = cvs
    c = 1.0 + 4.0 * np.arange(R) / max(R - 1, 1)
    w.params = {"kspring": np.full(len(cvs), 1000.0, np.float32),
                "centers": np.stack([c] * len(cvs), axis=1).astype(np.float32)}
    return w


@pytest.mark.parametrize("case", ["gap", "angle3", "limit", "over_limit"])
def test_fused_range_step_shapes(torch, psg, case):
    """k_range_step on shapes config 3 does not have: groups that leave a GAP in their span (those atoms must keep
    their force bits), a three-group CV with an Rg CV on an overlapping range, a window of exactly `grid` slices,
    and one slice more than that (falls back to the separate kernels); all against the oracle"""
    props = torch.cuda.get_device_properties(0)
    n_lim = props.multi_processor_count * 2048
    if case == "gap":
        R, N, want = 5, 9000, 1
        cvs = [W._cv("distance", [("range", 100, 1900), ("range", 5000, 3500)])]
    elif case == "angle3":
        R, N, want = 4, 12000, 1
        cvs = [W._cv("angle", [("range", 0, 4000), ("range", 4000, 4000), ("range", 8000, 4000)]),
               W._cv("rgyr", [("range", 2000, 9000)])]
    elif case == "limit":
        R, N, want = 1, n_lim, 1
        cvs = [W._cv("rgyr", [("range", 0, N)]), W._cv("distance", [("range", 0, N // 2), ("range", N // 2, N - N // 2)])]
    else:
        R, N, want = 1, n_lim + 1, 4
        cvs = [W._cv("rgyr", [("range", 0, N)]), W._cv("distance", [("range", 0, N // 2), ("range", N // 2, N - N // 2)])]
    w = _range_workload(R, N, cvs, weighted=(case == "angle3"))
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    pos, f0 = w.positions(1), w.forces0()
    d_f = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    assert ctx.launch_count() - n0 == want
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0)
    _check_step(w, sysm, pos, out["xi"], out["V"], out["dVdxi"], d_f.cpu().numpy(), f0, xi_ref, b, f_ref, what=case + ": ")


def test_internal_cv_forces_have_no_net_force_or_torque(torch, psg):
    """sum_i F_i = 0 and sum_i r_i x F_i = 0 for internal CVs (BASELINE.json), on the GPU forces themselves"""
    w = small(1, stride=0)
    ctx = make_ctx(psg, w)
    ctx.load_hills(dev(torch, w.params["hill_centers"]), dev(torch, oracle_heights(w)))
    pos = w.positions(0)
    d_f = torch.zeros((w.R, w.N, 4), device="cuda")
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    f = d_f.cpu().numpy()[..., :3].astype(np.float64)
    x = pos[..., :3].astype(np.float64)
    scale = np.abs(f).sum(axis=(1, 2)) + 1e-30
    assert np.all(np.abs(f.sum(axis=1)).max(axis=1) <= 2e-6 * scale)
    assert np.all(np.abs(np.cross(x, f).sum(axis=1)).max(axis=1) <= 1e-5 * scale)


def test_step_host_matches_device_step(torch, psg):
    w = small(3)
    pos, f0 = w.positions(0), w.forces0()
    ctx = make_ctx(psg, w)
    d_f = dev(torch, f0)
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    ctx2 = make_ctx(psg, w)
    h_pos, h_f = torch.from_numpy(pos).pin_memory(), torch.from_numpy(f0.copy()).pin_memory()
    ctx2.step_host(h_pos, h_f, None, 1)
    assert np.array_equal(h_f.numpy(), d_f.cpu().numpy())


def test_step_is_cuda_graph_capturable(torch, psg):
    w = small(1, stride=0)
    heights = oracle_heights(w)
    s = torch.cuda.Stream()
    ctx = psg.Context(0, s)
    psg.configure_from_workload(ctx, w)
    ctx.load_hills(dev(torch, w.params["hill_centers"]), dev(torch, heights))
    d_pos = dev(torch, w.positions(0))
    d_f = torch.zeros((w.R, w.N, 4), device="cuda")
    ref = torch.zeros_like(d_f)
    with torch.cuda.stream(s):
        ctx.step(d_pos, ref, None, 1)
        ctx.step(d_pos, ref, None, 2)
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        ctx.step(d_pos, d_f, None, 1)
        ctx.step(d_pos, d_f, None, 2)
    d_f.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert np.allclose(d_f.cpu().numpy(), ref.cpu().numpy(), rtol=3e-7, atol=1e-9)


# ------------------------------------------------------------------------------------ minimum image
def _wrapped(w, pos, box):
    """the same atoms as an engine with periodic boundaries stores them: every coordinate wrapped into [0, L)"""
    p = pos.copy()
    p[..., :3] = np.mod(p[..., :3].astype(np.float64), np.asarray(box)).astype(np.float32)
    return p


@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_minimum_image_step_matches_oracle(torch, psg, cfg):
    """psg_set_box: with every atom wrapped into a box SMALLER than the molecules' excursions, the fused steps (k_hills
    prologue, k_abf_step) and psg_cv_eval give the oracle's minimum-image CVs, Jacobians and forces; ADP chains are
    ~0.5 nm across, the box is 1.3 nm, so most replicas have groups on both sides of a face"""
    w = small(cfg)
    box = (1.3, 1.45, 1.6) if cfg != 2 else (4.7, 5.1, 4.9)
    if cfg == 4:
        box = (3.9, 4.1, 4.3)       # the distance pair of config 4 is up to 1.5 nm apart: L/2 must exceed it
    ctx = make_ctx(psg, w)
    ctx.set_box(box)
    cvs = [{"type": {"distance": orc.DISTANCE, "angle": orc.ANGLE, "dihedral": orc.DIHEDRAL, "component": orc.COMPONENT,
                     "rgyr": orc.RGYR}[cv["kind"]], "groups": cv["groups"], "axis": cv["axis"], "period": cv["period"]}
           for cv in w.cvs]
    sysm = orc.System(w.R, w.N, 0 if w.shared_array else w.N, 4, cvs, w.slot_atom, None, w.atom_weight, box=box)
    pos = _wrapped(w, w.positions(1), box)
    f0 = w.forces0()
    centers = heights = abf_state = fs = None
    if w.method == "metad":
        centers, heights = w.params["hill_centers"], oracle_heights(w)
        ctx.load_hills(dev(torch, centers), dev(torch, heights))
    if w.method == "abf":
        nb = int(np.prod(w.params["shape"]))
        abf_state, fs = (np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64)), w.fsample(1)
    # separate call first: CVs and the compact Jacobian
    d_pos = dev(torch, pos)
    d_xi = torch.empty((w.R, w.n_cv), device="cuda")
    d_jac = torch.empty((w.R, w.slot_atom.shape[-1], 3), device="cuda")
    ctx.cv_eval(d_pos, d_xi, d_jac)
    xi_ref, jac_ref = sysm.cv_eval(pos)
    assert_close(d_xi.cpu().numpy(), xi_ref, "xi (minimum image)", period=w.period)
    assert_close(d_jac.cpu().numpy(), jac_ref[:, slot_rows(w)], "Jacobian (minimum image)")
    # the open-boundary result differs for the replicas that straddle a face: the box is really in play
    open_sys = oracle_system(w)
    assert np.abs(wrap(open_sys.cv_eval(pos, want_jac=False) - xi_ref, w.period)).max() > 1e-2
    # fused step
    d_f = dev(torch, f0)
    ctx.step(d_pos, d_f, None if fs is None else dev(torch, fs), 1)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    xi_ref, b, f_ref = oracle_step(w, sysm, pos, f0, centers, heights, abf_state, fs)
    if w.method == "abf":
        assert np.array_equal(out["bin"], b["bin"])
    _check_step(w, sysm, pos, out["xi"], out.get("V"), out["dVdxi"], d_f.cpu().numpy(), f0, xi_ref, b, f_ref,
                what=f"minimum image, config {cfg}: ")


def test_set_box_validation(torch, psg):
    w = small(3)
    ctx = make_ctx(psg, w)
    ctx.set_box((30.0, 30.0, 30.0))           # range groups follow the rule of explicit groups (first atom of the range)
    ctx.set_box(None)                          # switching it off is always fine
    w1 = small(1)
    c1 = make_ctx(psg, w1)
    with pytest.raises(psg.PsgError):
        c1.set_box((3.0, -1.0, 3.0))
    c1.set_box((0.0, 0.0, 0.0))


def test_minimum_image_range_groups_match_oracle(torch, psg):
    """SURVEY NEXT-4 "unwrapping large groups": umbrella windows over contiguous-range groups (Rg of the chain, distance of
    the two halves' centers of mass, mass-weighted) whose atoms were wrapped one by one into a periodic box; the step takes
    the streaming kernels (k_range_step is for open boundaries) and must match the oracle with the same box"""
    w = small(3, R=4, N=6007, weighted=True)
    ext = float(np.ptp(w.positions(0)[..., :3], axis=1).max())
    L = np.ceil(np.array([2.6, 2.3, 3.0]) * ext)             # every chain spans less than half of the box
    sysm = orc.System(w.R, w.N, w.N, 4, [{"type": {"rgyr": orc.RGYR, "distance": orc.DISTANCE}[cv["kind"]], "groups": cv["groups"],
                                          "axis": 0, "period": 0.0} for cv in w.cvs], None, atom_weight=w.atom_weight, box=L)
    pos = w.positions(0).copy()
    assert np.ptp(pos[..., :3], axis=1).max() < 0.45 * L.min()
    unwrapped = pos[..., :3].astype(np.float64) + 0.93 * L          # the chains straddle the upper faces
    pos[..., :3] = np.mod(unwrapped, L).astype(np.float32)
    assert (np.abs(pos[..., :3] - unwrapped) > 1).mean() > 0.2        # a good part of every chain is wrapped
    pos[..., :3] = np.where(pos[..., :3] >= L.astype(np.float32), 0.0, pos[..., :3])
    f0 = w.forces0()
    ctx = make_ctx(psg, w)
    ctx.set_box(L)
    d_f = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    assert ctx.launch_count() - n0 == 4                      # moments, CVs, bias, dense apply
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    xi_ref = sysm.cv_eval(pos, want_jac=False)
    assert_close(out["xi"], xi_ref, "wrapped range groups: xi")
    b = oracle_bias(w, xi_ref.astype(np.float32))
    assert_close(out["V"], b["V"], "V")
    assert_close(out["dVdxi"], b["dVdxi"], "dV/dxi")
    f_ref = sysm.apply_forces(pos, b["dVdxi"], f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "wrapped range groups: forces")
    assert np.array_equal(d_f.cpu().numpy()[..., 3].view(np.uint32), f0[..., 3].view(np.uint32))
    # and the torn chain without the box is something else
    ctx.set_box(None)
    ctx.step(dev(torch, pos), dev(torch, f0), None, 1)
    ctx.sync_check()
    assert np.abs(ctx.read_step_outputs()["xi"].cpu().numpy() - xi_ref).max() > 0.5
    ctx.close()


# ------------------------------------------------------------------------------------ ABF force estimator
@pytest.mark.parametrize("cfg,R", [(1, 70), (2, 300), (4, 130)])
def test_abf_force_estimator_matches_oracle(torch, psg, cfg, R):
    """psg_abf_estimate over five MD steps of a synthetic trajectory (positions and velocities change every step, a bias is
    fed back from the second step on) against the oracle's reading R-ABF-EST: dihedral pairs that share three atoms
    (config 1), barycenter groups (config 2), per-replica index lists on a shared array with colliding walkers (config 4).
    The sample is a difference quotient of W over dt, so its rounding floor is ~ulp(W)/dt: compared with
    |d| <= max(1e-5 |ref|, 1e-6, 4e-7 * max|W| / dt)."""
    w = small(cfg) if cfg != 1 else small(cfg, R=R)
    ctx = make_ctx(psg, w, with_method=False)
    sysm = oracle_system(w)
    rng = np.random.default_rng(1000 + cfg)
    n_arr = 1 if w.shared_array else w.R
    mass = rng.uniform(1.0, 16.0, size=w.N).astype(np.float32)
    dt = 0.002
    hist = np.zeros((w.R, 2, w.n_cv))
    d_fs = torch.empty((w.R, w.n_cv), device="cuda")
    d_mass = dev(torch, mass)
    vel0 = rng.normal(scale=0.5, size=(n_arr, w.N, 4)).astype(np.float32)
    for step in range(5):
        pos = w.positions(step % w.K)
        vel = (vel0 + 0.05 * step * rng.normal(size=vel0.shape)).astype(np.float32)
        fb = None if step == 0 else rng.normal(scale=20.0, size=(w.R, w.n_cv)).astype(np.float32)
        ctx.abf_estimate(dev(torch, pos), dev(torch, vel), d_mass, dt, None if fb is None else dev(torch, fb), d_fs)
        ctx.sync_check()
        ref, W = sysm.abf_estimate(pos, vel, mass, dt, fb, hist, first=(step == 0))
        got = d_fs.cpu().numpy()
        tol = np.maximum(np.maximum(1e-5 * np.abs(ref), 1e-6), 4e-7 * np.abs(W).max(axis=0) / dt)
        assert np.all(np.abs(got - ref) <= tol), f"step {step}: max err {np.abs(got - ref).max()}"
    # after a reset the history starts again: the sample is the fed-back bias alone
    ctx.abf_estimate_reset()
    fb = np.full((w.R, w.n_cv), 3.5, np.float32)
    ctx.abf_estimate(dev(torch, pos), dev(torch, vel), d_mass, dt, dev(torch, fb), d_fs)
    assert np.array_equal(d_fs.cpu().numpy(), fb)


def test_abf_estimator_feeds_the_abf_step(torch, psg):
    """estimator -> psg_step (ABF) -> the mean force of that step fed back to the next estimate: the chained device path
    against the same chain in the oracle, bins and histogram bit-exact"""
    w = small(2)
    ctx = make_ctx(psg, w)
    sysm = oracle_system(w)
    rng = np.random.default_rng(77)
    mass = rng.uniform(1.0, 16.0, size=w.N).astype(np.float32)
    dt = 0.002
    nb = int(np.prod(w.params["shape"]))
    abf = (np.zeros(nb, np.int32), np.zeros((nb, 2), np.float64))
    hist = np.zeros((w.R, 2, w.n_cv))
    d_fs = torch.empty((w.R, w.n_cv), device="cuda")
    d_f = dev(torch, w.forces0())
    fb_ref = None
    d_fb = None
    for step in range(1, 5):
        pos = w.positions(step % w.K)
        # velocities with a strong common drift along the CV directions keep the samples same-sign dominated
        vel = (rng.normal(scale=0.02, size=(w.R, w.N, 4)) + 0.3 * step).astype(np.float32)
        ctx.abf_estimate(dev(torch, pos), dev(torch, vel), dev(torch, mass), dt, d_fb, d_fs)
        ctx.step(dev(torch, pos), d_f, d_fs, step)
        ctx.sync_check()
        out = ctx.read_step_outputs()
        fs_ref, _ = sysm.abf_estimate(pos, vel, mass, dt, fb_ref, hist, first=(step == 1))
        fs_gpu = d_fs.cpu().numpy()
        # the oracle's chain continues from the DEVICE's binary32 samples, so that a last-bit difference of a sample cannot
        # move a walker across a bin edge of the comparison (the sample itself is compared above and here)
        assert np.all(np.abs(fs_gpu - fs_ref) <= np.maximum(np.maximum(1e-5 * np.abs(fs_ref), 1e-6), 4e-7 * 50.0 / dt))
        xi_ref = sysm.cv_eval(pos, want_jac=False)
        b = oracle_bias(w, xi_ref.astype(np.float32), None, None, abf, fs_gpu)
        assert np.array_equal(out["bin"].cpu().numpy(), b["bin"])
        assert_close(out["dVdxi"].cpu().numpy(), b["dVdxi"], f"mean force, step {step}")
        fb_ref = out["dVdxi"].cpu().numpy().astype(np.float64)
        d_fb = out["dVdxi"]
    hp, fp, nbins = ctx.abf_state()
    from paper_2301_04835_b200.psg import _view
    assert np.array_equal(_view(hp, (nbins,), torch.int32, 0).cpu().numpy(), abf[0])


def test_displacement_cv_harmonic_step(torch, psg):
    """Displacement: the three components of the barycenter difference of two weighted
    explicit groups as three CVs, harmonically restrained, through psg_cv_eval and the whole step, with and without a box"""
    rng = np.random.default_rng(31)
    R, N = 37, 60
    xyz = rng.uniform(0.0, 3.0, size=(R, N, 3)).astype(np.float32)
    pos = np.concatenate([xyz, rng.normal(size=(R, N, 1)).astype(np.float32)], axis=2)
    slots = np.array([3, 7, 11, 20, 21], np.int32)
    wts = np.array([1.0, 12.0, 16.0, 1.0, 14.0], np.float32)
    for box in (None, (3.0, 3.0, 3.0)):
        ctx = psg.Context(0)
        ctx.set_layout(R, N, N, 4, 4)
        # every slot belongs to exactly one (CV, group): the three CVs list the five atoms three times
        sl = np.concatenate([slots, slots, slots])
        cvs = [{"type": psg.CV_DISPLACEMENT, "groups": [("slots", 5 * ax, 3), ("slots", 5 * ax + 3, 2)], "axis": ax, "period": 0.0}
               for ax in range(3)]
        ctx.set_cvs(cvs, sl, np.concatenate([wts, wts, wts]))
        if box is not None:
            ctx.set_box(box)
        k = np.array([300.0, 500.0, 700.0], np.float32)
        cen = rng.normal(scale=0.3, size=(R, 3)).astype(np.float32)
        ctx.set_harmonic(k, cen)
        o_cvs = [{"type": orc.DISPLACEMENT, "groups": c["groups"], "axis": c["axis"], "period": 0.0} for c in cvs]
        sysm = orc.System(R, N, N, 4, o_cvs, sl, np.concatenate([wts, wts, wts]), None, box=box)
        f0 = rng.normal(scale=100.0, size=(R, N, 4)).astype(np.float32)
        d_f = dev(torch, f0)
        ctx.step(dev(torch, pos), d_f, None, 1)
        ctx.sync_check()
        out = {kk: v.cpu().numpy() for kk, v in ctx.read_step_outputs().items()}
        xi_ref = sysm.cv_eval(pos, want_jac=False)
        V, dV = orc.harmonic(xi_ref.astype(np.float32).astype(np.float64), k, cen, np.zeros(3))
        f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
        assert_close(out["xi"], xi_ref, "displacement xi")
        assert_close(out["V"], V, "V")
        assert_close(out["dVdxi"], dV, "dV/dxi")
        assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "forces")
        ctx.close()


# ------------------------------------------------------------------------------------ DistanceToInterface
@pytest.mark.parametrize("R,n_i,bins,axis", [(3, 700, 40, 0), (9, 5000, 100, 2), (1, 1025, 2, 1)])
def test_distance_to_interface_matches_oracle(torch, psg, R, n_i, bins, axis):
    """the paper's worked CV (Eq. 4-8, App. A): liquid slabs with a diffuse edge, one per replica; value and the
    force of a harmonic restraint on it (interface atoms through the softmax, mobile atoms through the barycenter) against
    the oracle; chunks of 1,024 atoms with a ragged tail; bins = 2 is the one-entry softmax"""
    rng = np.random.default_rng(50 + R)
    n_m = 3
    N = n_m + n_i + 5
    pos = rng.normal(scale=2.0, size=(R, N, 4)).astype(np.float32)
    for r in range(R):
        edge = 0.3 + 0.2 * r
        x = np.concatenate([rng.uniform(-4.0, edge, size=n_i - n_i // 8), edge + np.abs(rng.normal(scale=0.4, size=n_i // 8))])
        pos[r, n_m:n_m + n_i, axis] = x.astype(np.float32)
    mob, wm = np.array([0, 2, 1], np.int32), np.array([1.0, 4.0, 2.0], np.float32)
    sigma, scope, coeff = 0.25, (-3.0, 3.5), 0.9
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.interface_cv_set(mob, wm, n_m, n_i, axis, sigma, scope, bins, coeff)
    d_pos = dev(torch, pos)
    d_xi = torch.empty(R, device="cuda")
    ctx.interface_cv_eval(d_pos, d_xi)
    ctx.sync_check()
    ref = [orc.dist_to_interface(pos[r], mob, wm, n_m, n_i, axis, sigma, scope, bins, coeff) for r in range(R)]
    xi_ref = np.array([q[0] for q in ref])
    assert_close(d_xi.cpu().numpy(), xi_ref, "distance to interface")
    k, x0 = 800.0, 0.1
    dV = (k * (xi_ref.astype(np.float32).astype(np.float64) - x0)).astype(np.float32)
    f0 = rng.normal(scale=100.0, size=(R, N, 4)).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.interface_cv_apply(d_pos, dev(torch, dV), d_f)
    ctx.sync_check()
    f = d_f.cpu().numpy()
    f_ref = f0[..., :3].astype(np.float64)
    for r in range(R):
        _, jm, dx, _ = ref[r]
        f_ref[r, n_m:n_m + n_i, axis] += -float(dV[r]) * dx
        for m, a in enumerate(mob):
            f_ref[r, a] += -float(dV[r]) * jm[m]
    assert_forces_close(f[..., :3], f_ref, f0[..., :3], "interface CV forces")
    untouched = np.ones(N, bool)
    untouched[n_m:n_m + n_i] = False
    untouched[mob] = False
    assert np.array_equal(f[:, untouched].view(np.uint32), f0[:, untouched].view(np.uint32))
    other = [x for x in range(4) if x != axis]
    assert np.array_equal(f[:, n_m:n_m + n_i][..., other].view(np.uint32), f0[:, n_m:n_m + n_i][..., other].view(np.uint32))


# ------------------------------------------------------------------------------------ error behaviour
def test_distance_to_interface_as_a_cv_of_the_step(torch, psg):
    """PSG_CV_DIST_TO_INTERFACE (Eq. 4-8, App. A) as a psg_cv_desc type: next to a Distance CV, under a harmonic
    bias and under ABF, through psg_step (the separate kernels in sequence); value, bias and forces against the oracle's
    pieces (its DistanceToInterface with derivatives, its harmonic / ABF stage, its Distance Jacobian)"""
    rng = np.random.default_rng(31)
    R, N, axis = 5, 1400, 2
    mob = np.array([3, 9, 1200], np.int32)                    # the last mobile atom lies inside the interface range
    mw = np.array([1.0, 2.5, 0.5], np.float32)
    ib, ni = 40, 1300
    dti = {"sigma": 0.25, "scope": (1.0, 5.0), "bins": 33, "coeff": 3.0}
    pos = np.zeros((R, N, 4), np.float32)
    pos[..., :3] = rng.uniform(0.0, 6.0, size=(R, N, 3))
    pos[:, ib:ib + ni, axis] = np.where(rng.uniform(size=(R, ni)) < 0.5, rng.uniform(0.5, 2.8, size=(R, ni)), rng.uniform(2.8, 5.5, size=(R, ni)) * 0.7 + 1.0)
    pos[..., 3] = 7.0
    slots = np.concatenate([mob, [700, 701]]).astype(np.int32)          # slots 0..2 mobile, 3 and 4 the Distance pair
    sw = np.concatenate([mw, [1.0, 1.0]]).astype(np.float32)
    cvs = [{"type": psg.CV_DIST_TO_INTERFACE, "groups": [("slots", 0, 3), ("range", ib, ni)], "axis": axis, "period": 0.0, "dti": dti},
           {"type": psg.CV_DISTANCE, "groups": [("slots", 3, 1), ("slots", 4, 1)], "axis": 0, "period": 0.0}]
    o_dist = orc.System(R, N, N, 4, [{"type": orc.DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)], "axis": 0, "period": 0.0}],
                        np.array([700, 701], np.int32), None, None)
    xi_ref = np.zeros((R, 2))
    jm, dx = [], []
    for r in range(R):
        x, j, d, _ = orc.dist_to_interface(pos[r], mob, mw, ib, ni, axis, dti["sigma"], dti["scope"], dti["bins"], dti["coeff"])
        xi_ref[r, 0] = x; jm.append(j); dx.append(d)
    xi_ref[:, 1] = o_dist.cv_eval(pos, want_jac=False)[:, 0]
    f0 = (rng.standard_normal((R, N, 4)) * 50).astype(np.float32)

    def forces_ref(dV):
        f = f0[..., :3].astype(np.float64)
        f = o_dist.apply_forces(pos, dV[:, 1:2], f)
        for r in range(R):
            np.add.at(f[r], mob, -dV[r, 0] * jm[r])
            f[r, ib:ib + ni, axis] += -dV[r, 0] * dx[r]
        return f

    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.set_cvs(cvs, slots, sw, None)
    # -- harmonic
    ks, cen = np.array([400.0, 150.0], np.float32), np.stack([np.linspace(-0.5, 0.5, R), np.full(R, 2.0)], axis=1).astype(np.float32)
    ctx.set_harmonic(ks, cen)
    d_f = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    assert ctx.launch_count() - n0 == 6          # k_cv_eval, two interface kernels, k_harmonic, k_apply_sparse, k_dti_apply
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    assert_close(out["xi"], xi_ref, "xi (interface CV + distance)")
    V, dV = orc.harmonic(xi_ref.astype(np.float32).astype(np.float64), ks, cen, np.zeros(2))
    assert_close(out["V"], V, "V")
    assert_close(out["dVdxi"], dV, "dV/dxi")
    assert_forces_close(d_f.cpu().numpy()[..., :3], forces_ref(dV), f0[..., :3], "forces through the interface CV")
    assert np.array_equal(d_f.cpu().numpy()[..., 3].view(np.uint32), f0[..., 3].view(np.uint32))
    # -- ABF on the same two CVs: bins bit-exact, the mean force scattered through both Jacobians
    lower, upper = np.array([-3.0, 0.0], np.float32), np.array([3.0, 9.0], np.float32)
    shape, periodic = np.array([12, 9], np.int32), np.array([0, 0], np.int32)
    ctx.set_abf(lower, upper, shape, periodic, 2)
    fs = rng.normal(scale=10.0, size=(R, 2)).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.step(dev(torch, pos), d_f, dev(torch, fs), 1)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    hist, fsum = np.zeros(108, np.int32), np.zeros((108, 2), np.float64)
    b, dVa = orc.abf_update(out["xi"], fs, lower, upper, shape, periodic, 2, hist, fsum)
    assert np.array_equal(out["bin"], b) and (b >= 0).sum() >= 2     # (out-of-grid replicas get no mean force)
    assert_close(out["dVdxi"], dVa, "ABF mean force")
    assert_forces_close(d_f.cpu().numpy()[..., :3], forces_ref(dVa), f0[..., :3], "ABF forces through the interface CV")
    # -- argument checks
    bad = [dict(cvs[0], groups=[("range", 0, 3), ("range", ib, ni)]), cvs[1]]
    with pytest.raises(psg.PsgError):
        ctx.set_cvs(bad, slots, sw, None)
    with pytest.raises(psg.PsgError):
        ctx.set_cvs([cvs[0], dict(cvs[0], groups=[("slots", 3, 2), ("range", ib, ni)])], slots, sw, None)   # two of them
    ctx.close()


def test_argument_validation(torch, psg):
    ctx = psg.Context(0)
    with pytest.raises(psg.PsgError) as e:
        ctx.set_cvs([{"type": psg.CV_DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)]}], np.arange(2))
    assert e.value.code == -5                                  # PSG_ESTATE: layout first
    ctx.set_layout(2, 10, 10, 4, 4)
    with pytest.raises(psg.PsgError) as e:
        ctx.set_cvs([{"type": psg.CV_DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)]}], np.array([0, 10]))
    assert e.value.code == -1                                  # index out of range
    with pytest.raises(psg.PsgError):
        ctx.set_layout(2, 10, 10, 5, 4)
    ctx.set_cvs([{"type": psg.CV_DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)]}], np.array([0, 9]))
    x = torch.zeros((2, 10, 4), device="cuda")
    with pytest.raises(psg.PsgError) as e:
        ctx.step(x, x.clone(), None, 1)
    assert e.value.code == -5                                  # no method selected
    with pytest.raises(psg.PsgError) as e:
        ctx.apply_bias_forces(x, torch.zeros((2, 1), device="cuda"), x.clone())
    assert e.value.code == -5                                  # no cached Jacobian
    with pytest.raises(psg.PsgError) as e:
        ctx.cv_eval(x, None, None)
    assert e.value.code == -1
    with pytest.raises(ValueError):
        ctx.cv_eval(x.double(), torch.zeros((2, 1), device="cuda"), None)


# ------------------------------------------------------------------------------------ gyration-tensor shape CVs
def _shape_molecules(rng, R, N, box=None):
    """R replicas of N atoms: an anisotropic blob per replica (axes 2 : 1 : 0.5 after a random rotation, so that the three
    eigenvalues are well separated), somewhere in a 6 nm region; wrapped into ``box`` when one is given"""
    pos = np.empty((R, N, 3), np.float32)
    for r in range(R):
        q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
        pos[r] = (rng.normal(size=(N, 3)) * [0.5, 0.25, 0.12]) @ q.T + rng.uniform(0.0, 6.0, size=3)
    if box is not None:
        pos = np.mod(pos, np.asarray(box, np.float32)).astype(np.float32)
    return pos


@pytest.mark.parametrize("box", [None, (4.0, 4.5, 5.0)])
@pytest.mark.parametrize("which", [0, 1])
def test_shape_cvs_match_oracle(torch, psg, which, box):
    """PrincipalMoment(0..2), Asphericity, Acylindricity, ShapeAnisotropy (reading R-SHAPE) of weighted
    explicit groups with per-replica indices and stride-3 positions: values, the compact Jacobian, and the forces of a
    harmonic restraint through the whole step; with a box the molecules are wrapped and most straddle a face"""
    rng = np.random.default_rng(70 + which)
    R, N = 41, 48
    pos = _shape_molecules(rng, R, N, box)
    sizes = [12, 9, 7, 5]
    n_slots = sum(sizes)
    slot = np.stack([rng.permutation(N)[:n_slots] for _ in range(R)]).astype(np.int32)
    sw = rng.uniform(1, 16, size=n_slots).astype(np.float32)
    begin = np.concatenate([[0], np.cumsum(sizes)[:-1]])
    kinds = [[("PRINCIPAL_MOMENT", 0), ("PRINCIPAL_MOMENT", 1), ("PRINCIPAL_MOMENT", 2), ("ASPHERICITY", 0)],
             [("ACYLINDRICITY", 0), ("SHAPE_ANISOTROPY", 0), ("RGYR", 0), ("PRINCIPAL_MOMENT", 1)]][which]
    o_cvs = [{"type": getattr(orc, k), "groups": [("slots", int(begin[i]), sizes[i])], "axis": ax, "period": 0.0}
             for i, (k, ax) in enumerate(kinds)]
    g_cvs = [{"type": getattr(psg, "CV_" + k), "groups": [("slots", int(begin[i]), sizes[i])], "axis": ax, "period": 0.0}
             for i, (k, ax) in enumerate(kinds)]
    sysm = orc.System(R, N, N, 3, o_cvs, slot, sw, None, box=box)
    xi_ref, jac_ref = sysm.cv_eval(pos)
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 3, 3)
    ctx.set_cvs(g_cvs, slot, sw, None)
    if box is not None:
        ctx.set_box(box)
    d_xi = torch.empty((R, 4), device="cuda")
    d_jac = torch.empty((R, n_slots, 3), device="cuda")
    d_pos = dev(torch, pos)
    ctx.cv_eval(d_pos, d_xi, d_jac)
    ctx.sync_check()
    assert_close(d_xi.cpu().numpy(), xi_ref, "shape xi")
    assert_close(d_jac.cpu().numpy(), jac_ref, "shape jacobian")
    if box is not None:   # the box is really in play: the open-boundary tensor of a split molecule is far larger
        open_xi = orc.System(R, N, N, 3, o_cvs, slot, sw, None).cv_eval(pos, want_jac=False)
        assert (np.abs(open_xi - xi_ref) > 1e-3 * np.abs(xi_ref)).any()
    ks = np.array([400, 900, 2000, 700], np.float32)
    cen = (xi_ref * rng.uniform(0.5, 1.5, size=xi_ref.shape)).astype(np.float32)
    ctx.set_harmonic(ks, cen)
    f0 = (rng.standard_normal((R, N, 3)) * 100).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.step(d_pos, d_f, None, 1)
    ctx.sync_check()
    V, dV = orc.harmonic(xi_ref.astype(np.float32).astype(np.float64), ks, cen, np.zeros(4))
    f_ref = sysm.apply_forces(pos, dV, f0.astype(np.float64))
    assert_forces_close(d_f.cpu().numpy(), f_ref, f0, "shape forces")
    out = ctx.read_step_outputs()
    assert_close(out["V"].cpu().numpy(), V, "shape V")
    assert_close(out["dVdxi"].cpu().numpy(), dV, "shape dV/dxi")
    ctx.close()


def test_shape_cv_metad_and_abf_steps(torch, psg):
    """the shape CVs under the other two methods: a metadynamics step on (ShapeAnisotropy, Rg) -- the generic kernels, since
    the per-atom Jacobian needs r_i - c -- and the one-launch ABF step on (PrincipalMoment 0, Acylindricity) with bit-exact
    bins"""
    rng = np.random.default_rng(81)
    R, N = 300, 40
    pos = np.concatenate([_shape_molecules(rng, R, N), np.zeros((R, N, 1), np.float32)], axis=2)
    slot = np.concatenate([np.arange(0, 14), np.arange(10, 30)]).astype(np.int32)     # the two groups share atoms 10..13
    groups = [[("slots", 0, 14)], [("slots", 14, 20)]]
    f0 = (rng.standard_normal((R, N, 4)) * 100).astype(np.float32)
    # -- metadynamics
    o_cvs = [{"type": orc.SHAPE_ANISOTROPY, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": orc.RGYR, "groups": groups[1], "axis": 0, "period": 0.0}]
    g_cvs = [{"type": psg.CV_SHAPE_ANISOTROPY, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": psg.CV_RGYR, "groups": groups[1], "axis": 0, "period": 0.0}]
    sysm = orc.System(R, N, N, 4, o_cvs, slot, None, None)
    xi_ref, _ = sysm.cv_eval(pos)
    n_h = 500
    sigma = np.array([0.05, 0.03], np.float32)
    centers = (xi_ref[rng.integers(0, R, size=n_h)] + rng.normal(scale=0.04, size=(n_h, 2))).astype(np.float32)
    heights = rng.uniform(0.2, 1.2, size=n_h).astype(np.float32)
    V, dV, T = orc.metad(xi_ref.astype(np.float32).astype(np.float64), centers, heights, sigma, np.zeros(2))
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))     # the ORACLE's gradient through the oracle's Jacobian
    _, jac = sysm.cv_eval(pos)                                             # rows in slot order here (CV 0: 14 slots, CV 1: 20)
    slot_cv = np.array([0] * 14 + [1] * 20)
    extra = np.zeros((R, N, 3))
    for r in range(R):
        np.add.at(extra[r], slot, 2e-7 * T[r, slot_cv][:, None] * np.abs(jac[r]))
    for mode in (psg.HILLS_F32, psg.HILLS_F64):
        ctx = psg.Context(0)
        ctx.set_layout(R, N, N, 4, 4)
        ctx.set_cvs(g_cvs, slot, None, None)
        ctx.set_metad(sigma, 1.2, 0.0, n_h + 8, 0)
        ctx.set_hill_precision(mode)
        ctx.load_hills(dev(torch, centers), dev(torch, heights))
        d_f = dev(torch, f0)
        ctx.step(dev(torch, pos), d_f, None, 1)
        ctx.sync_check()
        out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
        assert_close(out["xi"], xi_ref, "metad shape xi")
        assert_close(out["V"], V, "metad shape V")
        if mode == psg.HILLS_F64:      # binary64 terms: the literal rule, and forces with the binary32 += rounding only
            assert_close(out["dVdxi"], dV, "metad shape dV/dxi (binary64 terms)")
            assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "metad shape forces (binary64 terms)")
        else:                          # binary32 terms: the conditioning bound of DESIGN.md "Hill sum precision"
            assert (np.abs(out["dVdxi"] - dV) <= np.maximum(np.maximum(1e-5 * np.abs(dV), 1e-6), 2e-7 * T)).all()
            assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "metad shape forces", extra)
        ctx.close()
    # -- ABF
    o_cvs = [{"type": orc.PRINCIPAL_MOMENT, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": orc.ACYLINDRICITY, "groups": groups[1], "axis": 0, "period": 0.0}]
    g_cvs = [{"type": psg.CV_PRINCIPAL_MOMENT, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": psg.CV_ACYLINDRICITY, "groups": groups[1], "axis": 0, "period": 0.0}]
    sysm = orc.System(R, N, N, 4, o_cvs, slot, None, None)
    xi_ref, _ = sysm.cv_eval(pos)
    lower, upper = xi_ref.min(axis=0).astype(np.float32) * 0.9, xi_ref.max(axis=0).astype(np.float32) * 1.1
    shape, periodic, n_thr = np.array([7, 5], np.int32), np.array([0, 0], np.int32), 3
    fs = rng.normal(scale=20.0, size=(R, 2)).astype(np.float32)
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.set_cvs(g_cvs, slot, None, None)
    ctx.set_abf(lower, upper, shape, periodic, n_thr)
    d_f = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.step(dev(torch, pos), d_f, dev(torch, fs), 1)
    assert ctx.launch_count() - n0 == 1
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    assert_close(out["xi"], xi_ref, "abf shape xi")
    hist, fsum = np.zeros(35, np.int32), np.zeros((35, 2), np.float64)
    b, dV = orc.abf_update(out["xi"], fs, lower, upper, shape, periodic, n_thr, hist, fsum)   # bins from the SAME binary32 xi
    assert np.array_equal(out["bin"], b)
    assert_close(out["dVdxi"], dV, "abf shape dV/dxi")
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "abf shape forces")
    ctx.close()


@pytest.mark.parametrize("boxed", [False, True])
def test_shape_cvs_over_range_groups_match_oracle(torch, psg, boxed):
    """gyration-tensor shape CVs over CONTIGUOUS RANGES (the polymer windows of config 3 are where PrincipalMoment /
    Asphericity are used): second moments by k_range_second, Jacobian w_i M (r_i - c) applied by the
    dense kernel; mass-weighted, overlapping ranges, next to an Rg CV, under a harmonic bias; with and without a box"""
    rng = np.random.default_rng(77)
    R, N = 3, 5003
    xyz = np.cumsum(0.15 * rng.standard_normal((R, N, 3)) * np.array([1.6, 1.0, 0.6]), axis=1) + 40.0
    pos = np.zeros((R, N, 4), np.float32)
    pos[..., :3] = xyz
    pos[..., 3] = 1.25
    aw = rng.uniform(1.0, 12.0, size=N).astype(np.float32)
    box = None
    if boxed:
        ext = float(np.ptp(xyz, axis=1).max())
        box = np.ceil(np.array([2.4, 2.7, 2.2]) * ext)
        pos[..., :3] = np.mod(xyz, box).astype(np.float32)
        assert (np.abs(pos[..., :3] - xyz) > 1).any()
    defs = [("asphericity", [("range", 0, N)], 0), ("principal_moment", [("range", 400, 3100)], 1), ("rgyr", [("range", 0, N)], 0),
            ("shape_anisotropy", [("range", 2500, N - 2500)], 0)]
    okind = {"asphericity": orc.ASPHERICITY, "principal_moment": orc.PRINCIPAL_MOMENT, "rgyr": orc.RGYR, "shape_anisotropy": orc.SHAPE_ANISOTROPY}
    gkind = {"asphericity": psg.CV_ASPHERICITY, "principal_moment": psg.CV_PRINCIPAL_MOMENT, "rgyr": psg.CV_RGYR,
             "shape_anisotropy": psg.CV_SHAPE_ANISOTROPY}
    sysm = orc.System(R, N, N, 4, [{"type": okind[k], "groups": g, "axis": ax, "period": 0.0} for k, g, ax in defs], None, atom_weight=aw, box=box)
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.set_cvs([{"type": gkind[k], "groups": g, "axis": ax, "period": 0.0} for k, g, ax in defs], None, None, aw)
    if boxed:
        ctx.set_box(box)
    xi_ref = sysm.cv_eval(pos, want_jac=False)
    ks = np.array([30.0, 20.0, 100.0, 500.0], np.float32)
    cen = (xi_ref * rng.uniform(0.8, 1.2, size=xi_ref.shape)).astype(np.float32)
    ctx.set_harmonic(ks, cen)
    f0 = (rng.standard_normal((R, N, 4)) * 30).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.step(dev(torch, pos), d_f, None, 1)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    assert_close(out["xi"], xi_ref, "shape CVs over ranges: xi")
    V, dV = orc.harmonic(xi_ref.astype(np.float32).astype(np.float64), ks, cen, np.zeros(4))
    assert_close(out["V"], V, "V")
    assert_close(out["dVdxi"], dV, "dV/dxi")
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "shape CVs over ranges: forces")
    assert np.array_equal(d_f.cpu().numpy()[..., 3].view(np.uint32), f0[..., 3].view(np.uint32))
    ctx.close()


def test_shape_cv_argument_errors(torch, psg):
    ctx = psg.Context(0)
    ctx.set_layout(2, 30, 30, 4, 4)
    ctx.set_cvs([{"type": psg.CV_ASPHERICITY, "groups": [("range", 0, 30)], "axis": 0, "period": 0.0}], np.zeros(0, np.int32))   # a range is fine
    with pytest.raises(psg.PsgError):      # ... but not beyond the array
        ctx.set_cvs([{"type": psg.CV_ASPHERICITY, "groups": [("range", 10, 30)], "axis": 0, "period": 0.0}], np.zeros(0, np.int32))
    with pytest.raises(psg.PsgError):      # which eigenvalue?
        ctx.set_cvs([{"type": psg.CV_PRINCIPAL_MOMENT, "groups": [("slots", 0, 5)], "axis": 3, "period": 0.0}], np.arange(5, dtype=np.int32))
    ctx.close()


# ------------------------------------------------------------------------------------ grid-stored metadynamics
@pytest.mark.parametrize("case", ["2d_periodic_open", "1d_open", "3d_mixed"])
def test_metad_grid_matches_oracle(torch, psg, case):
    """PAPER.md:L151, reading R-GRID: several well-tempered deposit events of R walkers (some masked out) onto a node grid, the
    node array compared with the oracle's after every event, then the interpolated bias and gradient at fresh points inside,
    on the faces and outside the grid; shapes are not multiples of the 128-node tile"""
    from paper_2301_04835_b200.psg import _view
    rng = np.random.default_rng({"2d_periodic_open": 1, "1d_open": 2, "3d_mixed": 3}[case])
    lower, upper, shape, periodic, sigma = {
        "2d_periodic_open": ((-math.pi, 0.2), (math.pi, 2.4), (67, 45), (1, 0), (0.35, 0.2)),
        "1d_open": ((-1.0,), (3.0,), (1001,), (0,), (0.15,)),
        "3d_mixed": ((0.0, -math.pi, 1.0), (2.0, math.pi, 4.0), (19, 24, 13), (0, 1, 0), (0.3, 0.5, 0.4)),
    }[case]
    n, R = len(shape), 300
    lo, up = np.array(lower), np.array(upper)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    ctx = psg.Context(0)
    ctx.set_layout(R, 8, 8, 4, 4)
    w0, kT = 1.2, 2.5
    ctx.metad_grid_set(lower, upper, shape, periodic, sigma, w0, kT)
    gp, nodes, hp = ctx.metad_grid_state()
    assert nodes == g.nodes
    for event in range(4):
        xi = (lo + (up - lo) * rng.uniform(-0.05, 1.05, size=(R, n))).astype(np.float32)   # some walkers just outside
        mask = None if event == 0 else (rng.uniform(size=R) < 0.7).astype(np.uint8)
        ctx.metad_grid_deposit(dev(torch, xi), None if mask is None else dev(torch, mask))
        ctx.sync_check()
        h_ref = g.deposit(xi, np.array(sigma), w0, kT, mask)
        h_gpu = _view(hp, (R,), torch.float64, 0).cpu().numpy()
        assert np.allclose(h_gpu, h_ref, rtol=1e-12, atol=0), f"heights, event {event}"
        if mask is not None:
            assert np.array_equal(h_gpu == 0.0, mask == 0)
        grid = _view(gp, (nodes, 1 + n), torch.float64, 0).cpu().numpy()
        scale = np.abs(g.values).max(axis=0)
        assert np.all(np.abs(grid - g.values) <= 1e-12 * scale), f"node array, event {event}"
    pts = (lo + (up - lo) * rng.uniform(-0.2, 1.2, size=(R, n))).astype(np.float32)
    pts[:n] = lo.astype(np.float32)                    # on the lower faces / the first node
    pts[n:2 * n] = up.astype(np.float32)               # on the upper faces (periodic: the first node again)
    d_V, d_dV = torch.empty(R, device="cuda"), torch.empty((R, n), device="cuda")
    ctx.metad_grid_eval(dev(torch, pts), d_V, d_dV)
    ctx.sync_check()
    V, dV = g.eval(pts.astype(np.float64))
    assert_close(d_V.cpu().numpy(), V, "grid V")
    assert_close(d_dV.cpu().numpy(), dV, "grid dV/dxi")
    assert np.abs(V).max() > 1.0                        # the test is not comparing zeros
    ctx.close()


def test_metad_grid_drives_the_force_scatter(torch, psg):
    """the grid bias in the per-step path: psg_cv_eval -> psg_metad_grid_eval -> psg_apply_bias_forces on dihedral CVs, forces
    against the oracle's scatter of the oracle's interpolated gradient"""
    w = small(1)
    ctx = make_ctx(psg, w, with_method=False)
    sysm = oracle_system(w)
    P = 2 * math.pi
    lower, upper, shape, periodic, sigma = (-math.pi, -math.pi), (math.pi, math.pi), (90, 90), (1, 1), (0.35, 0.35)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    ctx.metad_grid_set(lower, upper, shape, periodic, sigma, 1.2, 0.0)
    d_xi = torch.empty((w.R, 2), device="cuda")
    for frame in range(3):                               # three events at the walkers' own CV values
        ctx.cv_eval(dev(torch, w.positions(frame)), d_xi, None)
        ctx.metad_grid_deposit(d_xi)
        ctx.sync_check()
        g.deposit(d_xi.cpu().numpy(), np.array(sigma), 1.2)
    pos, f0 = w.positions(3 % w.K), w.forces0()
    d_pos, d_f = dev(torch, pos), dev(torch, f0)
    d_V, d_dV = torch.empty(w.R, device="cuda"), torch.empty((w.R, 2), device="cuda")
    ctx.cv_eval(d_pos, d_xi, None)
    ctx.metad_grid_eval(d_xi, d_V, d_dV)
    ctx.apply_bias_forces(d_pos, d_dV, d_f)
    ctx.sync_check()
    xi32 = d_xi.cpu().numpy()
    assert_close(xi32, sysm.cv_eval(pos, want_jac=False), "xi", period=w.period)
    V, dV = g.eval(xi32.astype(np.float64))              # both sides interpolate at the SAME binary32 xi (reading R-XI32)
    assert_close(d_V.cpu().numpy(), V, "grid V on the path")
    assert_close(d_dV.cpu().numpy(), dV, "grid dV/dxi on the path")
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "grid metad forces")
    # the same step as ONE launch: identical xi, V, dV/dxi; forces differ only by the rounding of the Jacobian cache
    d_f2 = dev(torch, f0)
    n0 = ctx.launch_count()
    ctx.metad_grid_step(d_pos, d_f2)
    assert ctx.launch_count() - n0 == 1
    ctx.sync_check()
    out = ctx.read_step_outputs()
    assert np.array_equal(out["xi"].cpu().numpy().view(np.uint32), xi32.view(np.uint32))
    assert np.array_equal(out["V"].cpu().numpy().view(np.uint32), d_V.cpu().numpy().view(np.uint32))
    assert np.array_equal(out["dVdxi"].cpu().numpy().view(np.uint32), d_dV.cpu().numpy().view(np.uint32))
    assert_forces_close(d_f2.cpu().numpy()[..., :3], f_ref, f0[..., :3], "grid metad forces, one launch")
    assert np.array_equal(d_f2.cpu().numpy()[..., 3].view(np.uint32), f0[..., 3].view(np.uint32))     # the pad is not touched
    ctx.close()


def test_metad_grid_as_the_method_of_psg_step(torch, psg):
    """PSG_METHOD_METAD_GRID (PAPER.md:L151 + the deposit interval of L147): psg_step deposits onto the grid every `stride`
    steps (well-tempered heights from the grid BEFORE the event) and interpolates; every step against the oracle's grid,
    the node array after the last event, psg_step_host, psg_bias_eval / psg_deposit_hill routed to the grid, and the
    refusal of a grid whose periodicity does not match the CVs"""
    from paper_2301_04835_b200.psg import _view
    w = small(1, stride=0)
    sysm = oracle_system(w)
    lower, upper, shape, periodic, sigma = (-math.pi, -math.pi), (math.pi, math.pi), (72, 60), (1, 1), (0.35, 0.35)
    w0, kT, stride = 1.2, w.params["kB_deltaT"], 3
    ctx = make_ctx(psg, w, with_method=False)
    with pytest.raises(psg.PsgError):          # dihedrals on an open grid
        ctx.set_metad_grid(lower, upper, shape, (0, 1), sigma, w0, kT, stride)
    with pytest.raises(psg.PsgError):          # a periodic grid that does not span the period
        ctx.set_metad_grid((-3.0, -math.pi), upper, shape, periodic, sigma, w0, kT, stride)
    ctx.set_metad_grid(lower, upper, shape, periodic, sigma, w0, kT, stride)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    f0 = w.forces0()
    d_f = dev(torch, f0)
    n_events = 0
    for step in range(1, 8):
        pos = w.positions(step % w.K)
        f_before = d_f.cpu().numpy()
        n0 = ctx.launch_count()
        ctx.step(dev(torch, pos), d_f, None, step)
        ctx.sync_check()
        xi_ref = sysm.cv_eval(pos, want_jac=False)
        out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
        assert_close(out["xi"], xi_ref, "xi", period=w.period)
        if step % stride == 0:
            h = g.deposit(out["xi"], np.array(sigma), w0, kT)      # at the SAME binary32 xi (reading R-XI32)
            n_events += 1
            assert ctx.launch_count() - n0 == 4                   # k_cv_eval, heights + node update, the one-launch step
            assert h.min() < w0 or n_events == 1
        else:
            assert ctx.launch_count() - n0 == 1
        V, dV = g.eval(out["xi"].astype(np.float64))
        assert_close(out["V"], V, f"grid V, step {step}")
        assert_close(out["dVdxi"], dV, f"grid dV/dxi, step {step}")
        f_ref = sysm.apply_forces(pos, dV, f_before[..., :3].astype(np.float64))
        assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f_before[..., :3], f"grid forces, step {step}")
    assert n_events == 2
    gp, nodes, _ = ctx.metad_grid_state()
    vals = _view(gp, (nodes, 3), torch.float64, 0).cpu().numpy()
    assert nodes == g.nodes and np.abs(vals - g.values).max() <= 1e-12 * max(1.0, np.abs(g.values).max())
    # the calls of the boundary follow the method
    xi = dev(torch, W.random_xi(w, 5))
    d_V, d_dV = torch.empty(w.R, device="cuda"), torch.empty((w.R, 2), device="cuda")
    ctx.bias_eval(xi, d_V, d_dV)
    ctx.sync_check()
    V, dV = g.eval(xi.cpu().numpy().astype(np.float64))
    assert_close(d_V.cpu().numpy(), V, "psg_bias_eval on the grid")
    ctx.deposit_hill(xi)
    ctx.sync_check()
    g.deposit(xi.cpu().numpy(), np.array(sigma), w0, kT)
    vals = _view(gp, (nodes, 3), torch.float64, 0).cpu().numpy()
    assert np.abs(vals - g.values).max() <= 1e-12 * max(1.0, np.abs(g.values).max())
    # host-array step (a non-deposit step)
    pos = w.positions(0)
    h_f = f0.copy()
    ctx.step_host(torch.from_numpy(pos), torch.from_numpy(h_f), None, 1)
    _, dV = g.eval(sysm.cv_eval(pos, want_jac=False).astype(np.float32).astype(np.float64))
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(h_f[..., :3], f_ref, f0[..., :3], "grid forces through psg_step_host")
    # a new layout drops the grid (it is sized by the old one)
    ctx.set_layout(w.R + 1, w.N, w.N, 4, 4)
    with pytest.raises(psg.PsgError):
        ctx.metad_grid_state()
    ctx.close()


def test_relayout_grows_the_host_staging_buffers(torch, psg):
    """psg_step_host after psg_set_layout to a LARGER system must not reuse staging buffers sized for the old one"""
    outs = []
    for R in (3, 40):
        w = W.make(1, R=R, n_hills=90, steps=2, stride=0)
        if not outs:
            ctx = make_ctx(psg, w)
        else:
            psg.configure_from_workload(ctx, w)          # the same ctx, re-laid out
        heights = oracle_heights(w)
        ctx.load_hills(dev(torch, w.params["hill_centers"]), dev(torch, heights))
        pos, f0 = w.positions(0), w.forces0()
        h_f = f0.copy()
        ctx.step_host(torch.from_numpy(pos), torch.from_numpy(h_f), None, 1)
        d_f = dev(torch, f0)
        ctx.step(dev(torch, pos), d_f, None, 1)
        ctx.sync_check()
        assert np.array_equal(h_f.view(np.uint32), d_f.cpu().numpy().view(np.uint32))
        outs.append(R)
    ctx.close()


def test_metad_grid_step_other_cv_kinds(torch, psg):
    """the one-launch grid step on CVs whose per-atom Jacobian needs r_i - c (Rg, shape anisotropy: the k_hills step cannot
    take these) and, through the three-launch route, on CVs over atom ranges (config 3's windows)"""
    rng = np.random.default_rng(91)
    R, N = 130, 40
    pos = np.concatenate([_shape_molecules(rng, R, N), np.zeros((R, N, 1), np.float32)], axis=2)
    slot = np.concatenate([np.arange(0, 14), np.arange(10, 30)]).astype(np.int32)
    groups = [[("slots", 0, 14)], [("slots", 14, 20)]]
    o_cvs = [{"type": orc.SHAPE_ANISOTROPY, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": orc.RGYR, "groups": groups[1], "axis": 0, "period": 0.0}]
    g_cvs = [{"type": psg.CV_SHAPE_ANISOTROPY, "groups": groups[0], "axis": 0, "period": 0.0},
             {"type": psg.CV_RGYR, "groups": groups[1], "axis": 0, "period": 0.0}]
    sysm = orc.System(R, N, N, 4, o_cvs, slot, None, None)
    xi_ref = sysm.cv_eval(pos, want_jac=False)
    lower, upper = xi_ref.min(axis=0) - 0.02, xi_ref.max(axis=0) + 0.02
    shape, periodic, sigma = (40, 33), (0, 0), (0.05, 0.03)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, 4, 4)
    ctx.set_cvs(g_cvs, slot, None, None)
    ctx.metad_grid_set(lower, upper, shape, periodic, sigma, 1.2, 0.0)
    seed_xi = (xi_ref[rng.integers(0, R, size=R)] + rng.normal(scale=0.03, size=(R, 2))).astype(np.float32)
    ctx.metad_grid_deposit(dev(torch, seed_xi))
    g.deposit(seed_xi, np.array(sigma), 1.2)
    f0 = (rng.standard_normal((R, N, 4)) * 100).astype(np.float32)
    d_f = dev(torch, f0)
    ctx.metad_grid_step(dev(torch, pos), d_f)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    assert_close(out["xi"], xi_ref, "xi")
    V, dV = g.eval(out["xi"].astype(np.float64))
    assert_close(out["V"], V, "V")
    assert_close(out["dVdxi"], dV, "dV/dxi")
    assert np.abs(dV).max() > 1.0
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "forces")
    ctx.close()
    # -- atom ranges
    w = small(3)
    ctx = make_ctx(psg, w, with_method=False)
    sysm = oracle_system(w)
    pos, f0 = w.positions(0), w.forces0()
    xi_ref = sysm.cv_eval(pos, want_jac=False)
    n = w.n_cv
    lower, upper = xi_ref.min(axis=0) - 0.5, xi_ref.max(axis=0) + 0.5
    g = orc.MetadGrid(lower, upper, (31,) * n, (0,) * n)
    ctx.metad_grid_set(lower, upper, (31,) * n, (0,) * n, (0.4,) * n, 50.0, 0.0)
    seed_xi = (xi_ref + rng.normal(scale=0.3, size=xi_ref.shape)).astype(np.float32)
    ctx.metad_grid_deposit(dev(torch, seed_xi))
    g.deposit(seed_xi, np.full(n, 0.4), 50.0)
    d_f = dev(torch, f0)
    ctx.metad_grid_step(dev(torch, pos), d_f)
    ctx.sync_check()
    out = {k: v.cpu().numpy() for k, v in ctx.read_step_outputs().items()}
    assert_close(out["xi"], xi_ref, "range xi")
    V, dV = g.eval(out["xi"].astype(np.float64))
    assert_close(out["dVdxi"], dV, "range dV/dxi")
    f_ref = sysm.apply_forces(pos, dV, f0[..., :3].astype(np.float64))
    assert_forces_close(d_f.cpu().numpy()[..., :3], f_ref, f0[..., :3], "range forces")
    ctx.close()


def test_metad_grid_argument_errors(torch, psg):
    ctx = psg.Context(0)
    with pytest.raises(psg.PsgError):
        ctx.metad_grid_set((0.0,), (1.0,), (8,), (0,), (0.1,), 1.0)          # no layout yet
    ctx.set_layout(4, 8, 8, 4, 4)
    with pytest.raises(psg.PsgError):
        ctx.metad_grid_eval(torch.zeros((4, 1), device="cuda"), torch.zeros(4, device="cuda"), None)   # no grid yet
    for bad in [dict(shape=(1,)), dict(upper=(-1.0,)), dict(sigma=(0.0,)), dict(w0=0.0)]:
        kw = dict(lower=(0.0,), upper=(1.0,), shape=(8,), periodic=(0,), sigma=(0.1,), w0=1.0)
        kw.update(bad)
        with pytest.raises(psg.PsgError):
            ctx.metad_grid_set(**kw)
    ctx.close()


# ------------------------------------------------------------------------------------ multiple walkers over several contexts
def test_split_deposit_equals_single_context_deposit(torch, psg):
    """psg_hill_heights + psg_append_hills: two contexts of R walkers each (two ranks' worth, run one after the other on this
    GPU -- no kernel waits on another) exchange (xi, height) and append; their hill lists equal, bit for bit, the list of one
    context holding all 2R walkers after psg_deposit_hill, over well-tempered events with masked-out walkers"""
    rng = np.random.default_rng(17)
    w = small(1)
    R, n = w.R, w.n_cv
    w2 = W.make(1, R=2 * R, n_hills=SMALL[1]["n_hills"], steps=SMALL[1]["steps"], stride=SMALL[1]["stride"])
    sigma, w0, kT, cap = w.params["sigma"], w.params["w0"], w.params["kB_deltaT"], 40 * R
    assert kT > 0
    ctxs = []
    for ww in (w, w, w2):
        c = make_ctx(psg, ww, with_method=False)
        c.set_metad(sigma, w0, kT, cap, 0)
        ctxs.append(c)
    a, b, whole = ctxs
    for event in range(4):
        xi = rng.uniform(-math.pi, math.pi, size=(2 * R, n)).astype(np.float32)
        mask = None if event == 0 else (rng.uniform(size=2 * R) < 0.6).astype(np.uint8)
        d_xi = dev(torch, xi)
        d_mask = None if mask is None else dev(torch, mask)
        hs = []
        for c, sl in ((a, slice(0, R)), (b, slice(R, 2 * R))):
            d_h = torch.empty(R, device="cuda")
            c.hill_heights(d_xi[sl].contiguous(), None if mask is None else d_mask[sl].contiguous(), d_h)
            hs.append(d_h)
        all_h = torch.cat(hs)                              # what the all-gather delivers to every rank
        for c in (a, b):
            c.append_hills(d_xi, all_h)
        whole.deposit_hill(d_xi, d_mask)
        lists = []
        for c in ctxs:
            c.sync_check()
            cen, hgt = c.get_hills()
            lists.append((cen.cpu().numpy(), hgt.cpu().numpy()))
        n_exp = 2 * R if mask is None else int(mask.sum())
        assert lists[2][1].shape[0] == (lists[2][1].shape[0] if event else n_exp)
        for cen, hgt in lists[:2]:
            assert cen.shape == lists[2][0].shape, f"event {event}: hill count"
            assert np.array_equal(cen.view(np.uint32), lists[2][0].view(np.uint32)), f"event {event}: centres"
            assert np.array_equal(hgt.view(np.uint32), lists[2][1].view(np.uint32)), f"event {event}: heights"
    assert lists[2][1].min() < 0.999 * w0                  # well-tempered heights really varied
    # (the lists are bit-identical here because every context's hill sum uses the same chunk length at <= 560 hills; in
    # general a rank's V_old equals the single context's up to binary32 rounding -- include/psg.h, psg_append_hills)
    # zero heights are skipped on the device, so the host cannot rule this overflow out: the kernel clamps at capacity and
    # the next synchronising call reports it
    n_before = a.n_hills()
    a.append_hills(torch.zeros((cap, n), device="cuda"), torch.ones(cap, device="cuda"))
    with pytest.raises(psg.PsgError) as ei:
        a.sync_check()
    assert ei.value.code == -4
    with pytest.raises(psg.PsgError):
        a.n_hills()
    assert n_before < cap
    for c in ctxs:
        c.close()


def test_masked_deposit_needs_no_capacity_padding_and_overflow_is_reported(torch, psg):
    """capacity is exact: masked rounds fill the store to the last slot without PSG_ECAPACITY; one hill too many is dropped
    by the kernel (never written beyond capacity) and reported by psg_sync_check; an unmasked overflow is refused on the host"""
    w = small(1, stride=0)
    R, cap = w.R, 2 * w.R + 5
    ctx = make_ctx(psg, w, with_method=False)
    ctx.set_metad(w.params["sigma"], 1.2, 0.0, cap, 0)
    xi = dev(torch, W.random_xi(w, 3))
    ctx.deposit_hill(xi)
    ctx.deposit_hill(xi)
    mask = np.zeros(R, np.uint8); mask[:5] = 1
    ctx.deposit_hill(xi, dev(torch, mask))            # exactly full now
    ctx.sync_check()
    assert ctx.n_hills() == cap
    V = torch.empty(R, device="cuda"); dV = torch.empty((R, 2), device="cuda")
    ctx.bias_eval(xi, V, dV); ctx.sync_check()
    V_full = V.cpu().numpy().copy()
    with pytest.raises(psg.PsgError) as ei:            # unmasked: the host knows the count exactly -> refused, nothing launched
        ctx.deposit_hill(xi)
    assert ei.value.code == -4
    one = np.zeros(R, np.uint8); one[7] = 1
    ctx.deposit_hill(xi, dev(torch, one))              # masked: launched, clamped on the device
    with pytest.raises(psg.PsgError) as ei:
        ctx.sync_check()
    assert ei.value.code == -4
    ctx.bias_eval(xi, V, dV)
    torch.cuda.synchronize()
    assert np.array_equal(V.cpu().numpy(), V_full), "a clamped deposit must not change the stored list"
    ctx.close()


def test_graph_captured_deposit_step_replays_and_later_launches_see_the_new_hills(torch, psg):
    """a deposit-phase psg_step captured in a CUDA graph appends R hills per REPLAY; launches issued outside the
    capture afterwards must sum over all of them (the ctx switches to the device counter until psg_get_hills)"""
    w = small(1, stride=5)
    R = w.R
    s = torch.cuda.Stream()
    ctx = psg.Context(0, s)
    psg.configure_from_workload(ctx, w, with_method=False)
    ctx.set_metad(w.params["sigma"], 1.2, w.params["kB_deltaT"], 10 * R, 5)
    ref = make_ctx(psg, w, with_method=False)
    ref.set_metad(w.params["sigma"], 1.2, w.params["kB_deltaT"], 10 * R, 5)
    d_pos = dev(torch, w.positions(0))
    d_f, d_fr = dev(torch, w.forces0()), dev(torch, w.forces0())
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        ctx.step(d_pos, d_f, None, 5)                 # a deposit step
    d_f.copy_(d_fr)
    torch.cuda.synchronize()
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    for _ in range(3):
        ref.step(d_pos, d_fr, None, 5)
    ref.sync_check()
    xi = dev(torch, W.random_xi(w, 9))
    out = []
    for c in (ctx, ref):
        V = torch.empty(R, device="cuda"); dV = torch.empty((R, 2), device="cuda")
        if c is ctx:
            with torch.cuda.stream(s):
                c.bias_eval(xi, V, dV)                # NOT captured: must still see the 3 R hills of the replays
        else:
            c.bias_eval(xi, V, dV)
        torch.cuda.synchronize()
        out.append((V.cpu().numpy(), dV.cpu().numpy()))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert ctx.n_hills() == ref.n_hills() == 3 * R
    assert np.allclose(d_f.cpu().numpy(), d_fr.cpu().numpy(), rtol=1e-5, atol=1e-4)
    ctx.close(); ref.close()
