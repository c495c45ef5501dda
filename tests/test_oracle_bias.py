"""Pins for the oracle's bias functions (harmonic, metadynamics hill sum, well-tempered
deposition, ABF grid update) and for force application.  No CUDA here.

Expected values are closed forms evaluated with python's math module on the spot
(exp(-1/2), 6 - 2 pi, ...), brute-force loops on tiny inputs written independently in
python, finite differences of the oracle's V against its gradient, and invariants.
PAPER.md:L125 (harmonic), L147-L151 (metadynamics / WTMD), L143 + L501-L507 (ABF),
L39 (forces added to the backend).
"""
import math

import numpy as np
import pytest

import oracle as orc

TWO_PI = 2.0 * math.pi
KB_DT = 0.008314462618 * 300.0 * 5.0  # kB * T * (gamma - 1), gamma = 6, T = 300 K (BASELINE.json config 0)


# ------------------------------------------------------------------ harmonic
def test_harmonic_closed_forms():
    V, dV = orc.harmonic([[1.25]], [1000.0], [[1.0]], [0.0])
    assert V[0] == pytest.approx(31.25, rel=1e-15) and dV[0, 0] == pytest.approx(250.0, rel=1e-15)
    # periodic: xi = 3, xi0 = -3 -> nearest image distance 6 - 2 pi
    V, dV = orc.harmonic([[3.0]], [100.0], [[-3.0]], [TWO_PI])
    d = 6.0 - TWO_PI
    assert dV[0, 0] == pytest.approx(100.0 * d, rel=1e-14) and V[0] == pytest.approx(50.0 * d * d, rel=1e-14)
    # same point, non-periodic CV: no wrapping
    V, dV = orc.harmonic([[3.0]], [100.0], [[-3.0]], [0.0])
    assert dV[0, 0] == 600.0 and V[0] == 1800.0


def test_harmonic_multi_cv_is_sum():
    V, dV = orc.harmonic([[1.0, 2.0], [0.0, 0.0]], [10.0, 4.0], [[0.5, 1.0], [0.0, 0.0]], [0.0, 0.0])
    assert V[0] == pytest.approx(0.5 * 10 * 0.25 + 0.5 * 4 * 1.0) and list(dV[0]) == [5.0, 4.0]
    assert V[1] == 0.0 and list(dV[1]) == [0.0, 0.0]


# ------------------------------------------------------------------ hill sum
def test_single_hill_closed_forms():
    V, dV, T = orc.metad([[1.0]], [[0.0]], [1.0], [1.0], [0.0])
    assert V[0] == pytest.approx(math.exp(-0.5), rel=1e-15)        # 0.6065306597126334
    assert dV[0, 0] == pytest.approx(-math.exp(-0.5), rel=1e-15)
    assert T[0, 0] == pytest.approx(math.exp(-0.5), rel=1e-15)
    # gradient vanishes at the centre, V = height there
    V, dV, _ = orc.metad([[0.25, -1.0]], [[0.25, -1.0]], [1.5], [0.35, 0.1], [0.0, 0.0])
    assert V[0] == 1.5 and np.all(dV == 0.0)


def test_periodic_hill_uses_nearest_image():
    sig, W = 0.35, np.float32(1.2)
    V, dV, _ = orc.metad([[3.0]], [[-3.0]], [W], [sig], [TWO_PI])
    d = 6.0 - TWO_PI                                    # -0.2831853...
    e = float(W) * math.exp(-0.5 * (d / sig) ** 2)
    assert V[0] == pytest.approx(e, rel=1e-14)
    assert dV[0, 0] == pytest.approx(-e * d / sig ** 2, rel=1e-14) and dV[0, 0] > 0
    # without periodicity the hill is 6 rad = 17 sigma away: nothing
    V2, _, _ = orc.metad([[3.0]], [[-3.0]], [W], [sig], [0.0])
    assert V2[0] < 1e-60


def test_two_hills_2d_brute_force_value():
    xi = (0.5, -1.0)
    s = [(0.0, float(np.float32(-1.2))), (3.0, 3.0)]   # the hill store is binary32
    W = [np.float32(1.2), np.float32(0.6)]
    sg = (0.35, 0.35)
    V_ref, g_ref = 0.0, [0.0, 0.0]
    for (s0, s1), w in zip(s, W):
        d0 = xi[0] - s0; d0 -= TWO_PI * round(d0 / TWO_PI)
        d1 = xi[1] - s1; d1 -= TWO_PI * round(d1 / TWO_PI)
        e = float(w) * math.exp(-0.5 * ((d0 / sg[0]) ** 2 + (d1 / sg[1]) ** 2))
        V_ref += e; g_ref[0] -= e * d0 / sg[0] ** 2; g_ref[1] -= e * d1 / sg[1] ** 2
    V, dV, _ = orc.metad([xi], s, W, sg, [TWO_PI, TWO_PI])
    assert V[0] == pytest.approx(V_ref, rel=1e-14)
    np.testing.assert_allclose(dV[0], g_ref, rtol=1e-13)
    assert V_ref == pytest.approx(0.36738243635115686, rel=1e-7)  # SURVEY.md 8(c) pin table (fp32 heights)


@pytest.mark.parametrize("n_cv,periodic", [(1, (True,)), (2, (True, True)), (3, (True, True, False))])
def test_hill_sum_brute_force_fd_and_periodicity(n_cv, periodic):
    rng = np.random.default_rng(40 + n_cv)
    n_h, R = 16, 5
    period = np.array([TWO_PI if p else 0.0 for p in periodic])
    lo = np.where(period > 0, -math.pi, 0.3); hi = np.where(period > 0, math.pi, 1.5)
    centers = rng.uniform(lo, hi, size=(n_h, n_cv)).astype(np.float32)
    heights = rng.uniform(0.1, 1.2, size=n_h).astype(np.float32)
    sigma = np.array([0.35, 0.35, 0.05][:n_cv])
    xi = rng.uniform(lo, hi, size=(R, n_cv))
    V, dV, T = orc.metad(xi, centers, heights, sigma, period)
    # brute-force double loop, python floats
    for r in range(R):
        v = 0.0; g = [0.0] * n_cv; t = [0.0] * n_cv
        for h in range(n_h):
            d = []
            for k in range(n_cv):
                dk = xi[r, k] - float(centers[h, k])
                if period[k] > 0:
                    dk -= period[k] * round(dk / period[k])
                d.append(dk)
            e = float(heights[h]) * math.exp(-0.5 * sum((d[k] / sigma[k]) ** 2 for k in range(n_cv)))
            v += e
            for k in range(n_cv):
                g[k] += -e * d[k] / sigma[k] ** 2; t[k] += abs(e * d[k] / sigma[k] ** 2)
        assert V[r] == pytest.approx(v, rel=1e-13)
        np.testing.assert_allclose(dV[r], g, rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(T[r], t, rtol=1e-12)
    # central FD of V against the returned gradient
    h = 1e-5
    for k in range(n_cv):
        e = np.zeros(n_cv); e[k] = h
        Vp, _, _ = orc.metad(xi + e, centers, heights, sigma, period)
        Vm, _, _ = orc.metad(xi - e, centers, heights, sigma, period)
        np.testing.assert_allclose((Vp - Vm) / (2 * h), dV[:, k], rtol=1e-6, atol=1e-8)
    # V(xi + P) = V(xi) along periodic CVs
    for k in range(n_cv):
        if period[k] > 0:
            sh = np.zeros(n_cv); sh[k] = period[k]
            Vs, dVs, _ = orc.metad(xi + sh, centers, heights, sigma, period)
            np.testing.assert_allclose(Vs, V, rtol=1e-12)
            np.testing.assert_allclose(dVs, dV, rtol=1e-9, atol=1e-12)


# -------------------------------------------------------- well-tempered heights
def test_well_tempered_heights_sequence():
    cap = 8
    centers = np.zeros((cap, 1), np.float32); heights = np.zeros(cap, np.float32)
    xi = np.array([[0.7]], np.float32)
    n = 0
    for _ in range(3):
        n = orc.deposit_hills(xi, None, 1.2, KB_DT, [0.35], [TWO_PI], n, centers, heights)
    assert n == 3 and np.all(centers[:3, 0] == np.float32(0.7))
    w1 = 1.2
    w2 = 1.2 * math.exp(-float(np.float32(w1)) / KB_DT)
    w3 = 1.2 * math.exp(-(float(np.float32(w1)) + float(np.float32(w2))) / KB_DT)
    assert heights[0] == np.float32(w1) and heights[1] == np.float32(w2) and heights[2] == np.float32(w3)
    assert KB_DT == pytest.approx(12.471693927, rel=1e-10)
    assert w2 == pytest.approx(1.0899193173897141, rel=1e-7) and w3 == pytest.approx(0.9987130595028008, rel=1e-7)


def test_standard_metadynamics_heights_constant():
    cap = 6
    centers = np.zeros((cap, 2), np.float32); heights = np.zeros(cap, np.float32)
    xi = np.array([[0.1, 0.2], [0.1, 0.2]], np.float32)
    n = orc.deposit_hills(xi, None, 1.2, 0.0, [0.35, 0.35], [TWO_PI, TWO_PI], 0, centers, heights)
    n = orc.deposit_hills(xi, None, 1.2, -1.0, [0.35, 0.35], [TWO_PI, TWO_PI], n, centers, heights)
    assert n == 4 and np.all(heights[:4] == np.float32(1.2))


def test_multi_walker_deposit_is_synchronous_and_masked():
    """reading R-MW: all walkers see the OLD list; masked walkers deposit nothing; append in replica order"""
    cap = 8
    centers = np.zeros((cap, 1), np.float32); heights = np.zeros(cap, np.float32)
    xi = np.array([[0.5], [0.5], [2.0]], np.float32)
    n = orc.deposit_hills(xi, None, 1.2, KB_DT, [0.35], [TWO_PI], 0, centers, heights)
    assert n == 3 and np.all(heights[:3] == np.float32(1.2))  # walker 1 did not see walker 0's hill
    n = orc.deposit_hills(xi, np.array([1, 0, 1], np.uint8), 1.2, KB_DT, [0.35], [TWO_PI], n, centers, heights)
    assert n == 5 and centers[3, 0] == np.float32(0.5) and centers[4, 0] == np.float32(2.0)
    V, _, _ = orc.metad(xi.astype(np.float64), centers[:3], heights[:3], [0.35], [TWO_PI])
    assert heights[3] == np.float32(1.2 * math.exp(-V[0] / KB_DT))
    assert heights[4] == np.float32(1.2 * math.exp(-V[2] / KB_DT))


# ----------------------------------------------------------------------- ABF
def _grid1(n_cv=1):
    lower = np.array([0.2] * n_cv, np.float32); upper = np.array([2.0] * n_cv, np.float32)
    shape = np.array([64] * n_cv, np.int32); periodic = np.zeros(n_cv, np.int32)
    return lower, upper, shape, periodic


def test_abf_bin_table():
    lower, upper, shape, periodic = _grid1()
    xi = np.array([[0.2], [1.0], [1.99], [2.0], [0.19999], [0.25], [np.nan], [-5.0], [1e30]], np.float32)
    hist = np.zeros(64, np.int32); fsum = np.zeros((64, 1))
    b, _ = orc.abf_update(xi, np.ones_like(xi), lower, upper, shape, periodic, 500, hist, fsum)
    assert list(b) == [0, 28, 63, -1, -1, 1, -1, -1, -1]
    assert hist.sum() == 4 and hist[0] == hist[28] == hist[63] == hist[1] == 1


def test_abf_bin_is_binary32_arithmetic():
    """the oracle's bin == numpy float32 scalar arithmetic (separately rounded sub and mul) on
    random inputs and on all 65 bin edges: guards against fp contraction / excess precision."""
    lower, upper, shape, periodic = _grid1()
    invd = np.float32(np.float64(64) / (np.float64(upper[0]) - np.float64(lower[0])))
    assert invd == np.float32(35.555557)
    rng = np.random.default_rng(0)
    edges = (np.float64(lower[0]) + np.arange(65) * (1.8 / 64)).astype(np.float32)
    xs = np.concatenate([rng.uniform(0.1, 2.1, 20000).astype(np.float32), edges,
                         np.nextafter(edges, np.float32(0)), np.nextafter(edges, np.float32(3))])
    hist = np.zeros(64, np.int32); fsum = np.zeros((64, 1))
    b, _ = orc.abf_update(xs[:, None], np.zeros((xs.size, 1), np.float32), lower, upper, shape, periodic, 500, hist, fsum)
    t = np.floor((xs - lower[0]) * invd)          # float32 array ops: each op rounded to binary32
    ref = np.where((t >= 0) & (t < 64), t, -1).astype(np.int32)
    assert np.array_equal(b, ref)
    assert hist.sum() == int((ref >= 0).sum())


def test_abf_two_phase_mean_force_and_threshold():
    lower, upper, shape, periodic = _grid1(2)
    hist = np.zeros(64 * 64, np.int32); fsum = np.zeros((64 * 64, 2))
    # replicas 0 and 1 fall in the same bin (28, 0) -> flat 28*64 + 0 (last CV fastest); replica 2 outside
    xi = np.array([[1.0, 0.21], [1.01, 0.22], [5.0, 1.0]], np.float32)
    f = np.array([[10.0, -4.0], [20.0, -8.0], [99.0, 99.0]], np.float32)
    b, dV = orc.abf_update(xi, f, lower, upper, shape, periodic, 4, hist, fsum)
    flat = 28 * 64 + 0
    assert list(b) == [flat, flat, -1] and hist[flat] == 2 and hist.sum() == 2
    np.testing.assert_allclose(fsum[flat], [30.0, -12.0])
    # both replicas read the FULLY updated bin; hist (2) < N (4) -> divide by N
    np.testing.assert_allclose(dV, [[7.5, -3.0], [7.5, -3.0], [0.0, 0.0]])
    # past the threshold the divisor is the count itself
    for _ in range(3):
        b, dV = orc.abf_update(xi, f, lower, upper, shape, periodic, 4, hist, fsum)
    assert hist[flat] == 8
    np.testing.assert_allclose(dV[0], [15.0, -6.0])


def test_abf_periodic_grid_wraps():
    lower = np.array([-math.pi], np.float32); upper = np.array([math.pi], np.float32)
    shape = np.array([32], np.int32); periodic = np.array([1], np.int32)
    hist = np.zeros(32, np.int32); fsum = np.zeros((32, 1))
    xi = np.array([[0.5], [0.5 + TWO_PI], [0.5 - TWO_PI], [-math.pi - 0.01], [math.pi + 0.01]], np.float32)
    b, _ = orc.abf_update(xi, np.ones_like(xi), lower, upper, shape, periodic, 500, hist, fsum)
    assert b[0] == b[1] == b[2] == 18 and b[3] == 31 and b[4] == 0 and hist.sum() == 5


# ------------------------------------------------------------ force application
def _adp_like(rng, R, N=22):
    pos = np.zeros((R, N, 4), np.float32)
    pos[..., :3] = np.cumsum(rng.normal(size=(R, N, 3)) * 0.1, axis=1) + 1.5
    pos[..., 3] = 1.0
    cvs = [{"type": orc.DIHEDRAL, "groups": [("slots", i, 1) for i in range(4)], "period": TWO_PI},
           {"type": orc.DIHEDRAL, "groups": [("slots", 4 + i, 1) for i in range(4)], "period": TWO_PI}]
    idx = np.array([4, 6, 8, 14, 6, 8, 14, 16], np.int32)
    return pos, cvs, idx


def test_forces_sum_over_shared_atoms_and_are_rigid_invariant():
    rng = np.random.default_rng(8)
    R, N = 3, 22
    pos, cvs, idx = _adp_like(rng, R)
    s = orc.System(R, N, N, 4, cvs, idx)
    xi, jac = s.cv_eval(pos)
    dV = rng.normal(size=(R, 2))
    F = s.apply_forces(pos, dV, np.zeros((R, N, 3)))
    for r in range(R):
        ref = np.zeros((N, 3))
        for slot, a in enumerate(idx):
            ref[a] += -dV[r, slot // 4] * jac[r, slot]      # atoms 6, 8, 14 get both CVs
        np.testing.assert_allclose(F[r], ref, rtol=1e-14, atol=1e-15)
        x = pos[r, :, :3].astype(np.float64)
        assert np.max(np.abs(F[r].sum(axis=0))) < 1e-9                   # sum F_i = 0
        assert np.max(np.abs(np.cross(x, F[r]).sum(axis=0))) < 1e-9      # sum r_i x F_i = 0
        untouched = np.setdiff1d(np.arange(N), idx)
        assert np.all(F[r, untouched] == 0.0)
    # += semantics
    F2 = s.apply_forces(pos, dV, np.ones((R, N, 3)))
    np.testing.assert_allclose(F2, F + 1.0, rtol=1e-14)


def test_force_is_minus_gradient_of_bias_end_to_end():
    """-F_i = dV_bias/dr_i through CV o metadynamics, by central differences of the bias energy."""
    rng = np.random.default_rng(12)
    pos, cvs, idx = _adp_like(rng, 1)
    pos[..., :3] = np.round(pos[..., :3] * 4096) / 4096
    s = orc.System(1, 22, 22, 4, cvs, idx)
    centers = rng.uniform(-math.pi, math.pi, size=(40, 2)).astype(np.float32)
    heights = rng.uniform(0.2, 1.2, size=40).astype(np.float32)
    sig, per = [0.35, 0.35], [TWO_PI, TWO_PI]

    def bias(p):
        return orc.metad(s.cv_eval(p, want_jac=False), centers, heights, sig, per)[0][0]

    xi = s.cv_eval(pos, want_jac=False)
    _, dV, _ = orc.metad(xi, centers, heights, sig, per)
    F = s.apply_forces(pos, dV, np.zeros((1, 22, 3)))[0]
    def cdiff(a, x, h):
        pp = pos.copy(); pm = pos.copy()
        pp[0, a, x] += np.float32(h); pm[0, a, x] -= np.float32(h)   # exact: pos is on a 2^-12 lattice
        return (bias(pp) - bias(pm)) / (2 * h)

    for a in (4, 6, 8, 14, 16, 0):
        for x in range(3):
            fd = (4 * cdiff(a, x, 2.0 ** -13) - cdiff(a, x, 2.0 ** -12)) / 3   # Richardson, O(h^4)
            assert -F[a, x] == pytest.approx(fd, rel=1e-6, abs=1e-6)


def test_forces_shared_array_collisions_accumulate():
    rng = np.random.default_rng(13)
    N, R = 40, 6
    pos = np.zeros((N, 4), np.float32); pos[:, :3] = rng.normal(size=(N, 3))
    cvs = [{"type": orc.DISTANCE, "groups": [("slots", 0, 1), ("slots", 1, 1)]}]
    idx = np.array([[0, 1], [0, 2], [1, 2], [0, 1], [5, 6], [6, 0]], np.int32)  # heavy collisions
    s = orc.System(R, N, 0, 4, cvs, idx)
    xi, jac = s.cv_eval(pos)
    dV = rng.normal(size=(R, 1))
    F = s.apply_forces(pos, dV, np.zeros((1, N, 3)))[0]
    ref = np.zeros((N, 3))
    for r in range(R):
        for slot in range(2):
            ref[idx[r, slot]] += -dV[r, 0] * jac[r, slot]
    np.testing.assert_allclose(F, ref, rtol=1e-13, atol=1e-15)


def test_forces_range_groups_rgyr_and_com_distance():
    """config-3 shaped CVs: Rg of everything + distance between the COMs of two halves"""
    rng = np.random.default_rng(14)
    R, N = 2, 64
    pos = np.zeros((R, N, 4), np.float32)
    pos[..., :3] = np.cumsum(rng.normal(size=(R, N, 3)) * 0.15, axis=1)
    cvs = [{"type": orc.RGYR, "groups": [("range", 0, N)]},
           {"type": orc.DISTANCE, "groups": [("range", 0, N // 2), ("range", N // 2, N // 2)]}]
    s = orc.System(R, N, N, 4, cvs, None)
    xi, jac = s.cv_eval(pos)
    assert jac.shape == (R, 2 * N, 3)
    dV = rng.normal(size=(R, 2))
    F = s.apply_forces(pos, dV, np.zeros((R, N, 3)))
    for r in range(R):
        x = pos[r, :, :3].astype(np.float64)
        # definitions, written with numpy
        c = x.mean(0); rg = math.sqrt(((x - c) ** 2).sum() / N)
        ca, cb = x[: N // 2].mean(0), x[N // 2:].mean(0)
        d = np.linalg.norm(cb - ca)
        assert xi[r, 0] == pytest.approx(rg, rel=1e-13) and xi[r, 1] == pytest.approx(d, rel=1e-13)
        ref = -dV[r, 0] * (x - c) / (N * rg)
        u = (cb - ca) / d
        ref[: N // 2] += -dV[r, 1] * (-u) / (N // 2)
        ref[N // 2:] += -dV[r, 1] * (u) / (N // 2)
        np.testing.assert_allclose(F[r], ref, rtol=1e-11, atol=1e-14)
        assert np.max(np.abs(F[r].sum(axis=0))) < 1e-9
        assert np.max(np.abs(np.cross(x, F[r]).sum(axis=0))) < 1e-9
