"""The seeded input generators: deterministic, shaped as BASELINE.json's configs, and carrying
the parameter values the paper prints (tests/golden/paper_parameters.txt)."""
import math
import os

import numpy as np

import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_parameters.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = v.split()
    return out


def test_paper_parameters_are_used():
    g = _gold()
    assert W.ADP_PHI == [int(x) for x in g["adp_phi_atoms"]] and W.ADP_PSI == [int(x) for x in g["adp_psi_atoms"]]
    w = W.make(1, R=8, n_hills=64)
    assert list(w.slot_atom) == W.ADP_PHI + W.ADP_PSI
    assert np.all(w.params["sigma"] == np.float32(float(g["metad_sigma_rad"][0])))
    assert w.params["w0"] == float(g["metad_height_kjmol"][0])
    assert w.params["stride"] == int(g["metad_stride"][0])
    assert W.make(2, R=4, N=100).params["n_threshold"] == int(g["abf_n_threshold"][0])
    assert abs(W.KB_DELTA_T - 12.471693927) < 1e-8


def test_deterministic_and_shapes():
    a, b = W.make(1, R=16, n_hills=100), W.make(1, R=16, n_hills=100)
    assert np.array_equal(a.positions(3), b.positions(3)) and np.array_equal(a.forces0(), b.forces0())
    assert np.array_equal(a.params["hill_centers"], b.params["hill_centers"])
    assert a.positions(0).shape == (16, 22, 4) and a.positions(0).dtype == np.float32
    assert not np.array_equal(a.positions(0), a.positions(1))
    assert np.array_equal(a.positions(0), a.positions(a.K))
    c = a.params["hill_centers"]
    assert c.min() >= -math.pi and c.max() < math.pi
    # full-size bookkeeping of config 1: 50,000 hills + 20 deposit events x 512 walkers = 60,240
    full = W.make(1)
    assert full.params["capacity"] == 60240 and full.R == 512 and full.steps == 10000
    assert len(full.hill_rounds()) == 98 and full.hill_rounds()[-1] == (49664, 50000)


def test_chain_geometry():
    w = W.make(1, R=64, n_hills=10)
    x = w.positions(0)[..., :3].astype(np.float64)
    bonds = np.linalg.norm(x[:, 1:] - x[:, :-1], axis=-1)
    assert np.allclose(bonds, 0.15, atol=1e-6)
    assert np.allclose(x[:, 0], 1.5)


def test_config2_hit_placement_and_edge_guard():
    w = W.make(2, R=200, N=500)
    for k in range(2):
        p = w.positions(k)[..., :3].astype(np.float64)
        for c in range(2):
            a, b = w.slot_atom[4 * c: 4 * c + 2], w.slot_atom[4 * c + 2: 4 * c + 4]
            d = np.linalg.norm(p[:, b].mean(1) - p[:, a].mean(1), axis=1)
            assert d.min() > 0.099 and d.max() < 2.101
            t = (d - 0.2) / (1.8 / 64)
            assert np.all(np.abs(t - np.round(t)) > 5e-4)
    assert w.fsample(0).shape == (200, 2) and w.fsample(0).dtype == np.float32
    lit = W.make(2, R=8, N=500, variant="lit")
    assert lit.positions(0)[..., :3].max() < 10.0


def test_config3_and_4():
    w = W.make(3, R=3, N=1000)
    x = w.positions(0)[..., :3].astype(np.float64)
    assert np.allclose(np.linalg.norm(x[:, 1:] - x[:, :-1], axis=-1), 0.15, atol=2e-5)
    assert w.params["centers"][0, 0] == 1.0 and w.params["centers"][-1, 0] == 5.0
    w4 = W.make(4, N=5000, R=32, n_hills=64)
    assert w4.slot_atom.shape == (32, 10) and w4.shared_array and w4.positions(0).shape == (1, 5000, 4)
    for r in range(32):
        assert len(set(w4.slot_atom[r].tolist())) == 10
    p = w4.positions(0)[0, :, :3].astype(np.float64)
    d = np.linalg.norm(p[w4.slot_atom[:, 9]] - p[w4.slot_atom[:, 8]], axis=1)
    assert d.min() >= 0.3 - 1e-5 and d.max() <= 1.5 + 1e-5
    assert w4.params["hill_centers"].shape == (64, 3)
