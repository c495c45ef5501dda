"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the oracle and therefore holds NONE of
the method's arithmetic: no CV formula, no bias, no binning.  It only draws random
geometry / hill centres / force samples and describes the CVs in a neutral form
(strings and index lists) that each side translates into its own structs.
Quantities the method itself computes (well-tempered hill heights) are NOT produced
here: a workload lists the hill *centres* and the deposit rounds, and the caller
fills the heights with whichever implementation it is exercising.

The only geometry used is input conditioning (documented in DESIGN.md, "Input
recipe"): rejecting nearly collinear bond triples and placing a group at a drawn
distance from another.

The paper's own workloads (alanine dipeptide in OpenMM, PAPER.md:L81, L483-L487;
the 51,200-particle diblock melt, L320-L344; the 40,981-atom polymer, L408) need
engines, force fields and input files that are not available; these inputs take
their shapes and parameters (Table B.1) and stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED = 23010483
TWO_PI = 2.0 * math.pi
KB = 0.008314462618            # kJ/(mol K)
KB_DELTA_T = KB * 300.0 * 5.0  # kB * T * (gamma - 1), T = 300 K, gamma = 6 (BASELINE.json config 0)

# purposes (third word of the seed sequence)
_P_POS, _P_JIT, _P_FRC, _P_HILL, _P_IDX, _P_PLACE, _P_FS, _P_W, _P_XI = range(9)


def _rng(config: int, purpose: int, *extra: int) -> np.random.Generator:
    return np.random.default_rng([SEED, config, purpose, *extra])


def _unit_vectors(rng, shape):
    v = rng.normal(size=tuple(shape) + (3,))
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _min_sin_bond_angles(xyz, quad):
    """smallest sine of the angle between successive 'bonds' of a 4-atom tuple (input guard only)"""
    p = xyz[..., quad, :]
    b = p[..., 1:, :] - p[..., :-1, :]
    s = []
    for i in range(2):
        c = np.cross(b[..., i, :], b[..., i + 1, :])
        s.append(np.linalg.norm(c, axis=-1) /
                 (np.linalg.norm(b[..., i, :], axis=-1) * np.linalg.norm(b[..., i + 1, :], axis=-1)))
    return np.minimum(s[0], s[1])


@dataclass
class Workload:
    config: int
    name: str
    R: int                      # replicas / walkers / windows
    N: int                      # atoms per position array
    shared_array: bool          # True: all replicas index ONE array (replica stride 0)
    cvs: list                   # neutral CV descriptions, see _cv()
    slot_atom: np.ndarray | None   # int32 [n_slots] or [R][n_slots]
    method: str                 # "metad" | "abf" | "harmonic"
    params: dict
    steps: int
    K: int                      # number of position frames; step s uses frame s % K
    atom_weight: np.ndarray | None = None
    _base: np.ndarray | None = field(default=None, repr=False)
    _extra: dict = field(default_factory=dict, repr=False)

    @property
    def n_cv(self):
        return len(self.cvs)

    @property
    def n_arrays(self):
        return 1 if self.shared_array else self.R

    @property
    def period(self):
        return np.array([cv["period"] for cv in self.cvs], dtype=np.float64)

    # ---- engine arrays -------------------------------------------------------
    def positions(self, frame: int) -> np.ndarray:
        """float32 [n_arrays][N][4]; w holds an arbitrary per-atom value the path must ignore."""
        k = frame % self.K
        if self.config == 2:
            return _cfg2_frame(self, k)
        pos = self._base.copy()
        if k > 0:
            jit = _rng(self.config, _P_JIT, k).normal(scale=0.005, size=pos[..., :3].shape)
            pos[..., :3] = (pos[..., :3].astype(np.float64) + jit).astype(np.float32)
        return pos

    def forces0(self) -> np.ndarray:
        """engine forces before biasing: N(0, 100) kJ/mol/nm, float32 [n_arrays][N][4]"""
        rng = _rng(self.config, _P_FRC)
        f = rng.standard_normal(size=(self.n_arrays, self.N, 4), dtype=np.float32) * np.float32(100.0)
        return f

    def fsample(self, frame: int) -> np.ndarray:
        """ABF instantaneous generalized-force samples, float32 [R][n_cv] (an INPUT of the path)"""
        assert self.method == "abf"
        rng = _rng(self.config, _P_FS, frame % self.K)
        mu = np.array(self.params["fsample_mean"])[: self.n_cv]
        return (mu + rng.normal(scale=self.params["fsample_std"], size=(self.R, self.n_cv))).astype(np.float32)

    def hill_rounds(self):
        """[(begin, end)] slices of params['hill_centers'] that are deposited together"""
        n, rs = self.params["n_hills"], self.params["round"]
        return [(b, min(b + rs, n)) for b in range(0, n, rs)]


def _cv(kind, groups, period=0.0, axis=0):
    """neutral CV: kind in {"distance","angle","dihedral","component","rgyr"}; groups are
    ("slots", begin, size) slices of the slot list or ("range", first_atom, n_atoms)."""
    return {"kind": kind, "groups": list(groups), "period": float(period), "axis": int(axis)}


def _with_w(xyz, rng):
    out = np.empty(xyz.shape[:-1] + (4,), np.float32)
    out[..., :3] = xyz
    out[..., 3] = rng.uniform(-1, 1, size=xyz.shape[:-1])   # e.g. a charge: never read, never written
    return out


# ----------------------------------------------------------------- configs 0 / 1
ADP_PHI, ADP_PSI = [4, 6, 8, 14], [6, 8, 14, 16]      # PAPER.md:L81 (Fig. 2), 0-based


def _adp_chains(config, R, N=22):
    rng = _rng(config, _P_POS)
    out = np.empty((R, N, 3))
    todo = np.arange(R)
    while todo.size:
        u = _unit_vectors(rng, (todo.size, N - 1))
        xyz = np.concatenate([np.zeros((todo.size, 1, 3)), np.cumsum(0.15 * u, axis=1)], axis=1) + 1.5
        ok = (_min_sin_bond_angles(xyz, ADP_PHI) >= 0.1) & (_min_sin_bond_angles(xyz, ADP_PSI) >= 0.1)
        out[todo[ok]] = xyz[ok]
        todo = todo[~ok]
    return out


def _hill_centers(config, n_hills, n_cv):
    rng = _rng(config, _P_HILL)
    c = np.empty((n_hills, n_cv), np.float32)
    c[:, :2] = rng.uniform(-math.pi, math.pi, size=(n_hills, 2)).astype(np.float32)
    c[:, :2] = np.where(c[:, :2] >= np.float32(math.pi), np.float32(-math.pi), c[:, :2])  # keep [-pi, pi)
    if n_cv == 3:
        c[:, 2] = rng.uniform(0.3, 1.5, size=n_hills).astype(np.float32)
    return c


def _metad_params(config, n_cv, n_hills, rnd, capacity, stride):
    sigma = [0.35, 0.35, 0.05][:n_cv]          # PAPER.md:L511 sigma = 0.35 rad; BASELINE.json config 4
    return {"sigma": np.array(sigma, np.float32), "w0": 1.2, "kB_deltaT": KB_DELTA_T,   # PAPER.md:L512 h = 1.2 kJ/mol
            "n_hills": n_hills, "round": rnd, "capacity": capacity, "stride": stride,
            "hill_centers": _hill_centers(config, n_hills, n_cv)}


def _adp(config, R, n_hills, rnd, steps, stride, K):
    rng = _rng(config, _P_W)
    base = _with_w(_adp_chains(config, R).astype(np.float32), rng)
    cvs = [_cv("dihedral", [("slots", i, 1) for i in range(4)], TWO_PI),
           _cv("dihedral", [("slots", 4 + i, 1) for i in range(4)], TWO_PI)]
    n_dep = 0 if stride <= 0 else (steps // stride) * R
    return Workload(config, f"config{config}", R, 22, False, cvs, np.array(ADP_PHI + ADP_PSI, np.int32), "metad",
                    _metad_params(config, 2, n_hills, rnd, n_hills + n_dep, stride), steps, K, _base=base)


def config0(n_hills=1000, steps=1000):
    """22 atoms, phi/psi, WTMD with 1,000 hills, 1 replica, no deposits in the timed loop."""
    return _adp(0, 1, n_hills, 1, steps, 0, 16)


def config1(R=512, n_hills=50000, steps=10000, stride=500):
    """multiple-walker WTMD: R replicas, shared hill list deposited in rounds of R, +R hills every `stride` steps
    (PAPER.md:L513 stride = 500)."""
    return _adp(1, R, n_hills, R, steps, stride, 8)


# ---------------------------------------------------------------------- config 2
def config2(R=4096, N=50000, steps=1000, variant="hit"):
    """ABF on R replicas of an N-atom system; 2 distance CVs between barycenters of 4 atom pairs;
    ONE 64x64 grid over [0.2, 2.0)^2 shared by all replicas; N_threshold = 500."""
    idx = _rng(2, _P_IDX).permutation(N)[:8].astype(np.int32)
    cvs = [_cv("distance", [("slots", 0, 2), ("slots", 2, 2)]), _cv("distance", [("slots", 4, 2), ("slots", 6, 2)])]
    params = {"lower": np.array([0.2, 0.2], np.float32), "upper": np.array([2.0, 2.0], np.float32),
              "shape": np.array([64, 64], np.int32), "periodic": np.array([0, 0], np.int32), "n_threshold": 500,
              "fsample_mean": (25.0, -15.0), "fsample_std": 5.0, "variant": variant}
    return Workload(2, "config2-" + variant, R, N, False, cvs, idx, "abf", params, steps, 2)


def _cfg2_frame(w: Workload, k: int) -> np.ndarray:
    """uniform positions in a 10 nm box, one rng stream per replica (so any subset can be regenerated);
    'hit' variant: per frame, the second group of each CV is rigidly translated so that the barycenter
    distance is a drawn d in [0.1, 2.1) nm kept 1e-3 bin widths away from every bin edge."""
    key = ("frame", k)
    if key in w._extra:
        return w._extra[key]
    pos = np.empty((w.R, w.N, 4), np.float32)
    for r in range(w.R):
        pos[r] = _rng(2, _P_POS, r).random(size=(w.N, 4), dtype=np.float32) * np.float32(10.0)
    pos[..., 3] = pos[..., 3] * np.float32(0.2) - np.float32(1.0)
    if w.params["variant"] == "hit":
        rng = _rng(2, _P_PLACE, k)
        lo, width = 0.2, 1.8 / 64
        for c in range(2):
            a = w.slot_atom[4 * c: 4 * c + 2]
            b = w.slot_atom[4 * c + 2: 4 * c + 4]
            d = rng.uniform(0.1, 2.1, size=w.R)
            while True:
                t = (d - lo) / width
                bad = np.abs(t - np.round(t)) < 1e-3
                if not bad.any():
                    break
                d[bad] = rng.uniform(0.1, 2.1, size=int(bad.sum()))
            u = _unit_vectors(rng, (w.R,))
            ca = pos[:, a, :3].astype(np.float64).mean(axis=1)
            cb = pos[:, b, :3].astype(np.float64).mean(axis=1)
            shift = ca + d[:, None] * u - cb
            pos[:, b, :3] = (pos[:, b, :3].astype(np.float64) + shift[:, None, :]).astype(np.float32)
    w._extra[key] = pos
    return pos


# ---------------------------------------------------------------------- config 3
def config3(R=256, N=100000, steps=200, weighted=False):
    """umbrella windows on polymer-like random walks (0.15 nm steps): Rg of all atoms and the distance
    between the centers of mass of the two halves; harmonic k = 1000 kJ/mol/nm^2, centres evenly in [1, 5] nm."""
    rng = _rng(3, _P_POS)
    xyz = np.empty((R, N, 3), np.float32)
    for r in range(R):
        xyz[r] = np.concatenate([np.zeros((1, 3)), np.cumsum(0.15 * _unit_vectors(rng, (N - 1,)), axis=0)]).astype(np.float32)
    base = _with_w(xyz, _rng(3, _P_W))
    h = N // 2
    cvs = [_cv("rgyr", [("range", 0, N)]), _cv("distance", [("range", 0, h), ("range", h, N - h)])]
    c = 1.0 + 4.0 * np.arange(R) / max(R - 1, 1)
    params = {"kspring": np.array([1000.0, 1000.0], np.float32),
              "centers": np.stack([c, c], axis=1).astype(np.float32)}
    aw = _rng(3, _P_W, 1).uniform(1.0, 16.0, size=N).astype(np.float32) if weighted else None
    return Workload(3, "config3" + ("-weighted" if weighted else ""), R, N, False, cvs, None, "harmonic", params,
                    steps, 2, atom_weight=aw, _base=base)


# ---------------------------------------------------------------------- config 4
def config4(N=1000000, R=1024, n_hills=200000, steps=1000):
    """one shared N-atom array, R walkers with their own index lists: 2 dihedrals + 1 distance;
    WTMD with n_hills hills, sigma = (0.35, 0.35, 0.05), no deposits in the timed loop."""
    box = 21.5 * (N / 1.0e6) ** (1.0 / 3.0)                      # ~100 atoms / nm^3
    rng = _rng(4, _P_POS)
    xyz = rng.random(size=(N, 3), dtype=np.float32) * np.float32(box)
    irng = _rng(4, _P_IDX)
    idx = np.empty((R, 10), np.int32)
    todo = np.arange(R)
    while todo.size:
        cand = np.stack([irng.choice(N, size=10, replace=False) for _ in range(todo.size)]).astype(np.int32)
        x = xyz[cand].astype(np.float64)
        ok = (_min_sin_bond_angles(x, [0, 1, 2, 3]) >= 0.1) & (_min_sin_bond_angles(x, [4, 5, 6, 7]) >= 0.1)
        idx[todo[ok]] = cand[ok]
        todo = todo[~ok]
    # the distance pair's second atom sits 0.3..1.5 nm from the first, so that the 3rd hill coordinate matters.
    # moved atoms never belong to a dihedral (checked), so the guard above stays valid.
    prng = _rng(4, _P_PLACE)
    dih_atoms = set(idx[:, :8].reshape(-1).tolist())
    firsts = set(idx[:, 8].tolist())
    moved = set()
    for r in range(R):
        while int(idx[r, 9]) in dih_atoms or int(idx[r, 9]) in firsts or int(idx[r, 9]) in moved:
            idx[r, 9] = prng.integers(N)
        moved.add(int(idx[r, 9]))
        d = prng.uniform(0.3, 1.5)
        u = _unit_vectors(prng, ())
        xyz[idx[r, 9]] = (xyz[idx[r, 8]].astype(np.float64) + d * u).astype(np.float32)
    base = _with_w(xyz[None], _rng(4, _P_W))
    cvs = [_cv("dihedral", [("slots", i, 1) for i in range(4)], TWO_PI),
           _cv("dihedral", [("slots", 4 + i, 1) for i in range(4)], TWO_PI),
           _cv("distance", [("slots", 8, 1), ("slots", 9, 1)])]
    return Workload(4, "config4", R, N, True, cvs, idx, "metad", _metad_params(4, 3, n_hills, R, n_hills, 0),
                    steps, 4, _base=base)


def make(config: int, **kw) -> Workload:
    return {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}[config](**kw)


def random_xi(w: Workload, tag: int = 0) -> np.ndarray:
    """float32 [R][n_cv] CV values for exercising the bias calls on their own: periodic CVs uniform in
    [-pi, pi), others in [0.3, 1.5)."""
    rng = _rng(w.config, _P_XI, tag)
    per = w.period > 0
    lo = np.where(per, -math.pi, 0.3)
    hi = np.where(per, math.pi, 1.5)
    return rng.uniform(lo, hi, size=(w.R, w.n_cv)).astype(np.float32)
