"""Pins for the oracle's ABF instantaneous-force estimator (reading R-ABF-EST).

The paper gives no formula ("based on the algorithm described in [43]"), so the estimator is a reading:
W = (J J^T)^-1 J p, dW/dt by the second-order backward difference, plus the bias applied at the previous step.
What pins the arithmetic is mathematics: constructed trajectories whose generalized force is known in closed form (the
difference formula is exact for momenta up to quadratic in time), the least-squares characterisation of W (numpy's lstsq on
the separately pinned Jacobian), and orthogonality.  Nothing here calls the CUDA path.
"""
import numpy as np
import pytest

import oracle as orc


def _one_particle_system():
    cv = {"type": orc.COMPONENT, "groups": [("slots", 0, 1)], "axis": 0, "period": 0.0}
    return orc.System(1, 3, 3, 4, [cv], np.array([1], np.int32))


def _arr(xyz):
    a = np.zeros((1, len(xyz), 4), np.float32)
    a[0, :, :3] = np.asarray(xyz, np.float32)
    return a


@pytest.mark.parametrize("law", ["constant_force", "linear_force"])
def test_free_particle_under_a_known_force(law):
    """CV = x of a free particle of mass m: J = e_x, W = p_x.  Under a constant force F the momentum is linear in time, under
    F(t) = 2 a t it is quadratic; the second-order backward difference is exact for both from the third call on."""
    s = _one_particle_system()
    m, dt, F, a = 2.0, 0.25, 3.0, 1.5                     # all exactly representable
    mass = np.array([1.0, m, 1.0], np.float32)
    pos = _arr([[0, 0, 0], [1, 2, 3], [5, 5, 5]])
    hist = np.zeros((1, 2, 1))
    for n in range(6):
        t = n * dt
        p = 0.5 + F * t if law == "constant_force" else a * t * t
        vel = _arr([[9, 9, 9], [p / m, 0.7, -0.3], [1, 1, 1]])    # the other atoms and the y, z momentum must not matter
        fs, W = s.abf_estimate(pos, vel, mass, dt, None, hist, first=(n == 0))
        assert W[0, 0] == pytest.approx(p, rel=1e-12)
        if n == 0:
            assert fs[0, 0] == 0.0                                # history initialised to W(t)
        if n >= 2:
            want = F if law == "constant_force" else 2 * a * t
            assert fs[0, 0] == pytest.approx(want, rel=1e-12, abs=1e-12)


def test_previous_bias_is_added_back():
    s = _one_particle_system()
    mass = np.array([1.0, 2.0, 1.0], np.float32)
    pos = _arr([[0, 0, 0], [1, 2, 3], [5, 5, 5]])
    hist = np.zeros((1, 2, 1))
    out = []
    for n in range(4):
        vel = _arr([[0, 0, 0], [0.25 * n, 0, 0], [0, 0, 0]])      # p_x = 0.5 n  ->  dW/dt = 0.5 / dt
        fs, _ = s.abf_estimate(pos, vel, mass, 0.5, np.array([[7.25]]), hist, first=(n == 0))
        out.append(fs[0, 0])
    assert out[3] == pytest.approx(1.0 + 7.25, rel=1e-12)


def test_W_is_the_least_squares_solution_of_JT_W_equals_p():
    """two distance CVs and a dihedral that share atoms: G = J J^T has off-diagonal terms; W must equal numpy's lstsq solution
    of J^T W = p built from the oracle's (separately pinned) Jacobian"""
    rng = np.random.default_rng(8)
    n = 7
    xyz = rng.normal(size=(n, 3)) * 0.8
    cvs = [{"type": orc.DISTANCE, "groups": [("slots", 0, 2), ("slots", 2, 1)], "axis": 0, "period": 0.0},
           {"type": orc.DISTANCE, "groups": [("slots", 3, 1), ("slots", 4, 1)], "axis": 0, "period": 0.0},
           {"type": orc.DIHEDRAL, "groups": [("slots", 5, 1), ("slots", 6, 1), ("slots", 7, 1), ("slots", 8, 1)], "axis": 0,
            "period": 2 * np.pi}]
    slots = np.array([0, 1, 2, 2, 3, 1, 2, 3, 4], np.int32)         # atoms 1, 2, 3 appear in several CVs
    wts = np.array([1.0, 3.0, 1, 1, 1, 1, 1, 1, 1], np.float32)
    s = orc.System(1, n, n, 4, cvs, slots, slot_weight=wts)
    pos = _arr(xyz)
    vel = _arr(rng.normal(size=(n, 3)))
    mass = rng.uniform(1.0, 16.0, size=n).astype(np.float32)
    hist = np.zeros((1, 2, 3))
    _, W = s.abf_estimate(pos, vel, mass, 0.1, None, hist, first=True)
    _, jac = s.cv_eval(pos)
    J = np.zeros((3, n, 3))
    row = 0
    for k, cv in enumerate(cvs):
        for g in cv["groups"]:
            for i in range(g[2]):
                J[k, slots[g[1] + i]] += jac[0, row]
                row += 1
    p = (mass[:, None].astype(np.float64) * vel[0, :, :3].astype(np.float64)).reshape(-1)
    Wref, *_ = np.linalg.lstsq(J.reshape(3, -1).T, p, rcond=None)
    assert np.allclose(W[0], Wref, rtol=1e-10, atol=1e-12)
    # momentum orthogonal to every row of J: nothing is projected out
    Jm = J.reshape(3, -1)
    q = p - Jm.T @ np.linalg.solve(Jm @ Jm.T, Jm @ p)
    vel_q = _arr((q.reshape(n, 3) / mass[:, None]))
    _, W0 = s.abf_estimate(pos, vel_q, mass, 0.1, None, np.zeros((1, 2, 3)), first=True)
    assert np.abs(W0).max() < 1e-5 * np.abs(W).max()            # float32 velocities


def test_second_order_convergence_on_a_cubic():
    """p(t) = t^3: the backward difference has error dt^2 p'''/3 = 2 dt^2; halving dt divides it by 4"""
    s = _one_particle_system()
    mass = np.array([1.0, 1.0, 1.0], np.float32)
    pos = _arr([[0, 0, 0], [1, 2, 3], [5, 5, 5]])
    errs = []
    for dt in (0.125, 0.0625):
        hist = np.zeros((1, 2, 1))
        for n in range(5):
            t = 1.0 + n * dt
            fs, _ = s.abf_estimate(pos, _arr([[0, 0, 0], [t ** 3, 0, 0], [0, 0, 0]]), mass, dt, None, hist, first=(n == 0))
        errs.append(abs(fs[0, 0] - 3 * t * t))
    assert errs[0] == pytest.approx(2 * 0.125 ** 2, rel=0.02)
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05)
