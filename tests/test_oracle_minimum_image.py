"""Pins for the oracle's minimum-image convention (reading R-MI).

The paper is silent on periodic positions, so the convention is a reading: orthorhombic box lengths (0 = open), every
displacement between group centres is its nearest image, and the atoms of a group are taken as the images nearest to the
group's first atom.  What pins it is mathematics, not the oracle: constructed geometries across a boundary, invariance
under shifting any atom by box vectors, equality with the open-boundary result when nothing crosses a boundary, and
central finite differences.  Nothing here calls the CUDA path.
"""
import math

import numpy as np
import pytest

import oracle as orc

BOX = (3.0, 4.0, 5.0)


def _sys(cv_type, n_atoms, groups_atoms, box, weights=None):
    slots, groups, o = [], [], 0
    for g in groups_atoms:
        groups.append(("slots", o, len(g)))
        slots += list(g)
        o += len(g)
    cv = {"type": cv_type, "groups": groups, "axis": 0, "period": 2 * math.pi if cv_type == orc.DIHEDRAL else 0.0}
    return orc.System(1, n_atoms, n_atoms, 4, [cv], np.array(slots, np.int32), slot_weight=weights, box=box)


def _pos4(xyz):
    p = np.zeros((len(xyz), 4), np.float32)
    p[:, :3] = np.asarray(xyz, np.float32)
    p[:, 3] = -2.5
    return p


def test_distance_across_the_boundary():
    # x = 0.1 and x = 2.9 in a box of 3: the nearest image is 0.2 away, pointing in -x from atom 0 to atom 1
    s = _sys(orc.DISTANCE, 2, [[0], [1]], BOX)
    xi, jac = s.cv_eval(_pos4([[0.1, 1.0, 1.0], [2.9, 1.0, 1.0]])[None])
    assert xi[0, 0] == pytest.approx(0.2, abs=1e-6)
    assert np.allclose(jac[0, 1], [-1.0, 0.0, 0.0], atol=1e-6) and np.allclose(jac[0, 0], [1.0, 0.0, 0.0], atol=1e-6)
    # the same pair in an open box: 2.8
    s0 = _sys(orc.DISTANCE, 2, [[0], [1]], None)
    assert s0.cv_eval(_pos4([[0.1, 1.0, 1.0], [2.9, 1.0, 1.0]])[None], want_jac=False)[0, 0] == pytest.approx(2.8, abs=1e-6)
    # open in x only, periodic in y: the x separation is kept, the y separation wraps
    sy = _sys(orc.DISTANCE, 2, [[0], [1]], (0.0, 4.0, 0.0))
    xi = sy.cv_eval(_pos4([[0.1, 0.2, 1.0], [2.9, 3.9, 1.0]])[None], want_jac=False)
    assert xi[0, 0] == pytest.approx(math.hypot(2.8, 0.3), abs=1e-6)


def test_group_split_by_wrapping_is_made_whole():
    # a 3-atom group whose last atom was wrapped to the other side: barycenter at x = 0.0 (images 2.9-3, 0.0, 0.1), not 1.0
    s = _sys(orc.DISTANCE, 4, [[0, 1, 2], [3]], BOX)
    pos = _pos4([[0.0, 1, 1], [0.1, 1, 1], [2.9, 1, 1], [1.0, 1, 1]])
    assert s.cv_eval(pos[None], want_jac=False)[0, 0] == pytest.approx(1.0, abs=1e-6)
    # radius of gyration of the same three atoms: spread 0.1 around 0.0 -> sqrt((0.01 + 0.01 + 0) / 3)
    r = orc.System(1, 4, 4, 4, [{"type": orc.RGYR, "groups": [("slots", 0, 3)], "axis": 0, "period": 0.0}],
                   np.array([0, 1, 2], np.int32), box=BOX)
    assert r.cv_eval(pos[None], want_jac=False)[0, 0] == pytest.approx(math.sqrt(0.02 / 3.0), abs=1e-6)


@pytest.mark.parametrize("cv_type,groups", [(orc.DISTANCE, [[0, 1], [2]]), (orc.ANGLE, [[0], [1, 2], [3]]),
                                            (orc.DIHEDRAL, [[0], [1], [2], [3, 4]])])
def test_shifting_atoms_by_box_vectors_changes_nothing(cv_type, groups):
    rng = np.random.default_rng(11)
    n = 5
    # a compact molecule (extent << box / 2) somewhere in the box
    xyz = np.array([1.4, 2.0, 2.4]) + 0.35 * rng.standard_normal((n, 3))
    s = _sys(cv_type, n, groups, BOX, weights=np.linspace(1.0, 2.0, sum(len(g) for g in groups)).astype(np.float32))
    xi0, j0 = s.cv_eval(_pos4(xyz)[None])
    for trial in range(6):
        k = rng.integers(-2, 3, size=(n, 3))
        xi1, j1 = s.cv_eval(_pos4(xyz + k * np.array(BOX))[None])
        assert xi1[0, 0] == pytest.approx(xi0[0, 0], abs=2e-5)      # float32 coordinates of shifted atoms round differently
        assert np.allclose(j1, j0, atol=2e-4)
    # and with nothing crossing a boundary the box is invisible
    s_open = _sys(cv_type, n, groups, None, weights=np.linspace(1.0, 2.0, sum(len(g) for g in groups)).astype(np.float32))
    xi2, j2 = s_open.cv_eval(_pos4(xyz)[None])
    assert xi2[0, 0] == xi0[0, 0] and np.array_equal(j2, j0)


def test_jacobian_matches_finite_differences_across_the_boundary():
    rng = np.random.default_rng(5)
    n = 4
    xyz = np.array([0.05, 3.95, 0.1]) + 0.3 * rng.standard_normal((n, 3))    # straddles three faces
    xyz = np.mod(xyz, np.array(BOX))                                          # wrapped into the box, as an engine stores it
    s = _sys(orc.DIHEDRAL, n, [[0], [1], [2], [3]], BOX)
    pos = _pos4(xyz)
    pos[:, :3] = np.round(pos[:, :3] * 1024) / 1024                          # exactly representable steps
    xi, jac = s.cv_eval(pos[None])
    h = 2.0 ** -10
    for a in range(n):
        for x in range(3):
            p, m = pos.copy(), pos.copy()
            p[a, x] += h
            m[a, x] -= h
            d = s.cv_eval(p[None], want_jac=False)[0, 0] - s.cv_eval(m[None], want_jac=False)[0, 0]
            d -= 2 * math.pi * round(d / (2 * math.pi))
            assert d / (2 * h) == pytest.approx(jac[0, a, x], rel=1e-5, abs=1e-5)


def test_forces_of_a_wrapped_molecule_have_no_net_force():
    rng = np.random.default_rng(3)
    xyz = np.mod(np.array([2.95, 0.05, 4.9]) + 0.3 * rng.standard_normal((4, 3)), np.array(BOX))
    s = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], BOX)
    f = s.apply_forces(_pos4(xyz)[None], np.array([[7.0]]), np.zeros((1, 4, 3)))
    assert np.abs(f.sum(axis=1)).max() < 1e-9 * np.abs(f).sum()


def test_contiguous_range_groups_wrapped_atom_by_atom_are_made_whole():
    """range groups follow the same rule (images nearest to the range's FIRST atom): a chain whose atoms an engine has
    wrapped one by one into the box gives the CVs, Jacobians and forces of the unwrapped chain (extent < half the box).
    Dyadic coordinates and box lengths make every wrap exact in binary32, so the comparison is to rounding error."""
    rng = np.random.default_rng(12)
    n, L = 600, (16.0, 32.0, 16.0)
    steps = rng.integers(-64, 65, size=(n, 3)) / 1024.0                      # a random walk on a dyadic lattice
    xyz = np.array([15.5, 0.25, 8.0]) + np.cumsum(steps, axis=0)             # starts next to two faces, extent ~ 1.5
    assert np.ptp(xyz, axis=0).max() < 0.4 * min(L)
    wrapped = np.mod(xyz, np.array(L))
    assert (np.abs(wrapped - xyz) > 1).any()                                  # it really crosses faces
    h = n // 2
    cvs = [{"type": orc.RGYR, "groups": [("range", 0, n)], "axis": 0, "period": 0.0},
           {"type": orc.DISTANCE, "groups": [("range", 0, h), ("range", h, n - h)], "axis": 0, "period": 0.0}]
    aw = rng.uniform(1.0, 4.0, size=n).astype(np.float32)
    s_box = orc.System(1, n, n, 4, cvs, None, atom_weight=aw, box=L)
    s_open = orc.System(1, n, n, 4, cvs, None, atom_weight=aw, box=None)
    xi_w = s_box.cv_eval(_pos4(wrapped)[None], want_jac=False)
    xi_o = s_open.cv_eval(_pos4(xyz)[None], want_jac=False)
    assert np.allclose(xi_w, xi_o, rtol=1e-12, atol=1e-12)
    dV = np.array([[3.0, -2.0]])
    f_w = s_box.apply_forces(_pos4(wrapped)[None], dV, np.zeros((1, n, 3)))
    f_o = s_open.apply_forces(_pos4(xyz)[None], dV, np.zeros((1, n, 3)))
    assert np.allclose(f_w, f_o, rtol=1e-10, atol=1e-12)
    assert np.abs(f_w.sum(axis=1)).max() < 1e-9 * np.abs(f_w).sum()
    # without the box the wrapped chain is a different (torn) object
    xi_torn = s_open.cv_eval(_pos4(wrapped)[None], want_jac=False)
    assert abs(xi_torn[0, 0] - xi_o[0, 0]) > 1.0
