"""Pins for the oracle's collective variables and Jacobians (oracle/psg_oracle.c).

Nothing here calls the CUDA path.  Each check is fixed by mathematics, not by the
oracle: constructed geometries with known values, central finite differences of
the oracle's own VALUE against its analytic JACOBIAN (two different code paths),
homogeneity (Euler) identities and rigid-motion invariance.
PAPER.md:L185-L189 names the CVs; DESIGN.md lists the readings.
"""
import math

import numpy as np
import pytest

import oracle as orc

TWO_PI = 2.0 * math.pi


def _sys(cv_type, n_atoms, groups_atoms, weights=None, axis=0, period=0.0, stride=4):
    """one replica, explicit groups given as lists of atom indices"""
    slots, groups, o = [], [], 0
    for g in groups_atoms:
        groups.append(("slots", o, len(g)))
        slots += list(g)
        o += len(g)
    cv = {"type": cv_type, "groups": groups, "axis": axis, "period": period}
    return orc.System(1, n_atoms, n_atoms, stride, [cv], np.array(slots, np.int32), slot_weight=weights)


def _pos4(xyz, stride=4):
    xyz = np.asarray(xyz, np.float32)
    p = np.zeros((xyz.shape[0], stride), np.float32)
    p[:, :3] = xyz
    if stride == 4:
        p[:, 3] = 7.5  # w must be ignored
    return p


def _fd_jac(system, pos, h=2.0 ** -10):
    """central differences of xi wrt every coordinate of every slot atom. Positions are
    fp32, so h is a power of two and positions are pre-rounded to multiples of h/4:
    r +- h is then exact in binary32."""
    sa = system.slot_atom.reshape(-1)
    out = np.zeros((len(sa), 3))
    for s, a in enumerate(sa):
        for x in range(3):
            pp = pos.copy(); pm = pos.copy()
            pp[a, x] += np.float32(h); pm[a, x] -= np.float32(h)
            xp = system.cv_eval(pp, want_jac=False)[0, 0]
            xm = system.cv_eval(pm, want_jac=False)[0, 0]
            d = xp - xm
            if system.period[0] > 0:
                d -= system.period[0] * round(d / system.period[0])
            out[s, x] = d / (2 * h)
    return out


def _grid_round(xyz, q=2.0 ** -12):
    return np.round(np.asarray(xyz, np.float64) / q) * q


# ----------------------------------------------------------------- distance
def test_distance_345():
    s = _sys(orc.DISTANCE, 2, [[0], [1]])
    xi, jac = s.cv_eval(_pos4([[0, 0, 0], [3, 4, 0]]))
    assert xi[0, 0] == 5.0
    np.testing.assert_allclose(jac[0, 1], [0.6, 0.8, 0.0], atol=1e-15)
    np.testing.assert_allclose(jac[0, 0], [-0.6, -0.8, 0.0], atol=1e-15)


def test_distance_zero_has_zero_jacobian():
    s = _sys(orc.DISTANCE, 2, [[0], [1]])
    xi, jac = s.cv_eval(_pos4([[1, 2, 3], [1, 2, 3]]))
    assert xi[0, 0] == 0.0 and np.all(jac == 0.0)


def test_distance_groups_barycenter_and_weights():
    # group A = atoms 0,1 (weights 1,3), group B = atom 2
    pos = _pos4([[0, 0, 0], [4, 0, 0], [3, 4, 0]])
    s = _sys(orc.DISTANCE, 3, [[0, 1], [2]], weights=np.array([1, 3, 1], np.float32))
    xi, jac = s.cv_eval(pos)
    # barycenter A = (3,0,0) -> distance to (3,4,0) is 4 along +y
    assert xi[0, 0] == pytest.approx(4.0, abs=1e-15)
    np.testing.assert_allclose(jac[0], [[0, -0.25, 0], [0, -0.75, 0], [0, 1, 0]], atol=1e-15)


def test_stride3_equals_stride4():
    rng = np.random.default_rng(5)
    xyz = rng.normal(size=(4, 3))
    a = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], stride=4).cv_eval(_pos4(xyz, 4))
    b = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], stride=3).cv_eval(_pos4(xyz, 3))
    assert a[0][0, 0] == b[0][0, 0] and np.array_equal(a[1], b[1])


# -------------------------------------------------------------------- angle
def test_angle_right_and_equilateral():
    s = _sys(orc.ANGLE, 3, [[0], [1], [2]])
    xi, _ = s.cv_eval(_pos4([[1, 0, 0], [0, 0, 0], [0, 2, 0]]))
    assert xi[0, 0] == pytest.approx(math.pi / 2, abs=1e-15)
    xi, _ = s.cv_eval(_pos4([[0, 0, 0], [1, 0, 0], [0.5, math.sqrt(3) / 2, 0]]))
    assert xi[0, 0] == pytest.approx(math.pi / 3, abs=1e-7)  # fp32 input rounding of sqrt(3)/2
    # vertex is the SECOND group: (1,0,0)-(0,0,0)-(-1,1,0) is 135 degrees
    xi, _ = s.cv_eval(_pos4([[1, 0, 0], [0, 0, 0], [-1, 1, 0]]))
    assert xi[0, 0] == pytest.approx(0.75 * math.pi, abs=1e-15)


def test_angle_collinear_has_zero_jacobian():
    s = _sys(orc.ANGLE, 3, [[0], [1], [2]])
    xi, jac = s.cv_eval(_pos4([[1, 0, 0], [0, 0, 0], [-2, 0, 0]]))
    assert xi[0, 0] == pytest.approx(math.pi) and np.all(jac == 0.0)


# ----------------------------------------------------------------- dihedral
@pytest.mark.parametrize("phi", [0.3, -2.0, math.pi - 1e-3, -(math.pi - 1e-3), 0.0, 1.5, -0.7])
def test_dihedral_constructed_geometry(phi):
    """c2=(0,0,0), c3=(0,0,1), c1=(1,0,0), c4=(cos phi, sin phi, 1): the IUPAC dihedral is phi."""
    s = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], period=TWO_PI)
    pos = _pos4([[1, 0, 0], [0, 0, 0], [0, 0, 1], [math.cos(phi), math.sin(phi), 1]])
    xi, _ = s.cv_eval(pos)
    assert xi[0, 0] == pytest.approx(phi, abs=2e-7)  # fp32 rounding of cos/sin inputs
    # mirror image (y -> -y) flips the sign
    pos[:, 1] *= -1
    xi2, _ = s.cv_eval(pos)
    assert xi2[0, 0] == pytest.approx(-phi, abs=2e-7)


def test_dihedral_cis_trans():
    s = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], period=TWO_PI)
    cis, _ = s.cv_eval(_pos4([[1, 0, 0], [0, 0, 0], [0, 0, 1], [1, 0, 1]]))
    trans, _ = s.cv_eval(_pos4([[1, 0, 0], [0, 0, 0], [0, 0, 1], [-1, 0, 1]]))
    assert cis[0, 0] == 0.0 and abs(trans[0, 0]) == pytest.approx(math.pi, abs=1e-15)


def test_dihedral_degenerate_has_zero_jacobian():
    s = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], period=TWO_PI)
    _, jac = s.cv_eval(_pos4([[0, 0, -1], [0, 0, 0], [0, 0, 1], [1, 0, 1]]))  # b1 parallel b2
    assert np.all(jac == 0.0)


def _rot(axis, ang):
    axis = np.asarray(axis, float) / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + math.sin(ang) * K + (1 - math.cos(ang)) * K @ K


@pytest.mark.parametrize("cvt,n", [(orc.DISTANCE, 2), (orc.ANGLE, 3), (orc.DIHEDRAL, 4)])
def test_rigid_motion_invariance_of_value(cvt, n):
    """internal coordinates do not change under rotation + translation (to fp32 input rounding)."""
    rng = np.random.default_rng(11 + n)
    xyz = rng.normal(size=(n, 3))
    s = _sys(cvt, n, [[i] for i in range(n)], period=TWO_PI if cvt == orc.DIHEDRAL else 0.0)
    x0 = s.cv_eval(_pos4(xyz), want_jac=False)[0, 0]
    moved = xyz @ _rot([1, 2, 3], 0.83).T + np.array([0.5, -1.25, 2.0])
    x1 = s.cv_eval(_pos4(moved), want_jac=False)[0, 0]
    assert x1 == pytest.approx(x0, abs=5e-6)


# ------------------------------------------------- Jacobians: FD + identities
CASES = [
    (orc.DISTANCE, [[0], [1]], 0.0),
    (orc.DISTANCE, [[0, 1], [2, 3, 4]], 0.0),
    (orc.ANGLE, [[0], [1], [2]], 0.0),
    (orc.ANGLE, [[0, 3], [1], [2, 4]], 0.0),
    (orc.DIHEDRAL, [[0], [1], [2], [3]], TWO_PI),
    (orc.DIHEDRAL, [[0, 4], [1], [2, 5], [3]], TWO_PI),
]


@pytest.mark.parametrize("cvt,groups,period", CASES)
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_jacobian_fd_and_invariants(cvt, groups, period, seed):
    rng = np.random.default_rng(100 * cvt + seed)
    n = 1 + max(max(g) for g in groups)
    xyz = _grid_round(rng.normal(size=(n, 3)) * 1.5)
    nslots = sum(len(g) for g in groups)
    w = rng.uniform(1, 16, size=nslots).astype(np.float32) if seed % 2 else None
    s = _sys(cvt, n, groups, weights=w, period=period)
    pos = _pos4(xyz)
    xi, jac = s.cv_eval(pos)
    fd = _fd_jac(s, pos)
    # central FD with h = 2^-10 has O(h^2) ~ 1e-6 truncation: 1e-6 relative to the largest entry
    assert np.max(np.abs(fd - jac[0])) <= 1e-6 * max(1.0, np.max(np.abs(jac[0]))) * 4
    sa = s.slot_atom.reshape(-1)
    r = pos[sa, :3].astype(np.float64)
    J = jac[0]
    # translation invariance: sum_i J_i = 0; rotation invariance: sum_i r_i x J_i = 0
    assert np.max(np.abs(J.sum(axis=0))) < 1e-12
    assert np.max(np.abs(np.cross(r, J).sum(axis=0))) < 1e-12
    # Euler: distance is homogeneous of degree 1, angles of degree 0
    euler = float((r * J).sum())
    assert euler == pytest.approx(xi[0, 0] if cvt == orc.DISTANCE else 0.0, abs=1e-12)


def test_dihedral_fd_tight_richardson():
    """Richardson-extrapolated FD reaches 1e-8 relative: excludes an O(1e-6) formula error."""
    rng = np.random.default_rng(77)
    xyz = _grid_round(rng.normal(size=(4, 3)))
    s = _sys(orc.DIHEDRAL, 4, [[0], [1], [2], [3]], period=TWO_PI)
    pos = _pos4(xyz)
    _, jac = s.cv_eval(pos)
    f1 = _fd_jac(s, pos, 2.0 ** -8)
    f2 = _fd_jac(s, pos, 2.0 ** -9)
    rich = (4 * f2 - f1) / 3
    assert np.max(np.abs(rich - jac[0])) <= 1e-8 * np.max(np.abs(jac[0])) * 10


# ------------------------------------------------- component / center of mass
def test_component_is_mean_and_weighted_mean():
    rng = np.random.default_rng(3)
    xyz = rng.normal(size=(6, 3)).astype(np.float32)
    for axis in range(3):
        s = _sys(orc.COMPONENT, 6, [[0, 1, 2, 3, 4, 5]], axis=axis)
        xi, jac = s.cv_eval(_pos4(xyz))
        assert xi[0, 0] == pytest.approx(float(xyz[:, axis].astype(np.float64).mean()), abs=1e-15)
        e = np.zeros(3); e[axis] = 1
        np.testing.assert_allclose(jac[0].sum(axis=0), e, atol=1e-15)
    w = np.array([1, 2, 3, 4, 5, 6], np.float32)
    s = _sys(orc.COMPONENT, 6, [[0, 1, 2, 3, 4, 5]], weights=w, axis=1)
    xi, jac = s.cv_eval(_pos4(xyz))
    assert xi[0, 0] == pytest.approx(float((w * xyz[:, 1].astype(np.float64)).sum() / w.sum()), abs=1e-15)
    np.testing.assert_allclose(jac[0, :, 1], w / w.sum(), atol=1e-15)
    # translation covariance (exactly representable shift)
    xi2, _ = s.cv_eval(_pos4(xyz + np.float32(2.0)))
    assert xi2[0, 0] == pytest.approx(xi[0, 0] + 2.0, abs=1e-6)


def test_component_range_group_equals_explicit():
    rng = np.random.default_rng(4)
    xyz = rng.normal(size=(50, 3)).astype(np.float32)
    cv_r = {"type": orc.COMPONENT, "groups": [("range", 10, 30)], "axis": 2}
    cv_e = {"type": orc.COMPONENT, "groups": [("slots", 0, 30)], "axis": 2}
    a = orc.System(1, 50, 50, 4, [cv_r], None).cv_eval(_pos4(xyz))
    b = orc.System(1, 50, 50, 4, [cv_e], np.arange(10, 40, dtype=np.int32)).cv_eval(_pos4(xyz))
    assert a[0][0, 0] == b[0][0, 0] and np.array_equal(a[1], b[1])


# ---------------------------------------------------------- radius of gyration
def test_rgyr_cube_and_pair():
    a = 2.0
    corners = [[x, y, z] for x in (0, a) for y in (0, a) for z in (0, a)]
    s = _sys(orc.RGYR, 8, [list(range(8))])
    xi, jac = s.cv_eval(_pos4(corners))
    assert xi[0, 0] == pytest.approx(a * math.sqrt(3) / 2, abs=1e-15)  # 1.7320508075688772
    s2 = _sys(orc.RGYR, 2, [[0, 1]])
    xi2, _ = s2.cv_eval(_pos4([[0, 0, 0], [0, 3, 0]]))
    assert xi2[0, 0] == pytest.approx(1.5, abs=1e-15)
    # weighted two-point: Rg^2 = w1 w2 L^2 / W^2
    s3 = _sys(orc.RGYR, 2, [[0, 1]], weights=np.array([1, 3], np.float32))
    xi3, _ = s3.cv_eval(_pos4([[0, 0, 0], [0, 4, 0]]))
    assert xi3[0, 0] == pytest.approx(math.sqrt(3.0) * 4 / 4, abs=1e-15)


def test_rgyr_single_point_zero_jacobian():
    s = _sys(orc.RGYR, 1, [[0]])
    xi, jac = s.cv_eval(_pos4([[1, 2, 3]]))
    assert xi[0, 0] == 0.0 and np.all(jac == 0.0)


@pytest.mark.parametrize("weighted", [False, True])
def test_rgyr_scaling_euler_fd(weighted):
    rng = np.random.default_rng(9)
    n = 12
    xyz = _grid_round(rng.normal(size=(n, 3)) * 2)
    w = rng.uniform(1, 16, size=n).astype(np.float32) if weighted else None
    s = _sys(orc.RGYR, n, [list(range(n))], weights=w)
    pos = _pos4(xyz)
    xi, jac = s.cv_eval(pos)
    xi2, _ = s.cv_eval(_pos4(2.0 * xyz))
    assert xi2[0, 0] == pytest.approx(2.0 * xi[0, 0], rel=1e-14)
    J = jac[0]
    r = pos[:, :3].astype(np.float64)
    assert float((r * J).sum()) == pytest.approx(xi[0, 0], rel=1e-13)  # homogeneous of degree 1
    assert np.max(np.abs(J.sum(axis=0))) < 1e-14
    assert np.max(np.abs(np.cross(r, J).sum(axis=0))) < 1e-13
    fd = _fd_jac(s, pos)
    assert np.max(np.abs(fd - J)) <= 4e-6 * np.max(np.abs(J))
    # definition via pairwise distances: Rg^2 = sum_{i<j} w_i w_j |r_i-r_j|^2 / W^2
    ww = np.ones(n) if w is None else w.astype(np.float64)
    d2 = ((r[:, None, :] - r[None, :, :]) ** 2).sum(-1)
    assert xi[0, 0] == pytest.approx(math.sqrt((ww[:, None] * ww[None, :] * d2).sum() / 2) / ww.sum(), rel=1e-13)


def test_rgyr_range_group_with_atom_weights():
    rng = np.random.default_rng(10)
    xyz = rng.normal(size=(40, 3)).astype(np.float32)
    aw = rng.uniform(1, 16, size=40).astype(np.float32)
    cv_r = {"type": orc.RGYR, "groups": [("range", 5, 20)]}
    cv_e = {"type": orc.RGYR, "groups": [("slots", 0, 20)]}
    a = orc.System(1, 40, 40, 4, [cv_r], None, atom_weight=aw).cv_eval(_pos4(xyz))
    b = orc.System(1, 40, 40, 4, [cv_e], np.arange(5, 25, dtype=np.int32), slot_weight=aw[5:25]).cv_eval(_pos4(xyz))
    assert a[0][0, 0] == b[0][0, 0] and np.array_equal(a[1], b[1])


# ------------------------------------------------------------- batch layout
def test_replica_layout_shared_vs_own_arrays():
    rng = np.random.default_rng(21)
    R, N = 5, 30
    pos = np.zeros((R, N, 4), np.float32)
    pos[..., :3] = rng.normal(size=(R, N, 3))
    cvs = [{"type": orc.DIHEDRAL, "groups": [("slots", i, 1) for i in range(4)], "period": TWO_PI},
           {"type": orc.DISTANCE, "groups": [("slots", 4, 1), ("slots", 5, 1)]}]
    idx = np.array([4, 6, 8, 14, 2, 20], np.int32)
    xi, jac = orc.System(R, N, N, 4, cvs, idx).cv_eval(pos)
    for r in range(R):
        x1, j1 = orc.System(1, N, N, 4, cvs, idx).cv_eval(pos[r])
        assert np.array_equal(xi[r], x1[0]) and np.array_equal(jac[r], j1[0])
    # per-replica index lists into ONE shared array
    idx2 = np.stack([rng.permutation(N)[:6] for _ in range(R)]).astype(np.int32)
    xi2, _ = orc.System(R, N, 0, 4, cvs, idx2).cv_eval(pos[0])
    for r in range(R):
        x1, _ = orc.System(1, N, N, 4, cvs, idx2[r]).cv_eval(pos[0])
        assert np.array_equal(xi2[r], x1[0])


# ---------------------------------------------------------------------------- Displacement
def test_displacement_components_and_distance_agree():
    """the three Displacement components of two weighted groups are the barycenter difference, their norm is the Distance
    CV of the same groups, and each Jacobian row is +-(w_i / W) e_axis"""
    rng = np.random.default_rng(21)
    xyz = rng.normal(size=(5, 3))
    w = np.array([1.0, 3.0, 2.0, 2.0, 4.0], np.float32)
    groups = [[0, 1], [2, 3, 4]]
    c1 = (w[:2, None] * xyz[:2]).sum(0) / w[:2].sum()
    c2 = (w[2:, None] * xyz[2:]).sum(0) / w[2:].sum()
    comps = []
    for ax in range(3):
        s = _sys(orc.DISPLACEMENT, 5, groups, weights=w, axis=ax)
        xi, jac = s.cv_eval(_pos4(xyz)[None])
        assert xi[0, 0] == pytest.approx((c2 - c1)[ax], abs=1e-6)
        want = np.zeros((5, 3))
        want[:2, ax] = -w[:2] / w[:2].sum()
        want[2:, ax] = w[2:] / w[2:].sum()
        assert np.allclose(jac[0], want, atol=1e-12)
        comps.append(xi[0, 0])
    d = _sys(orc.DISTANCE, 5, groups, weights=w).cv_eval(_pos4(xyz)[None], want_jac=False)[0, 0]
    assert math.sqrt(sum(c * c for c in comps)) == pytest.approx(d, rel=1e-12)


def test_displacement_minimum_image():
    cv = {"type": orc.DISPLACEMENT, "groups": [("slots", 0, 1), ("slots", 1, 1)], "axis": 0, "period": 0.0}
    s = orc.System(1, 2, 2, 4, [cv], np.array([0, 1], np.int32), box=(3.0, 0.0, 0.0))
    xi = s.cv_eval(_pos4([[0.1, 0, 0], [2.9, 0, 0]])[None], want_jac=False)
    assert xi[0, 0] == pytest.approx(-0.2, abs=1e-6)
