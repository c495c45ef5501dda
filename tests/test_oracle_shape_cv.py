"""Pins for the oracle's gyration-tensor shape CVs (reading R-SHAPE).

The paper names PrincipalMoment, Asphericity, Acylindricity and ShapeAnisotropy without a formula, so the definitions are a
reading; what pins the arithmetic is mathematics: point sets whose gyration tensor is diagonal by construction (values by
hand), numpy.linalg.eigvalsh on a tensor assembled here with numpy, the trace identity with the separately pinned radius
of gyration, the eigenvalue-free form of the anisotropy 3/2 tr(S^2)/(tr S)^2 - 1/2, rotation and translation invariance,
and central finite differences of the values against the analytic Jacobians.  Nothing here calls the CUDA path.
"""
import numpy as np
import pytest

import oracle as orc

SHAPES = [(orc.PRINCIPAL_MOMENT, 0), (orc.PRINCIPAL_MOMENT, 1), (orc.PRINCIPAL_MOMENT, 2), (orc.ASPHERICITY, 0),
          (orc.ACYLINDRICITY, 0), (orc.SHAPE_ANISOTROPY, 0)]


def _eval(xyz, cv_type, axis=0, weights=None, want_jac=True, lead=2):
    """the group is atoms lead..lead+n-1 of a larger array (the leading atoms must not matter)"""
    n = len(xyz)
    pos = np.full((1, lead + n, 4), 7.5, np.float32)
    pos[0, lead:, :3] = np.asarray(xyz, np.float32)
    cv = {"type": cv_type, "groups": [("slots", 0, n)], "axis": axis, "period": 0.0}
    s = orc.System(1, lead + n, lead + n, 4, [cv], np.arange(lead, lead + n, dtype=np.int32),
                   slot_weight=None if weights is None else np.asarray(weights, np.float32))
    if want_jac:
        xi, jac = s.cv_eval(pos)
        return xi[0, 0], jac[0]
    return s.cv_eval(pos, want_jac=False)[0, 0], None


def _tensor(xyz, w=None):
    x = np.asarray(np.asarray(xyz, np.float32), np.float64)
    w = np.ones(len(x)) if w is None else np.asarray(np.asarray(w, np.float32), np.float64)
    c = (w[:, None] * x).sum(0) / w.sum()
    d = x - c
    return np.einsum("i,ix,iy->xy", w, d, d) / w.sum()


def test_octahedron_by_hand():
    # (+-a,0,0), (0,+-b,0), (0,0,+-c): S = diag(2a^2, 2b^2, 2c^2)/6, centred at the origin
    a, b, c = 3.0, 2.0, 1.0
    xyz = [[a, 0, 0], [-a, 0, 0], [0, b, 0], [0, -b, 0], [0, 0, c], [0, 0, -c]]
    l1, l2, l3 = a * a / 3, b * b / 3, c * c / 3
    assert _eval(xyz, orc.PRINCIPAL_MOMENT, 0)[0] == pytest.approx(l1, rel=1e-14)
    assert _eval(xyz, orc.PRINCIPAL_MOMENT, 1)[0] == pytest.approx(l2, rel=1e-14)
    assert _eval(xyz, orc.PRINCIPAL_MOMENT, 2)[0] == pytest.approx(l3, rel=1e-14)
    asp, acy = l1 - 0.5 * (l2 + l3), l2 - l3
    assert _eval(xyz, orc.ASPHERICITY)[0] == pytest.approx(asp, rel=1e-14)
    assert _eval(xyz, orc.ACYLINDRICITY)[0] == pytest.approx(acy, rel=1e-14)
    assert _eval(xyz, orc.SHAPE_ANISOTROPY)[0] == pytest.approx((asp ** 2 + 0.75 * acy ** 2) / (l1 + l2 + l3) ** 2, rel=1e-14)
    # the largest eigenvalue moves with the atoms on its own axis only: d l1 / d r = (2/N) x e_x for (+-a,0,0), 0 elsewhere
    _, jac = _eval(xyz, orc.PRINCIPAL_MOMENT, 0)
    want = np.zeros((6, 3))
    want[0, 0], want[1, 0] = 2 * a / 6, -2 * a / 6
    assert np.allclose(jac, want, atol=1e-14)


def test_rod_sphere_and_point_limits():
    t = np.linspace(-1.0, 1.0, 9)
    rod = np.outer(t, [0.6, 0.0, 0.8])                                  # collinear: l2 = l3 = 0
    var = np.mean(np.asarray(rod, np.float32).astype(np.float64) ** 2, axis=0).sum()
    assert _eval(rod, orc.PRINCIPAL_MOMENT, 0)[0] == pytest.approx(var, rel=1e-12)
    assert abs(_eval(rod, orc.PRINCIPAL_MOMENT, 1)[0]) < 1e-15 and abs(_eval(rod, orc.PRINCIPAL_MOMENT, 2)[0]) < 1e-15
    assert _eval(rod, orc.SHAPE_ANISOTROPY)[0] == pytest.approx(1.0, rel=1e-12)
    assert _eval(rod, orc.ASPHERICITY)[0] == pytest.approx(var, rel=1e-12)
    cube = [[x, y, z] for x in (-1, 1) for y in (-1, 1) for z in (-1, 1)]   # isotropic: every shape measure vanishes
    for ty in (orc.ASPHERICITY, orc.ACYLINDRICITY, orc.SHAPE_ANISOTROPY):
        assert abs(_eval(cube, ty)[0]) < 1e-15
    assert _eval(cube, orc.PRINCIPAL_MOMENT, 1)[0] == pytest.approx(1.0, rel=1e-14)
    xi, jac = _eval([[0.3, 0.2, 0.1]], orc.SHAPE_ANISOTROPY)                # a point: defined as 0, no force
    assert xi == 0.0 and not jac.any()
    disk = [[np.cos(a), np.sin(a), 0.0] for a in np.arange(8) * np.pi / 4]  # l = (1/2, 1/2, 0): kappa^2 = 1/4
    assert _eval(disk, orc.SHAPE_ANISOTROPY)[0] == pytest.approx(0.25, abs=1e-7)


def test_against_numpy_eigvalsh_trace_and_invariant_forms():
    rng = np.random.default_rng(12)
    for trial in range(5):
        n = int(rng.integers(4, 40))
        xyz = rng.normal(size=(n, 3)) * rng.uniform(0.3, 3.0, size=3) + rng.uniform(-5, 5, size=3)
        w = rng.uniform(1.0, 16.0, size=n) if trial % 2 else None
        S = _tensor(xyz, w)
        lam = np.linalg.eigvalsh(S)[::-1]
        for k in range(3):
            assert _eval(xyz, orc.PRINCIPAL_MOMENT, k, w, False)[0] == pytest.approx(lam[k], rel=1e-11)
        assert _eval(xyz, orc.ASPHERICITY, 0, w, False)[0] == pytest.approx(lam[0] - 0.5 * (lam[1] + lam[2]), rel=1e-11)
        assert _eval(xyz, orc.ACYLINDRICITY, 0, w, False)[0] == pytest.approx(lam[1] - lam[2], rel=1e-11)
        kap = 1.5 * np.trace(S @ S) / np.trace(S) ** 2 - 0.5           # needs no eigenvalues at all
        assert _eval(xyz, orc.SHAPE_ANISOTROPY, 0, w, False)[0] == pytest.approx(kap, rel=1e-11)
        rg = _eval(xyz, orc.RGYR, 0, w, False)[0]                      # pinned on its own in test_oracle_cv.py
        tr = sum(_eval(xyz, orc.PRINCIPAL_MOMENT, k, w, False)[0] for k in range(3))
        assert tr == pytest.approx(rg * rg, rel=1e-12)


@pytest.mark.parametrize("cv_type,axis", SHAPES)
def test_rotation_and_translation_invariance(cv_type, axis):
    rng = np.random.default_rng(21)
    xyz = rng.normal(size=(11, 3)) * [2.0, 1.0, 0.5]
    w = rng.uniform(1.0, 4.0, size=11)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    xi0, j0 = _eval(xyz, cv_type, axis, w)
    xi1, j1 = _eval(xyz @ q.T + [3.0, -2.0, 1.0], cv_type, axis, w)
    assert xi1 == pytest.approx(xi0, rel=2e-6)                           # float32 coordinates round differently
    assert np.allclose(j1, j0 @ q.T, atol=2e-6 * np.abs(j0).max())       # the Jacobian rotates with the molecule
    assert np.abs(j0.sum(axis=0)).max() < 1e-14 * np.abs(j0).sum()       # no net force
    torque = np.cross(np.asarray(xyz, np.float32).astype(np.float64), j0).sum(axis=0)
    assert np.abs(torque).max() < 1e-12 * np.abs(j0).sum()               # no net torque


@pytest.mark.parametrize("cv_type,axis", SHAPES)
def test_jacobian_matches_central_differences(cv_type, axis):
    rng = np.random.default_rng(33)
    xyz = np.round(rng.normal(size=(9, 3)) * [1.8, 1.1, 0.6] * 256) / 256     # well separated eigenvalues
    w = np.round(rng.uniform(1.0, 8.0, size=9) * 4) / 4
    _, jac = _eval(xyz, cv_type, axis, w)
    h = 2.0 ** -10
    for i in range(9):
        for x in range(3):
            a, b = xyz.copy(), xyz.copy()
            a[i, x] += h
            b[i, x] -= h
            fd = (_eval(a, cv_type, axis, w, False)[0] - _eval(b, cv_type, axis, w, False)[0]) / (2 * h)
            assert fd == pytest.approx(jac[i, x], rel=2e-5, abs=2e-7)


def test_anisotropy_jacobian_is_smooth_through_degenerate_eigenvalues():
    """kappa^2 = 3/2 tr(S^2)/(tr S)^2 - 1/2 is a smooth function of S, so its Jacobian must not depend on which eigenvectors
    the solver picks inside a degenerate pair: dkappa2/dr_i = (2 w_i/W) (3 S/t^2 - 3 tr(S^2)/t^3 I)(r_i - c)"""
    xyz = np.array([[2.0, 0, 0], [-2.0, 0, 0], [0, 1.0, 0], [0, -1.0, 0], [0, 0, 1.0], [0, 0, -1.0]])   # l2 = l3 exactly
    _, jac = _eval(xyz, orc.SHAPE_ANISOTROPY)
    S = _tensor(xyz)
    t = np.trace(S)
    M = 3 * S / t ** 2 - 3 * np.trace(S @ S) / t ** 3 * np.eye(3)
    assert np.allclose(jac, (2.0 / 6.0) * xyz @ M.T, atol=1e-14)


@pytest.mark.parametrize("cv_type,axis", SHAPES)
def test_contiguous_range_group_equals_the_tensor_assembled_here(cv_type, axis):
    """the same CVs over a contiguous atom range with per-atom weights (how a polymer window uses them): value against
    numpy.linalg.eigvalsh of the tensor assembled here, forces against central finite differences of the value"""
    rng = np.random.default_rng(21)
    n, first = 60, 7
    xyz = rng.standard_normal((first + n + 5, 3)) * np.array([2.0, 1.0, 0.5]) + 30.0
    aw = rng.uniform(1.0, 9.0, size=len(xyz)).astype(np.float32)
    pos = np.zeros((1, len(xyz), 4), np.float32)
    pos[0, :, :3] = xyz
    cv = {"type": cv_type, "groups": [("range", first, n)], "axis": axis, "period": 0.0}
    s = orc.System(1, len(xyz), len(xyz), 4, [cv], None, atom_weight=aw)
    lam = np.sort(np.linalg.eigvalsh(_tensor(pos[0, first:first + n, :3], aw[first:first + n])))[::-1]
    b, c = lam[0] - 0.5 * (lam[1] + lam[2]), lam[1] - lam[2]
    want = {orc.PRINCIPAL_MOMENT: lam[axis], orc.ASPHERICITY: b, orc.ACYLINDRICITY: c,
            orc.SHAPE_ANISOTROPY: (b * b + 0.75 * c * c) / lam.sum() ** 2}[cv_type]
    assert s.cv_eval(pos, want_jac=False)[0, 0] == pytest.approx(want, rel=1e-10)
    f = s.apply_forces(pos, np.array([[1.0]]), np.zeros((1, len(xyz), 3)))       # F = -d xi / d r
    assert np.all(f[0, :first] == 0) and np.all(f[0, first + n:] == 0)
    h = 2.0 ** -9
    for a in (first, first + 17, first + n - 1):
        for x in range(3):
            p, m = pos.copy(), pos.copy()
            p[0, a, x] += h
            m[0, a, x] -= h
            d = (s.cv_eval(p, want_jac=False)[0, 0] - s.cv_eval(m, want_jac=False)[0, 0]) / (2 * h)
            assert -f[0, a, x] == pytest.approx(d, rel=2e-5, abs=1e-7)
