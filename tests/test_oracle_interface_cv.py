"""Pins for the oracle's DistanceToInterface CV (Eq. 4-8, Appendix A).

The oracle follows the paper's listing line by line; what pins it is what the mathematics fixes: the two-bin case (the
softmax has one entry, so the interface is the midpoint of the scope whatever the atoms do), a hand-computed three-bin case
with one atom, a slab symmetric about the scope centre (two equal density steps -> the interface sits at the centre), a
sharp single interface recovered to within a bin, covariance under shifting atoms and scope together, the mobile group's
1:1 response, and central finite differences of the value against the analytic derivatives.  No CUDA here.
"""
import math

import numpy as np
import pytest

import oracle as orc


def _pos(x_axis, axis=0, n_extra=2, seed=0):
    """positions [N][4]: atoms 0..n_extra-1 are the mobile group, the rest the interface group with the given axis coords"""
    rng = np.random.default_rng(seed)
    n = n_extra + len(x_axis)
    p = rng.normal(size=(n, 4)).astype(np.float32)
    p[n_extra:, axis] = np.asarray(x_axis, np.float32)
    return p


def test_two_bins_midpoint_whatever_the_atoms_do():
    p = _pos(np.random.default_rng(1).uniform(-3, 5, size=40), axis=1)
    xi, jm, dx, _ = orc.dist_to_interface(p, [0, 1], [1.0, 3.0], 2, 40, 1, 0.4, (-1.0, 2.0), 2, 1.7)
    mobile = (p[0, 1] * 1.0 + p[1, 1] * 3.0) / 4.0
    assert xi == pytest.approx(mobile - 0.5, abs=1e-12)
    assert np.allclose(dx, 0.0, atol=1e-15)                       # a one-entry softmax does not move
    assert np.allclose(jm, [[0, 0.25, 0], [0, 0.75, 0]])


def test_three_bins_one_atom_by_hand():
    # one atom at x = 0.3; centres 0, 1, 2; sigma = 1; coeff = 2
    p = _pos([0.3], axis=0, n_extra=1)
    xi, _, _, mass = orc.dist_to_interface(p, [0], None, 1, 1, 0, 1.0, (0.0, 2.0), 3, 2.0)
    x = float(np.float32(0.3))
    e = [math.exp(-0.5 * (x - c) ** 2) for c in (0.0, 1.0, 2.0)]
    assert np.allclose(mass, e, rtol=1e-14)
    a, b = abs(e[1] - e[0]) * 2.0, abs(e[2] - e[1]) * 2.0
    pa, pb = math.exp(a) / (math.exp(a) + math.exp(b)), math.exp(b) / (math.exp(a) + math.exp(b))
    assert xi == pytest.approx(float(p[0, 0]) - (pa * 0.5 + pb * 1.5), rel=1e-13)


def test_symmetric_slab_puts_the_interface_at_the_centre():
    xs = np.arange(-1.0, 1.0 + 1e-9, 0.01)                        # a slab |x| <= 1: steps of equal height at -1 and +1
    p = _pos(xs, n_extra=1)
    xi, _, _, _ = orc.dist_to_interface(p, [0], None, 1, len(xs), 0, 0.1, (-3.0, 3.0), 121, 0.5)
    assert float(p[0, 0]) - xi == pytest.approx(0.0, abs=1e-6)


def test_sharp_single_interface_is_found_to_within_a_bin():
    x0 = 0.73
    xs = np.arange(-6.0, x0, 0.005)                                # dense liquid left of x0, nothing to the right
    p = _pos(xs, n_extra=1)
    lo, hi, bins = -2.0, 3.0, 101                                  # the far edge of the liquid lies outside the scope
    xi, _, _, _ = orc.dist_to_interface(p, [0], None, 1, len(xs), 0, 0.05, (lo, hi), bins, 5.0)
    assert abs((float(p[0, 0]) - xi) - x0) < (hi - lo) / (bins - 1)


def test_shift_covariance_and_mobile_response():
    rng = np.random.default_rng(4)
    xs = np.concatenate([rng.uniform(-2, 0.4, 300), rng.uniform(0.4, 3, 30)])
    p = _pos(xs, axis=2, n_extra=3, seed=2)
    args = dict(mobile_idx=[0, 1, 2], mobile_w=[2.0, 1.0, 1.0], ibegin=3, n_i=len(xs), axis=2, sigma=0.3, bins=50, coeff=0.8)
    xi0, _, _, _ = orc.dist_to_interface(p, scope=(-2.5, 3.5), **args)
    d = 0.375                                                      # exactly representable
    q = p.copy()
    q[3:, 2] += np.float32(d)                                      # interface atoms and scope move together ...
    xi1, _, _, _ = orc.dist_to_interface(q, scope=(-2.5 + d, 3.5 + d), **args)
    assert xi1 == pytest.approx(xi0 - d, abs=2e-6)                 # ... so does the interface (float32 coordinates)
    q = p.copy()
    q[:3, 2] += np.float32(d)                                      # the mobile group alone: 1:1
    xi2, _, _, _ = orc.dist_to_interface(q, scope=(-2.5, 3.5), **args)
    assert xi2 == pytest.approx(xi0 + d, abs=1e-6)


def test_derivatives_match_central_differences():
    rng = np.random.default_rng(9)
    xs = np.round(np.concatenate([rng.uniform(-1.5, 0.2, 60), rng.uniform(0.2, 2.5, 12)]) * 256) / 256
    p = _pos(xs, axis=0, n_extra=2, seed=5)
    kw = dict(mobile_idx=[0, 1], mobile_w=None, ibegin=2, n_i=len(xs), axis=0, sigma=0.35, scope=(-2.0, 3.0), bins=40, coeff=1.3)
    xi, jm, dx, _ = orc.dist_to_interface(p, **kw)
    h = 2.0 ** -12                                                 # exactly representable next to the 1/256 grid
    for i in list(range(0, len(xs), 7)) + [len(xs) - 1]:
        a, b = p.copy(), p.copy()
        a[2 + i, 0] += h
        b[2 + i, 0] -= h
        fd = (orc.dist_to_interface(a, **kw)[0] - orc.dist_to_interface(b, **kw)[0]) / (2 * h)
        assert fd == pytest.approx(dx[i], rel=2e-5, abs=1e-7)
    # the other coordinates of interface atoms do not matter
    a = p.copy()
    a[2:, 1] += 0.5
    assert orc.dist_to_interface(a, **kw)[0] == xi
    assert np.allclose(jm, [[0.5, 0, 0], [0.5, 0, 0]])
