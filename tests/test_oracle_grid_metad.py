"""Pins for the oracle's grid-stored metadynamics (reading R-GRID).

The paper says only that the bias may be stored "on a pre-defined grid", so layout and interpolation are a reading; what pins
the arithmetic: node values against the separately pinned hill sum (orc.metad), exact reproduction of multilinear functions
written straight into the node array, scipy's RegularGridInterpolator, second-order convergence to the exact hill sum, periodic
images, clamping outside an open grid, and well-tempered heights worked by hand.  Nothing here calls the CUDA path.
"""
import math

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import oracle as orc


def _nodes(lower, upper, shape, periodic):
    ax = []
    for lo, up, n, p in zip(lower, upper, shape, periodic):
        h = (up - lo) / (n if p else n - 1)
        ax.append(lo + h * np.arange(n))
    return ax


def test_nodes_hold_the_exact_hill_sum_and_gradient():
    lower, upper, shape, periodic = (-math.pi, 0.5), (math.pi, 2.0), (12, 7), (1, 0)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    rng = np.random.default_rng(2)
    sigma = np.array([0.6, 0.3])
    hills = np.stack([rng.uniform(-math.pi, math.pi, 9), rng.uniform(0.4, 2.1, 9)], axis=1).astype(np.float32)
    for c in hills:                                     # nine events of one walker each
        h = g.deposit(c[None], sigma, 1.25)
        assert h[0] == 1.25                             # standard metadynamics: constant height
    ax = _nodes(lower, upper, shape, periodic)
    pts = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 2)      # row-major, last CV fastest
    V, dV, _ = orc.metad(pts, hills, np.full(9, 1.25, np.float32), sigma, np.array([2 * math.pi, 0.0]))
    assert np.allclose(g.values[:, 0], V, rtol=1e-13, atol=1e-15)
    assert np.allclose(g.values[:, 1:], dV, rtol=1e-12, atol=1e-14)
    Vn, dVn = g.eval(pts)                               # evaluating AT the nodes returns them
    assert np.allclose(Vn, V, rtol=1e-13, atol=1e-15) and np.allclose(dVn, dV, rtol=1e-12, atol=1e-14)


def test_multilinear_functions_are_reproduced_exactly_and_scipy_agrees():
    lower, upper, shape, periodic = (-1.0, 2.0, 0.0), (1.0, 5.0, 1.0), (5, 4, 3), (0, 0, 0)
    g = orc.MetadGrid(lower, upper, shape, periodic)
    ax = _nodes(lower, upper, shape, periodic)
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    fn = [lambda x, y, z: 1.0 + 2.0 * x - 3.0 * y + 0.5 * z + 0.25 * x * y - 0.75 * y * z + 1.5 * x * y * z,
          lambda x, y, z: -2.0 + x * z, lambda x, y, z: 3.0 * y, lambda x, y, z: x - y + z]
    for c in range(4):
        g.values[:, c] = fn[c](X, Y, Z).reshape(-1)
    rng = np.random.default_rng(5)
    pts = np.stack([rng.uniform(lo, up, 200) for lo, up in zip(lower, upper)], axis=1)
    V, dV = g.eval(pts)
    assert np.allclose(V, fn[0](*pts.T), rtol=1e-13, atol=1e-13)
    for c in range(3):
        assert np.allclose(dV[:, c], fn[c + 1](*pts.T), rtol=1e-13, atol=1e-13)
    # a rough field: only a library interpolator knows the answer
    g.values[:] = rng.normal(size=g.values.shape)
    V, dV = g.eval(pts)
    for c in range(4):
        ref = RegularGridInterpolator(ax, g.values[:, c].reshape(shape), method="linear")(pts)
        assert np.allclose(V if c == 0 else dV[:, c - 1], ref, rtol=1e-12, atol=1e-13)
    # outside an open grid: the value on the nearest face
    out = np.array([[-4.0, 3.0, 0.5], [0.3, 9.0, -2.0]])
    assert np.allclose(g.eval(out)[0], g.eval(np.clip(out, lower, upper))[0], rtol=0, atol=0)


def test_second_order_convergence_to_the_exact_hill_sum():
    rng = np.random.default_rng(8)
    sigma = np.array([0.35, 0.25])
    hills = rng.uniform(-1.0, 1.0, size=(30, 2)).astype(np.float32)
    heights = np.full(30, 1.2, np.float32)
    pts = rng.uniform(-1.2, 1.2, size=(4000, 2))
    V, dV, _ = orc.metad(pts, hills, heights, sigma, np.zeros(2))
    errs = []
    for n in (41, 81, 161):
        g = orc.MetadGrid((-2.0, -2.0), (2.0, 2.0), (n, n), (0, 0))
        g.deposit(hills, sigma, 1.2)                    # thirty walkers, one event
        Vg, dVg = g.eval(pts)
        errs.append((np.abs(Vg - V).mean(), np.abs(dVg - dV).mean()))      # mean: the maximum depends on where the points fall in a cell
        h = 4.0 / (n - 1)
        # linear interpolation: |error| <= sum_k h_k^2/8 max|d2V/dxi_k^2|, and |V''| <= sum of heights / sigma^2
        assert np.abs(Vg - V).max() <= (h * h / 8) * (30 * 1.2) * (1 / sigma[0] ** 2 + 1 / sigma[1] ** 2)
    for a, b in zip(errs, errs[1:]):
        assert a[0] / b[0] == pytest.approx(4.0, rel=0.1) and a[1] / b[1] == pytest.approx(4.0, rel=0.1)


def test_periodic_images_and_wrapping():
    P = 2 * math.pi
    g = orc.MetadGrid((-math.pi,), (math.pi,), (64,), (1,))
    sigma = np.array([0.4])
    g.deposit(np.array([[3.0]], np.float32), sigma, 2.0)         # 0.14 below the upper edge
    x = np.array([[-3.1], [3.1], [-3.1 + P], [3.1 - 3 * P], [-math.pi], [math.pi]])
    V, dV = g.eval(x)
    assert V[0] == pytest.approx(V[2], rel=1e-12) and V[1] == pytest.approx(V[3], rel=1e-12)
    assert V[4] == pytest.approx(V[5], rel=1e-12)                # the two ends of the period are the same point
    Vx, dVx, _ = orc.metad(x[:2], np.array([[3.0]], np.float32), np.array([2.0], np.float32), sigma, np.array([P]))
    assert np.allclose(V[:2], Vx, rtol=0, atol=2.0 * (P / 64) ** 2 / 8 / 0.16)    # the image across the edge is felt
    assert V[0] > 1.5                                            # 0.083 from the hill through the boundary
    assert np.allclose(dV[:2, 0], dVx[:, 0], atol=0.1)


def test_well_tempered_heights_by_hand():
    g = orc.MetadGrid((0.0,), (4.0,), (5,), (0,))               # nodes at 0, 1, 2, 3, 4
    sigma, w0, kT = np.array([0.5]), 1.5, 2.0
    h1 = g.deposit(np.array([[2.0]], np.float32), sigma, w0, kT)
    assert h1[0] == w0                                           # empty grid: V = 0
    assert g.values[2, 0] == w0 and g.values[2, 1] == 0.0
    assert g.values[3, 0] == pytest.approx(w0 * math.exp(-2.0), rel=1e-15)
    assert g.values[3, 1] == pytest.approx(-w0 * math.exp(-2.0) * 1.0 / 0.25, rel=1e-15)
    # second event at 2.5: the grid says V = (V(2) + V(3))/2, not the exact Gaussian
    Vmid = 0.5 * (w0 + w0 * math.exp(-2.0))
    h2 = g.deposit(np.array([[2.5]], np.float32), sigma, w0, kT)
    assert h2[0] == pytest.approx(w0 * math.exp(-Vmid / kT), rel=1e-15)
    # two walkers in one event see the same grid (synchronous), the second does not feel the first; a masked walker deposits nothing
    g2 = orc.MetadGrid((0.0,), (4.0,), (5,), (0,))
    h = g2.deposit(np.array([[2.0], [2.0], [1.0]], np.float32), sigma, w0, kT, mask=[1, 1, 0])
    assert h[0] == w0 and h[1] == w0 and h[2] == 0.0
    assert g2.values[2, 0] == 2 * w0
