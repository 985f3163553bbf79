"""Pins of the oracle's shape functions and gather.

Every expected value comes from a closed form, a moment identity, or scipy's BSpline
(library routine) — never from the oracle itself or the CUDA path.
"""
import numpy as np
import pytest

import oracle
from oracle import OracleParams
from conftest import bspline_ref

ORDERS = (1, 2, 3)
STAG = ((0.5, 0, 0), (0, 0.5, 0), (0, 0, 0.5), (0, 0.5, 0.5), (0.5, 0, 0.5), (0.5, 0.5, 0))


@pytest.mark.parametrize("order", ORDERS)
def test_shape_equals_cardinal_bspline(order):
    d = np.linspace(-3.0, 3.0, 2401)
    got = np.array([oracle.shape(order, x) for x in d])
    np.testing.assert_allclose(got, bspline_ref(order, d), rtol=0, atol=2e-15)


@pytest.mark.parametrize("order", ORDERS)
def test_shape_moments(order):
    rng = np.random.default_rng(11)
    nodes = np.arange(-6, 7)
    for x in rng.uniform(-1.0, 1.0, 200):
        w = np.array([oracle.shape(order, x - i) for i in nodes])
        assert abs(w.sum() - 1.0) < 1e-14                      # partition of unity
        assert abs((nodes * w).sum() - x) < 1e-14              # first moment
        m2 = (((nodes - x) ** 2) * w).sum()
        f = x - np.floor(x)
        expect = {1: f * (1 - f), 2: 0.25, 3: 1.0 / 3.0}[order]  # second central moment
        assert abs(m2 - expect) < 1e-13
        assert (w >= 0).all() and np.count_nonzero(w) <= order + 1


def test_shape_known_values():
    assert oracle.shape(1, 0.25) == 0.75
    assert oracle.shape(2, 0.0) == 0.75 and oracle.shape(2, 0.5) == 0.5 and oracle.shape(2, 1.0) == 0.125
    assert abs(oracle.shape(3, 0.0) - 2 / 3) < 1e-16 and abs(oracle.shape(3, 1.0) - 1 / 6) < 1e-16
    for o in ORDERS:
        assert oracle.shape(o, (o + 1) / 2.0 + 1e-9) == 0.0
        assert oracle.shape(o, -0.3) == oracle.shape(o, 0.3)


def _linear_fields(grid, coef):
    """F_c[i,j,k] = a0 + a.(r_c) with r_c the Yee location of component c."""
    nx, ny, nz = grid
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    out = []
    for c in range(6):
        a0, a = coef[c]
        out.append(a0 + a[0] * (i + STAG[c][0]) + a[1] * (j + STAG[c][1]) + a[2] * (k + STAG[c][2]))
    return out


@pytest.mark.parametrize("order", ORDERS)
def test_gather_uniform_and_linear_exact(order):
    grid = (16, 12, 10)
    prm = OracleParams.make(grid, order=order)
    rng = np.random.default_rng(5)
    coef = [(rng.normal(), rng.normal(size=3)) for _ in range(6)]
    fields = _linear_fields(grid, coef)
    # away from the periodic seam (linear fields are not periodic)
    for _ in range(50):
        X = np.array([rng.uniform(3.0, n - 4.0) for n in grid])
        got = oracle.gather(prm, fields, X)
        exp = np.array([a0 + a @ X for a0, a in coef])
        np.testing.assert_allclose(got, exp, rtol=0, atol=5e-14)
    # uniform fields everywhere, including across the seam (config 1's fields)
    uni = [np.full((grid[2], grid[1], grid[0]), v) for v in (0.01, 0, 0, 0, 0, 0.1)]
    for X in ([0.1, 0.2, 0.3], [15.99, 11.99, 9.99], [0.0, 0.0, 0.0], [7.5, 0.49, 9.51]):
        np.testing.assert_allclose(oracle.gather(prm, uni, X), (0.01, 0, 0, 0, 0, 0.1), rtol=0, atol=1e-16)


@pytest.mark.parametrize("order", ORDERS)
def test_gather_one_hot_is_product_of_weights(order):
    grid = (8, 8, 8)
    prm = OracleParams.make(grid, order=order)
    rng = np.random.default_rng(7)
    for c in range(6):
        for _ in range(10):
            node = rng.integers(0, 8, 3)
            fields = [np.zeros((8, 8, 8)) for _ in range(6)]
            fields[c][node[2], node[1], node[0]] = 1.0
            X = node + np.array(STAG[c]) + rng.uniform(-1.2, 1.2, 3)
            got = oracle.gather(prm, fields, X)
            d = X - (node + np.array(STAG[c]))
            exp = np.prod(bspline_ref(order, d))
            assert abs(got[c] - exp) < 1e-15
            assert np.all(np.delete(got, c) == 0.0)            # no cross-talk between components


def test_gather_periodic_wrap_and_transposition():
    """A field varying only along one axis catches transposed indices / wrong strides."""
    grid = (8, 16, 24)
    prm = OracleParams.make(grid, order=2)
    k, j, i = np.meshgrid(np.arange(24), np.arange(16), np.arange(8), indexing="ij")
    for axis, idx, n in ((0, i, 8), (1, j, 16), (2, k, 24)):
        f = np.cos(2 * np.pi * idx / n)
        fields = [f.astype(float)] * 6
        X = np.array([2.3, 5.6, 17.2])
        Xs = X.copy()
        Xs[axis] += n                                          # periodic image
        g1, g2 = oracle.gather(prm, fields, X), oracle.gather(prm, fields, Xs)
        np.testing.assert_allclose(g1, g2, atol=1e-14)
        # TSC of cos: sum_i W(x-i) cos(2 pi i/n) = A(n) cos(2 pi x/n) only at nodes; check vs direct sum
        for c in range(6):
            xc = X[axis] - STAG[c][axis]
            nodes = np.arange(-4, n + 4)
            exp = (bspline_ref(2, xc - nodes) * np.cos(2 * np.pi * nodes / n)).sum()
            assert abs(g1[c] - exp) < 1e-14
