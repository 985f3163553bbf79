"""Pins of the oracle's ENERGY-CONSERVING (Galerkin) gather, SURVEY.md §8(f)2 / §8(c) step 3 "alternative":
order o-1 along every axis a component is staggered on, order o along the others.  Expected values come from scipy's
BSpline (values and DERIVATIVES of the cardinal spline) and closed forms, never from the oracle.  The defining
property is pin (iv): a field that is the discrete gradient of a node potential is gathered as the exact gradient of
the order-o interpolation of that potential — which is what makes the scheme conserve energy."""
import numpy as np
import pytest

import oracle
from oracle import OracleParams
from conftest import bspline_ref

STAG = ((0.5, 0, 0), (0, 0.5, 0), (0, 0, 0.5), (0, 0.5, 0.5), (0.5, 0, 0.5), (0.5, 0.5, 0))
GRID = (8, 8, 8)


def _b0(d):
    """order-0 spline (top hat), right-continuous at -1/2 like the oracle's nearest-grid-point rule"""
    d = np.asarray(d, dtype=np.float64)
    return ((d >= -0.5) & (d < 0.5)).astype(np.float64)


def _ref_w(order, d):
    return _b0(d) if order == 0 else bspline_ref(order, d)


def _bspline_derivative(order, d):
    from scipy.interpolate import BSpline
    knots = np.arange(order + 2, dtype=np.float64) - (order + 1) / 2.0
    b = BSpline.basis_element(knots, extrapolate=False).derivative()
    return np.nan_to_num(b(np.asarray(d, dtype=np.float64)), nan=0.0)


def _fields(rng):
    return [rng.normal(size=GRID[::-1]) for _ in range(6)]


@pytest.mark.parametrize("order", (1, 2, 3))
def test_uniform_field_is_reproduced(order):
    prm = OracleParams.make(GRID, order=order, gather=1)
    F = [np.full(GRID[::-1], v) for v in (0.3, -1.25, 2.0, 0.7, -0.1, 5.0)]
    rng = np.random.default_rng(1)
    for X in rng.uniform(0, 8, (50, 3)):
        np.testing.assert_allclose(oracle.gather(prm, F, X), (0.3, -1.25, 2.0, 0.7, -0.1, 5.0), rtol=0, atol=1e-14)


@pytest.mark.parametrize("order", (1, 2, 3))
def test_matches_the_definition_with_scipy_splines(order):
    """F_c(X) = sum F[i,j,k] prod_a W_{o_a}(X_a - (i_a + s_a)) with o_a = o-1 on staggered axes, brute force over the
    whole periodic grid with scipy's spline values (minimum-image distance)."""
    prm = OracleParams.make(GRID, order=order, gather=1)
    rng = np.random.default_rng(2)
    F = _fields(rng)
    for X in rng.uniform(0, 8, (12, 3)):
        got = oracle.gather(prm, F, X)
        for c in range(6):
            w = []
            for a in range(3):
                oa = order - 1 if STAG[c][a] else order
                d = X[a] - (np.arange(GRID[a]) + STAG[c][a])
                d = d - GRID[a] * np.round(d / GRID[a])
                w.append(_ref_w(oa, d))
            exp = np.einsum("kji,k,j,i->", F[c], w[2], w[1], w[0])
            assert abs(got[c] - exp) < 1e-13, (order, c)


def test_differs_from_the_momentum_conserving_gather_only_on_staggered_axes():
    """With a field that varies along x only, Ey (unstaggered along x) is gathered identically by both variants, Ex
    (staggered along x) is not."""
    rng = np.random.default_rng(3)
    prof = rng.normal(size=8)
    F = [np.broadcast_to(prof[None, None, :], GRID[::-1]).copy() for _ in range(6)]
    X = (3.3, 4.1, 2.7)
    a = oracle.gather(OracleParams.make(GRID, order=2, gather=0), F, X)
    b = oracle.gather(OracleParams.make(GRID, order=2, gather=1), F, X)
    assert max(abs(a[c] - b[c]) for c in (1, 2, 3)) < 1e-14
    assert abs(a[0] - b[0]) > 1e-3 and abs(a[4] - b[4]) > 1e-3 and abs(a[5] - b[5]) > 1e-3


@pytest.mark.parametrize("order", (1, 2, 3))
def test_gradient_of_a_potential_is_gathered_exactly(order):
    """(iv) E = -grad_h(phi) on the Yee grid (E_x[i+1/2,j,k] = -(phi[i+1,j,k] - phi[i,j,k])/dx, ...) is gathered as
    -grad of phi_o(X) = sum phi[ijk] W_o W_o W_o, evaluated with scipy's spline and spline derivative."""
    cell = (1.0, 0.5, 2.0)
    prm = OracleParams.make(GRID, cell=cell, order=order, gather=1)
    rng = np.random.default_rng(4)
    phi = rng.normal(size=GRID[::-1])
    E = [-(np.roll(phi, -1, 2 - a) - phi) / cell[a] for a in range(3)]
    F = E + [np.zeros(GRID[::-1])] * 3
    for X in rng.uniform(0, 8, (20, 3)):
        if order == 1 and np.any(np.abs(X - np.round(X)) < 1e-6):
            continue                      # W_1 has a kink at the nodes
        got = oracle.gather(prm, F, X)[:3]
        w, dw = [], []
        for a in range(3):
            d = X[a] - np.arange(GRID[a])
            d = d - GRID[a] * np.round(d / GRID[a])
            w.append(bspline_ref(order, d))
            dw.append(_bspline_derivative(order, d) / cell[a])
        exp = (-np.einsum("kji,k,j,i->", phi, w[2], w[1], dw[0]),
               -np.einsum("kji,k,j,i->", phi, w[2], dw[1], w[0]),
               -np.einsum("kji,k,j,i->", phi, dw[2], w[1], w[0]))
        np.testing.assert_allclose(got, exp, rtol=0, atol=1e-12)


def test_step_uses_the_selected_gather():
    """Oracle.step with gather=1: B = 0, u_new - u = (q/m) E_ec(X) dt with E_ec from the pinned gather above."""
    rng = np.random.default_rng(5)
    F = _fields(rng)
    for c in (3, 4, 5):
        F[c][:] = 0.0
    X = rng.uniform(0, 8, (3, 30))
    u0 = rng.normal(0, 0.1, (3, 30))
    orc = oracle.Oracle(GRID, dt=0.25, order=2, gather=1)
    orc.load_particles(*X, *u0, np.ones(30))
    orc.set_fields(F)
    assert orc.step(1) == 0
    P = orc.particles()
    prm = OracleParams.make(GRID, dt=0.25, order=2, gather=1)
    for p in range(30):
        E = oracle.gather(prm, F, X[:, p])[:3]
        np.testing.assert_allclose((P["ux"][p], P["uy"][p], P["uz"][p]), u0[:, p] - E * 0.25, rtol=0, atol=1e-15)
