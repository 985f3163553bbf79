"""Pins of the oracle's Esirkepov deposit and re-bucketing.

Independent checks: discrete continuity with rho built from scipy's B-splines, a six-path
brute-force deposition written here in numpy (no oracle code), the total-current identity,
the axis-parallel closed form, and the worked example of tests/golden/esirkepov_example.txt.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from oracle import OracleParams
from conftest import bspline_ref

ORDERS = (1, 2, 3)


def rho_ref(order, grid, cell, X, qw):
    """rho[k,j,i] = sum_p qw S(Xx-i)S(Xy-j)S(Xz-k)/V with scipy B-splines, periodic."""
    nx, ny, nz = grid
    V = cell[0] * cell[1] * cell[2]
    out = np.zeros((nz, ny, nx))
    for p in range(len(qw)):
        ws = []
        for a, n in enumerate(grid):
            nodes = np.arange(-8, n + 8)
            w = bspline_ref(order, X[p, a] - nodes)
            folded = np.zeros(n)
            np.add.at(folded, nodes % n, w)
            ws.append(folded)
        out += qw[p] / V * ws[2][:, None, None] * ws[1][None, :, None] * ws[0][None, None, :]
    return out


def div_J(J, cell):
    Jx, Jy, Jz = J
    return ((Jx - np.roll(Jx, 1, axis=2)) / cell[0] + (Jy - np.roll(Jy, 1, axis=1)) / cell[1]
            + (Jz - np.roll(Jz, 1, axis=0)) / cell[2])


def random_moves(rng, grid, n, dmax=0.5):
    X0 = rng.uniform(0, 1, (n, 3)) * np.array(grid)
    X1 = X0 + rng.uniform(-dmax, dmax, (n, 3))
    qw = rng.choice([-1.0, 1.0], n) * rng.uniform(0.5, 2.0, n)
    return X0, X1, qw


@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("grid,cell,dmax", [((4, 4, 4), (1.0, 1.0, 1.0), 0.5), ((8, 6, 5), (0.5, 2.0, 1.25), 0.95)])
def test_continuity(order, grid, cell, dmax):
    rng = np.random.default_rng(100 + order)
    dt = 0.37
    prm = OracleParams.make(grid, cell=cell, dt=dt, order=order)
    X0, X1, qw = random_moves(rng, grid, 40, dmax)
    J = None
    for p in range(40):
        J = oracle.deposit(prm, qw[p], X0[p], X1[p], J)
    drho = (rho_ref(order, grid, cell, X1, qw) - rho_ref(order, grid, cell, X0, qw)) / dt
    res = np.abs(drho + div_J(J, cell)).max() / np.abs(drho).max()
    assert res < 1e-12
    # the oracle's own rho agrees with the scipy one (pins orc_rho, used for the GPU residual)
    np.testing.assert_allclose(oracle.rho(prm, X0[:, 0], X0[:, 1], X0[:, 2], qw),
                               rho_ref(order, grid, cell, X0, qw), rtol=0, atol=1e-13)


def six_path_bruteforce(order, grid, cell, dt, qw, X0, X1):
    """Average over the 6 orderings of axis-aligned legs; each leg deposits the 1-D
    prefix-summed charge differences along its axis with the transverse weights frozen."""
    n = np.array(grid)
    V = np.prod(cell)
    J = [np.zeros((grid[2], grid[1], grid[0])) for _ in range(3)]
    nodes = [np.arange(-8, g + 8) for g in grid]

    def S(a, x):
        return bspline_ref(order, x - nodes[a])

    for perm in itertools.permutations(range(3)):
        cur = np.array(X0, dtype=float)
        for a in perm:
            nxt = cur.copy()
            nxt[a] = X1[a]
            dS = S(a, nxt[a]) - S(a, cur[a])
            flux = -(qw / V) * (cell[a] / dt) * np.cumsum(dS)          # at node+1/2 along a
            b1, b2 = [b for b in range(3) if b != a]
            T1, T2 = S(b1, cur[b1]), S(b2, cur[b2])
            for ia, fa in zip(nodes[a], flux):
                if fa == 0.0:
                    continue
                for i1, t1 in zip(nodes[b1], T1):
                    if t1 == 0.0:
                        continue
                    for i2, t2 in zip(nodes[b2], T2):
                        if t2 == 0.0:
                            continue
                        idx = [0, 0, 0]
                        idx[a], idx[b1], idx[b2] = ia % n[a], i1 % n[b1], i2 % n[b2]
                        J[a][idx[2], idx[1], idx[0]] += fa * t1 * t2 / 6.0
            cur = nxt
    return J


@pytest.mark.parametrize("order", ORDERS)
def test_six_path_bruteforce_4cubed(order):
    grid, cell, dt = (4, 4, 4), (1.0, 1.0, 1.0), 0.5
    prm = OracleParams.make(grid, cell=cell, dt=dt, order=order)
    rng = np.random.default_rng(200 + order)
    X0, X1, qw = random_moves(rng, grid, 12, 0.5)
    for p in range(12):
        got = oracle.deposit(prm, qw[p], X0[p], X1[p])
        ref = six_path_bruteforce(order, grid, cell, dt, qw[p], X0[p], X1[p])
        scale = max(np.abs(r).max() for r in ref)
        for g, r in zip(got, ref):
            assert np.abs(g - r).max() < 1e-13 * max(scale, 1e-30)


@pytest.mark.parametrize("order", ORDERS)
def test_total_current_identity(order):
    grid, cell, dt = (8, 8, 8), (0.5, 1.0, 2.0), 0.4
    prm = OracleParams.make(grid, cell=cell, dt=dt, order=order)
    rng = np.random.default_rng(300 + order)
    X0, X1, qw = random_moves(rng, grid, 30, 0.9)
    V = np.prod(cell)
    for p in range(30):
        J = oracle.deposit(prm, qw[p], X0[p], X1[p])
        for a in range(3):
            assert abs(J[a].sum() * V - qw[p] * (X1[p, a] - X0[p, a]) * cell[a] / dt) < 2e-14 * abs(qw[p]) / dt * max(cell)


@pytest.mark.parametrize("order", ORDERS)
def test_axis_parallel_closed_form(order):
    grid, dt = (8, 8, 8), 0.5
    prm = OracleParams.make(grid, dt=dt, order=order)
    X0 = np.array([3.3, 4.6, 2.2])
    for a in range(3):
        X1 = X0.copy()
        X1[a] += 0.45
        J = oracle.deposit(prm, -1.5, X0, X1)
        others = [b for b in range(3) if b != a]
        for b in others:
            assert np.all(J[b] == 0.0)
        # summed along the direction of motion: q w v x transverse area weights
        axis_np = 2 - a
        line = J[a].sum(axis=axis_np)
        nodes = np.arange(8)
        Tb = [bspline_ref(order, X0[b] - nodes) for b in others]          # b ascending: (x,y),(x,z),(y,z)
        exp = -1.5 * 0.45 / dt * np.outer(Tb[1], Tb[0])                    # [higher axis, lower axis]
        np.testing.assert_allclose(line, exp, rtol=0, atol=1e-14)


def test_worked_example(golden_dir):
    rows = np.loadtxt(os.path.join(golden_dir, "esirkepov_example.txt"))
    for row in rows:
        order = int(row[0])
        prm = OracleParams.make((8, 8, 8), dt=0.5, order=order)
        J = oracle.deposit(prm, -1.0, (3.25, 4.5, 2.75), (3.5, 4.375, 3.125))
        got = (J[0][2, 4, 3], J[0][3, 4, 3], J[1][3, 4, 3], J[2][2, 4, 3])
        np.testing.assert_allclose(got, row[1:5], rtol=0, atol=3e-16)
        np.testing.assert_allclose([j.sum() for j in J], row[5:8], rtol=0, atol=1e-14)


def test_zero_displacement_deposits_nothing():
    for order in ORDERS:
        prm = OracleParams.make((8, 8, 8), order=order)
        J = oracle.deposit(prm, 1.0, (1.2, 3.4, 5.6), (1.2, 3.4, 5.6))
        assert all(np.all(j == 0.0) for j in J)


def test_wrap_and_bucket():
    prm = OracleParams.make((16, 16, 16), supercell=(8, 8, 4))
    X, sc = oracle.wrap_and_bucket(prm, (-0.25, 16.5, 7.999))
    np.testing.assert_allclose(X, (15.75, 0.5, 7.999))
    assert sc == 1 + 2 * (0 + 2 * 1)
    X, sc = oracle.wrap_and_bucket(prm, (-1e-18, 8.0, 15.999999))
    assert X[0] == 0.0 and sc == 0 + 2 * (1 + 2 * 3)
    X, sc = oracle.wrap_and_bucket(prm, (15.999999999, 7.9999999, 4.0))
    assert sc == 1 + 2 * (0 + 2 * 1)
