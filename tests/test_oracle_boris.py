"""Pins of the oracle's Boris push and move.

Closed forms: |u| invariance for E=0, exact rotation angle 2 atan(|q/m||B|dt/(2 gamma)),
B=0 impulse, force-free E x B drift with dt^2 convergence, and the worked example stored in
tests/golden/boris_example.txt (SURVEY.md §8(c) step 4 pin (v)).
"""
import math
import os

import numpy as np

import oracle
from oracle import OracleParams


def test_u_norm_conserved_without_E():
    rng = np.random.default_rng(3)
    for _ in range(20):
        u = rng.normal(size=3) * 2.0
        B = rng.normal(size=3)
        u0 = np.linalg.norm(u)
        for _ in range(2000):
            u = oracle.boris(u, (0, 0, 0), B, -1.0, 0.5)
        assert abs(np.linalg.norm(u) - u0) / u0 < 1e-12


def test_exact_rotation_angle_and_sense():
    # q<0, Bz>0: counter-clockwise in the x-y plane; angle per step = 2 atan(|q/m| B dt / (2 gamma))
    for (qm, Bz, dt, u0) in ((-1.0, 0.1, 0.5, 0.01), (-1.0, 0.7, 0.3, 2.0), (2.0, 0.4, 0.5, 0.3)):
        u = np.array([u0, 0.0, 0.0])
        gamma = math.sqrt(1 + u0 * u0)
        un = oracle.boris(u, (0, 0, 0), (0, 0, Bz), qm, dt)
        ang = math.atan2(un[1], un[0])
        expect = 2.0 * math.atan(abs(qm) * Bz * dt / (2.0 * gamma))
        assert abs(abs(ang) - expect) < 1e-15
        assert (ang > 0) == (qm < 0)
        assert un[2] == 0.0
    # second-order agreement with the analytic gyrofrequency Omega = |q/m| B / gamma
    errs = []
    for dt in (0.5, 0.25, 0.125):
        un = oracle.boris((0.01, 0, 0), (0, 0, 0), (0, 0, 0.1), -1.0, dt)
        gamma = math.sqrt(1 + 1e-4)
        errs.append(abs(math.atan2(un[1], un[0]) - 0.1 / gamma * dt) / dt)
    assert 3.8 < errs[0] / errs[1] < 4.2 and 3.8 < errs[1] / errs[2] < 4.2


def test_B_zero_is_pure_impulse():
    rng = np.random.default_rng(4)
    for _ in range(20):
        u, E = rng.normal(size=3), rng.normal(size=3)
        qm, dt = rng.choice([-1.0, 1.0, 0.5]), rng.uniform(0.1, 0.5)
        un = oracle.boris(u, E, (0, 0, 0), qm, dt)
        np.testing.assert_allclose(un, u + qm * E * dt, rtol=4e-16, atol=4e-16)  # two half kicks: rounding order only


def test_parallel_B_component_untouched():
    un = oracle.boris((0.3, -0.2, 0.7), (0, 0, 0), (0, 0, 0.9), -1.0, 0.5)
    assert un[2] == 0.7
    un = oracle.boris((0.3, -0.2, 0.7), (0, 0, 0), (0.9, 0, 0), -1.0, 0.5)
    assert un[0] == 0.3


def test_ExB_drift_force_free_dt2():
    # config-1 fields: v_d = E x B / |B|^2 = (0,-0.1,0), independent of the charge sign.
    E, B = np.array([0.01, 0, 0]), np.array([0, 0, 0.1])
    vd = np.cross(E, B) / (B @ B)
    np.testing.assert_allclose(vd, (0, -0.1, 0), atol=1e-18)
    devs = []
    for dt in (0.5, 0.25, 0.125):
        for qm in (-1.0, 1.0):
            gd = 1.0 / math.sqrt(1.0 - vd @ vd)
            u = gd * vd
            worst = 0.0
            for _ in range(400):
                u = oracle.boris(u, E, B, qm, dt)
                v = u / math.sqrt(1 + u @ u)
                worst = max(worst, np.linalg.norm(v - vd))
        devs.append(worst)
    assert devs[0] < 1e-6                                        # SURVEY: 6.2e-7 at dt=0.5
    assert 3.5 < devs[0] / devs[1] < 4.5 and 3.5 < devs[1] / devs[2] < 4.5


def test_ExB_drift_from_rest_long_average():
    E, B = np.array([0.01, 0, 0]), np.array([0, 0, 0.1])
    u = np.zeros(3)
    acc = np.zeros(3)
    n = 100000
    for _ in range(n):
        u = oracle.boris(u, E, B, -1.0, 0.5)
        acc += u / math.sqrt(1 + u @ u)
    assert abs(acc[1] / n + 0.1) < 1e-3 * 0.1
    assert abs(acc[0] / n) < 1e-3 * 0.1


def test_worked_example(golden_dir):
    row = np.loadtxt(os.path.join(golden_dir, "boris_example.txt"))
    un = oracle.boris((0.01, -0.02, 0.005), (0.01, 0, 0), (0, 0, 0.1), -1.0, 0.5)
    np.testing.assert_allclose(un, row[0:3], rtol=0, atol=2e-17)
    assert abs(math.sqrt(1 + un @ un) - row[3]) < 1e-15
    prm = OracleParams.make((16, 16, 16), dt=0.5)
    X1 = oracle.move(prm, (5.0, 6.0, 7.0), un)
    np.testing.assert_allclose(X1 - (5.0, 6.0, 7.0), row[4:7], rtol=0, atol=2e-15)


def test_move_uses_cell_size_and_gamma():
    prm = OracleParams.make((16, 16, 16), cell=(0.5, 2.0, 1.0), dt=0.25)
    u = np.array([3.0, -4.0, 12.0])                               # gamma = sqrt(170)
    X1 = oracle.move(prm, (1.0, 2.0, 3.0), u)
    g = math.sqrt(170.0)
    np.testing.assert_allclose(X1, (1 + 3 / g * 0.25 / 0.5, 2 - 4 / g * 0.25 / 2.0, 3 + 12 / g * 0.25), atol=1e-15)
