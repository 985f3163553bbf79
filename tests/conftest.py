"""pytest configuration: the `gpu` marker and shared helpers.

`-m "not gpu"` tests pin the oracle to closed forms / invariants / brute force and check
host logic + the C-ABI symbol table; `-m gpu` tests are the CUDA-vs-oracle parity tests.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size workloads (minutes)")


def bspline_ref(order: int, d):
    """Independent cardinal B-spline of degree `order` centred at 0, from scipy's
    BSpline.basis_element (library routine, NOT the oracle's formulas)."""
    from scipy.interpolate import BSpline
    knots = np.arange(order + 2, dtype=np.float64) - (order + 1) / 2.0
    b = BSpline.basis_element(knots, extrapolate=False)
    v = b(np.asarray(d, dtype=np.float64))
    return np.nan_to_num(v, nan=0.0)


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")
