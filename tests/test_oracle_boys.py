"""Pins for the oracle's Boys function F_m(T), eq. 18, against things that are not
the oracle: the incomplete-gamma closed form at 40 digits (mpmath), Gauss-Legendre quadrature of the
defining integral, F_m(0) = 1/(2m+1), the recursion identity and golden values (tests/golden/boys.txt)."""
import os

import mpmath
import numpy as np
import pytest

import oracle

MMAX = 12
T_GRID = [0.0, 1e-12, 1e-8, 1e-4, 0.01, 0.3, 1.0, 2.5, 5.0, 9.99, 10.0, 17.3, 24.999999, 25.0, 25.000001,
          30.0, 36.0, 50.0, 80.0, 120.0, 1e3, 1e5, 1e8]


def boys_mp(m, T):
    mpmath.mp.dps = 40
    if T == 0:
        return mpmath.mpf(1) / (2 * m + 1)
    T = mpmath.mpf(T)
    return mpmath.gammainc(m + mpmath.mpf(1) / 2, 0, T) / (2 * T ** (m + mpmath.mpf(1) / 2))


def test_boys_at_zero():
    F = oracle.boys(MMAX, 0.0)
    for m in range(MMAX + 1):
        assert F[m] == pytest.approx(1.0 / (2 * m + 1), rel=1e-15)


@pytest.mark.parametrize("T", T_GRID)
def test_boys_vs_incomplete_gamma_40_digits(T):
    F = oracle.boys(MMAX, T)
    for m in range(MMAX + 1):
        ref = boys_mp(m, T)
        assert abs(F[m] - ref) <= 2e-14 * abs(ref), (m, T, F[m], float(ref))


def test_boys_dense_sweep_across_branch_switch():
    worst = 0.0
    for T in np.concatenate([np.linspace(0, 40, 161), np.logspace(-6, 6, 49)]):
        F = oracle.boys(MMAX, float(T))
        for m in (0, 1, 6, 12):
            ref = boys_mp(m, float(T))
            worst = max(worst, float(abs(F[m] - ref) / abs(ref)))
    assert worst < 2e-14


def test_boys_vs_quadrature_of_definition():
    # eq. 18 integrated directly with 200-node Gauss-Legendre on [0,1]
    x, w = np.polynomial.legendre.leggauss(200)
    t = 0.5 * (x + 1.0)
    w = 0.5 * w
    for T in (0.0, 0.7, 8.0, 33.0, 90.0):
        F = oracle.boys(MMAX, T)
        for m in range(MMAX + 1):
            ref = np.sum(w * t ** (2 * m) * np.exp(-T * t * t))
            assert F[m] == pytest.approx(ref, rel=1e-11)


def test_boys_recursion_identity():
    # 2T F_{m+1} = (2m+1) F_m - exp(-T)
    for T in (0.2, 3.0, 24.0, 26.0, 60.0):
        F = oracle.boys(MMAX, T)
        for m in range(MMAX):
            lhs = 2 * T * F[m + 1]
            rhs = (2 * m + 1) * F[m] - np.exp(-T)
            assert lhs == pytest.approx(rhs, rel=1e-10, abs=1e-17)


def test_boys_golden_file():
    """tests/golden/boys.txt: 30-digit values written by tests/golden/make_boys_golden.py (mpmath)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "boys.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 20
    for m, T, val in rows:
        F = oracle.boys(int(m), float(T))
        assert F[int(m)] == pytest.approx(float(val), rel=2e-14)
