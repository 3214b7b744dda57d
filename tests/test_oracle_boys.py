"""Pins for the oracle's Boys function.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import special

from oracle import oracle as O

TGRID = [0.0, 1e-8, 1e-3, 0.5, 5.0, 20.0, 34.9, 35.0, 35.1, 100.0, 1e3, 6e3]


def boys_mp(m, T):
    mp.mp.dps = 50
    return mp.quad(lambda t: t ** (2 * m) * mp.e ** (-T * t * t), [0, 1])


def test_boys_zero():
    F = O.boys(8, 0.0)
    for m in range(9):
        assert F[m] == pytest.approx(1.0 / (2 * m + 1), rel=1e-15)


@pytest.mark.parametrize("T", TGRID)
def test_boys_vs_mpmath_quadrature(T):
    F = O.boys(8, T)
    for m in range(9):
        ref = float(boys_mp(m, mp.mpf(T)))
        assert abs(F[m] - ref) <= 2e-14 * abs(ref), (m, T, F[m], ref)


@pytest.mark.parametrize("T", [1e-3, 0.5, 5.0, 20.0, 34.9, 35.1, 100.0])
def test_boys_vs_gammainc(T):
    F = O.boys(8, T)
    for m in range(9):
        ref = special.gamma(m + 0.5) * special.gammainc(m + 0.5, T) / (2 * T ** (m + 0.5))
        assert F[m] == pytest.approx(ref, rel=5e-13)


@pytest.mark.parametrize("T", [0.3, 7.0, 34.0, 36.0, 200.0])
def test_boys_f0_erf_and_recursion(T):
    F = O.boys(8, T)
    assert F[0] == pytest.approx(0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T)), rel=1e-14)
    for m in range(8):  # (2m+1) F_m = 2T F_{m+1} + e^{-T}
        assert (2 * m + 1) * F[m] == pytest.approx(2 * T * F[m + 1] + math.exp(-T), rel=1e-13)


def test_boys_derivative_identity():
    # dF_m/dT = -F_{m+1}, central difference
    T, h = 3.0, 1e-4
    Fp, Fm, F0 = O.boys(8, T + h), O.boys(8, T - h), O.boys(8, T)
    for m in range(8):
        assert (Fp[m] - Fm[m]) / (2 * h) == pytest.approx(-F0[m + 1], rel=1e-7)


def test_boys_large_T_limit():
    T = 5e3
    F = O.boys(8, T)
    for m in range(9):
        dfact = 1.0
        for k in range(1, 2 * m, 2):
            dfact *= k
        assert F[m] == pytest.approx(dfact / 2 ** (m + 1) * math.sqrt(math.pi / T ** (2 * m + 1)), rel=1e-13)
