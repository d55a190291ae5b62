"""Pins for the oracle Boys function (eq. 19; SURVEY.md §8(c) pins)."""
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import special

HERE = os.path.dirname(os.path.abspath(__file__))
LD_EPS = float(np.finfo(np.longdouble).eps)


def _mp_boys(m, T):
    """Independent library route: F_m(T) = Gamma(m+1/2) P(m+1/2, T) / (2 T^(m+1/2))."""
    mp.mp.dps = 50
    T = mp.mpf(T)
    if T == 0:
        return mp.mpf(1) / (2 * m + 1)
    return mp.gamma(m + mp.mpf(1) / 2) * mp.gammainc(m + mp.mpf(1) / 2, 0, T, regularized=True) / (2 * T ** (m + mp.mpf(1) / 2))


def _ld_to_mp(x):
    hi = float(x)
    lo = float(x - np.longdouble(hi))
    return mp.mpf(hi) + mp.mpf(lo)


def test_boys_at_zero(oracle):
    F = oracle.boys_ld(18, 0.0)
    for m in range(19):
        assert abs(float(F[m]) - 1.0 / (2 * m + 1)) < 1e-17


def test_boys_golden_25_digits(oracle):
    mp.mp.dps = 50
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "boys_25digit.txt")) if not l.startswith("#")]
    assert len(rows) == 11
    for m, T, v in rows:
        m, ex = int(m), mp.mpf(v)
        got = _ld_to_mp(oracle.boys_ld(18, float(T))[m])
        assert abs((got - ex) / ex) < 8 * LD_EPS, (m, T)
        # the stored value itself agrees with the independent library routine
        assert abs((_mp_boys(m, mp.mpf(T)) - ex) / ex) < mp.mpf(10) ** -23


def test_boys_F0_erf_closed_form(oracle):
    for T in [1e-6, 0.01, 0.3, 1.0, 4.0, 17.0, 35.0, 80.0, 119.9, 120.0, 500.0]:
        ex = 0.5 * np.sqrt(np.pi / T) * special.erf(np.sqrt(T))
        assert abs(float(oracle.boys_ld(10, T)[0]) - ex) <= 4e-16 * ex


def test_boys_dense_sweep_vs_mpmath(oracle):
    rng = np.random.default_rng(11)
    Ts = np.concatenate([rng.uniform(0, 40, 120), rng.uniform(40, 200, 60), [119.999, 120.0, 120.001, 1e-12, 1e-5]])
    for T in Ts:
        F = oracle.boys_ld(18, float(T))
        for m in (0, 1, 5, 9, 12, 14, 18):
            ex = _mp_boys(m, mp.mpf(float(T)))
            assert abs((_ld_to_mp(F[m]) - ex) / ex) < 40 * LD_EPS, (m, T)


def test_boys_recurrence_identity(oracle):
    """(2m+1) F_m = 2T F_{m+1} + e^{-T}: ties neighbouring orders together (a wrong index fails it)."""
    for T in [0.2, 3.0, 28.0, 75.0]:
        F = oracle.boys_ld(14, T)
        for m in range(14):
            lhs = (2 * m + 1) * F[m]
            rhs = 2 * np.longdouble(T) * F[m + 1] + np.exp(-np.longdouble(T))
            assert abs(float((lhs - rhs) / lhs)) < 1e-17


def test_boys_double_instantiation_close(oracle):
    for T in [0.0, 0.5, 12.0, 60.0, 130.0]:
        a, b = oracle.boys(16, T), oracle.boys_ld(16, T).astype(np.float64)
        assert np.max(np.abs(a - b) / b) < 2e-14
