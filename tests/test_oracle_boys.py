"""Pins for the oracle's Boys function (O2/O3 of DESIGN.md; PAPER.md:291, 295 use it through Rys moments)."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import special

TS = [0.0, 1e-8, 0.1, 5.0, 17.3, 29.9, 30.0, 30.1, 35.0, 100.0, 1e4, 1e7]


def boys_mp(m, T):
    mp.mp.dps = 40
    # the integrand lives at t ~ sqrt(m/T): give the quadrature break points there for large T
    pts = [0, 1]
    if T > 4:
        w = 1 / mp.sqrt(T)
        pts = sorted({mp.mpf(0), mp.mpf(1)} | {min(mp.mpf(1), k * w) for k in (1, 2, 4, 8, 16, 32)})
    if T > 1000:  # quadrature of so sharp a peak loses digits; use the incomplete-gamma identity at 40 digits
        T = mp.mpf(T)
        return mp.gammainc(m + mp.mpf(1) / 2, 0, T) / (2 * T ** (m + mp.mpf(1) / 2))
    return mp.quad(lambda t: t ** (2 * m) * mp.exp(-mp.mpf(T) * t * t), pts)


@pytest.mark.parametrize("T", TS)
def test_boys_vs_mpmath_quadrature(orc, T):
    F = orc.boys(14, T)
    for m in (0, 1, 2, 5, 9, 13, 14):
        ref = float(boys_mp(m, T))
        assert abs(F[m] - ref) <= 2e-14 * abs(ref) + 1e-300, (m, T, F[m], ref)


def test_boys_zero_and_gamma_form(orc):
    F = orc.boys(13, 0.0)
    for m in range(14):
        assert F[m] == pytest.approx(1.0 / (2 * m + 1), rel=1e-15)
    rng = np.random.default_rng(1)
    for T in rng.uniform(0.01, 80.0, 40):
        F = orc.boys(13, T)
        for m in range(14):
            ref = special.gammainc(m + 0.5, T) * special.gamma(m + 0.5) / (2.0 * T ** (m + 0.5))
            assert F[m] == pytest.approx(ref, rel=5e-13)
        assert F[0] == pytest.approx(0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T)), rel=1e-14)


def test_boys_switch_consistency(orc):
    lo, hi = orc.boys(13, 30.0), orc.boys(13, 30.0 + 1e-9)
    assert np.allclose(lo, hi, rtol=1e-9, atol=0)
    # recursion identity (2m+1) F_m = 2T F_{m+1} + exp(-T) on both branches
    for T in (3.0, 29.0, 31.0, 200.0):
        F = orc.boys(13, T)
        for m in range(13):
            assert (2 * m + 1) * F[m] == pytest.approx(2 * T * F[m + 1] + math.exp(-T), rel=2e-13)


@pytest.mark.parametrize("omega,rho,T", [(0.3, 0.7, 2.5), (0.3, 12.0, 40.0), (1.5, 0.2, 0.0), (0.05, 3.0, 90.0)])
def test_attenuated_boys_is_truncated_integral(orc, omega, rho, T):
    """s^{2m+1} F_m(s^2 T) = int_0^s t^{2m} exp(-T t^2) dt, s^2 = w^2/(w^2+rho)  (reading S8)."""
    mp.mp.dps = 40
    s = mp.sqrt(mp.mpf(omega) ** 2 / (mp.mpf(omega) ** 2 + mp.mpf(rho)))
    G = orc.boys_op(13, T, rho, omega)
    for m in (0, 1, 4, 13):
        ref = float(mp.quad(lambda t: t ** (2 * m) * mp.exp(-mp.mpf(T) * t * t), [0, s]))
        assert G[m] == pytest.approx(ref, rel=5e-14)
    # omega -> infinity is the full operator
    assert np.allclose(orc.boys_op(13, T, rho, 1e9), orc.boys(13, T), rtol=1e-13, atol=0)
