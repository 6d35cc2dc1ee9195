"""Pins for the oracle's Boys function (oracle/pcm_oracle.c: orc_boys).

The paper gives no Boys evaluation scheme (PAPER.md:122 cites refs 19, 48 only); SURVEY.md 8(c1)
fixes the series + recursion reading.  Pins: values at T=0, the library closed form through the
regularised incomplete gamma function, Gauss-Legendre quadrature of the defining integral, the
recursion identity, agreement of the two branches across the switch, stored check values.
"""
import json
import math
import os

import numpy as np
import pytest
from scipy import special

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_checkvalues.json")))


def boys_gamma(n, T):
    """F_n(T) = Gamma(n+1/2) P(n+1/2, T) / (2 T^{n+1/2})  (library routine scipy.special.gammainc)."""
    if T == 0.0:
        return 1.0 / (2 * n + 1)
    a = n + 0.5
    return special.gamma(a) * special.gammainc(a, T) / (2.0 * T ** a)


def test_boys_at_zero(orc):
    F = orc.boys(4, 0.0)
    for n in range(5):
        assert F[n] == pytest.approx(1.0 / (2 * n + 1), rel=1e-15)


@pytest.mark.parametrize("T", [1e-8, 1e-3, 0.1, 0.5, 1.0, 3.3, 7.7, 12.5, 20.0, 29.9, 34.999, 35.0, 35.001, 40.0, 60.0,
                               100.0, 1e3, 1e5])
def test_boys_vs_incomplete_gamma(orc, T):
    F = orc.boys(4, T)
    for n in range(5):
        assert F[n] == pytest.approx(boys_gamma(n, T), rel=2e-14), (n, T)


@pytest.mark.parametrize("T", [0.0, 0.7, 5.0, 18.0, 33.0, 36.0, 50.0])
def test_boys_vs_gauss_legendre(orc, T):
    """the defining integral int_0^1 t^{2n} exp(-T t^2) dt by 64-point Gauss-Legendre"""
    x, w = np.polynomial.legendre.leggauss(64)
    t = 0.5 * (x + 1.0)
    F = orc.boys(4, T)
    for n in range(5):
        ref = 0.5 * np.sum(w * t ** (2 * n) * np.exp(-T * t * t))
        assert F[n] == pytest.approx(ref, rel=1e-13), (n, T)


def test_boys_recursion_identity(orc):
    """(2n+1) F_n = 2T F_{n+1} + exp(-T)"""
    for T in np.concatenate([np.linspace(0.0, 60.0, 241), [80.0, 200.0]]):
        F = orc.boys(4, float(T))
        for n in range(4):
            lhs = (2 * n + 1) * F[n]
            rhs = 2 * T * F[n + 1] + math.exp(-T)
            assert lhs == pytest.approx(rhs, rel=5e-14)


def test_boys_branches_agree_across_switch(orc):
    """series/downward (T<35) and erf/upward (T>=35) must be continuous at the switch to 1e-14"""
    lo, hi = orc.boys(4, np.nextafter(35.0, 0.0)), orc.boys(4, 35.0)
    for n in range(5):
        assert lo[n] == pytest.approx(hi[n], rel=1e-14)
    # and F_0 equals the libm-erf closed form on both sides
    for T in (25.0, 30.0, 34.0, 36.0, 45.0):
        assert orc.boys(4, T)[0] == pytest.approx(0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T)), rel=2e-15)


def test_boys_lower_orders_do_not_depend_on_nmax(orc):
    for T in (0.3, 9.0, 33.0, 41.0):
        F4 = orc.boys(4, T)
        for nmax in range(4):
            F = orc.boys(nmax, T)
            np.testing.assert_allclose(F, F4[:nmax + 1], rtol=3e-15)


def test_boys_stored_check_values(orc):
    for e in GOLD["boys"]:
        assert orc.boys(4, e["T"])[e["n"]] == pytest.approx(e["value"], rel=1e-14)
