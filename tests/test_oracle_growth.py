"""Pins for the oracle's growth functions and kick/drift factors.

The pins are independent of the oracle's ODE: Einstein-de Sitter closed forms, the Heath (1977)
integral D1 ~ E int da/(aE)^3 evaluated with scipy.quad, and the Bouchet et al. fit for D2.
"""
import math

import numpy as np
import pytest
from scipy.integrate import quad

OM = 0.3075


def heath_d1(om, a):
    e = lambda x: math.sqrt(om / x ** 3 + 1 - om)
    f = lambda x: quad(lambda y: 1.0 / (y * e(y)) ** 3, 0.0, x, epsabs=0, epsrel=1e-12)[0] * e(x)
    return f(a) / f(1.0)


def test_eds_closed_forms(oracle):
    for a in (0.05, 0.1, 0.5, 1.0):
        g = oracle.growth(1.0, a)
        assert g["D1"] == pytest.approx(a, rel=1e-9)
        assert g["D2"] == pytest.approx(-3.0 / 7.0 * a * a, rel=1e-9)
        assert g["f1"] == pytest.approx(1.0, rel=1e-9)
        assert g["f2"] == pytest.approx(2.0, rel=1e-9)
        assert g["E"] == pytest.approx(a ** -1.5, rel=1e-13)
        assert g["Gf"] == pytest.approx(a ** 1.5, rel=1e-9)
        assert g["gf"] == pytest.approx(1.5 * a ** 0.5, rel=1e-9)


@pytest.mark.parametrize("a", [0.1, 0.3, 0.55, 1.0])
def test_lcdm_d1_matches_heath_integral(oracle, a):
    g = oracle.growth(OM, a)
    assert g["D1"] == pytest.approx(heath_d1(OM, a), rel=2e-7)
    # f1 = dlnD1/dlna by central difference of the independent integral
    h = 1e-4
    f_fd = (math.log(heath_d1(OM, a * math.exp(h))) - math.log(heath_d1(OM, a * math.exp(-h)))) / (2 * h)
    assert g["f1"] == pytest.approx(f_fd, rel=1e-6)


def test_lcdm_printed_values(oracle):
    """Values quoted in SURVEY.md 8(c) R5 (re-derived here by the real oracle)."""
    g01, g1 = oracle.growth(OM, 0.1), oracle.growth(OM, 1.0)
    assert g01["D1"] == pytest.approx(0.127589, abs=2e-6)
    assert g1["f1"] == pytest.approx(0.519990, abs=2e-6)
    assert g01["f1"] == pytest.approx(0.998774, abs=2e-6)
    assert g1["D2"] / g1["D1"] ** 2 == pytest.approx(-0.432195, abs=2e-6)
    assert g01["D2"] / g01["D1"] ** 2 == pytest.approx(-0.428578, abs=2e-6)
    assert g1["f2"] == pytest.approx(1.054699, abs=2e-6)
    assert g01["f2"] == pytest.approx(1.997595, abs=2e-6)
    # Bouchet et al. (1995) fit D2 ~ -(3/7) D1^2 Om(a)^(-1/143): a separate literature pin
    assert g1["D2"] == pytest.approx(-3.0 / 7.0 * OM ** (-1.0 / 143.0), rel=5e-4)
    # growth index approximation f1 ~ Om(a)^0.55
    assert g1["f1"] == pytest.approx(OM ** 0.55, rel=1e-2)


def test_growth_ode_consistency(oracle):
    """gf = dGf/da and Gf = a^3 E dD1/da by finite differences of the oracle's own D1, Gf."""
    a, h = 0.4, 1e-4
    gp, gm, g0 = oracle.growth(OM, a + h), oracle.growth(OM, a - h), oracle.growth(OM, a)
    assert (gp["Gf"] - gm["Gf"]) / (2 * h) == pytest.approx(g0["gf"], rel=1e-6)
    assert a ** 3 * g0["E"] * (gp["D1"] - gm["D1"]) / (2 * h) == pytest.approx(g0["Gf"], rel=1e-6)
    assert g0["gf"] == pytest.approx(1.5 * OM * g0["D1"] / (a * a * g0["E"]), rel=1e-12)


def test_factors_eds_closed_forms(oracle):
    ai, ac, af = 0.2, 0.25, 0.3
    assert oracle.drift_factor(1.0, ai, ac, af) == pytest.approx((af - ai) / ac ** 1.5, rel=1e-9)
    assert oracle.kick_factor(1.0, ai, ac, af) == pytest.approx((af ** 1.5 - ai ** 1.5) / (1.5 * ac), rel=1e-9)
    # plain (Quinn et al.) integrals in EdS
    assert oracle.drift_factor(1.0, ai, ac, af, 1) == pytest.approx(2 * (ai ** -0.5 - af ** -0.5), rel=1e-10)
    assert oracle.kick_factor(1.0, ai, ac, af, 1) == pytest.approx(2 * (af ** 0.5 - ai ** 0.5), rel=1e-10)


def test_factor_families_agree_to_second_order(oracle):
    """FastPM and Quinn factors differ at O(da^2) relative when a_c is the interval midpoint."""
    rel = []
    for da in (0.04, 0.02, 0.01):
        ai, af = 0.5 - da / 2, 0.5 + da / 2
        d0, d1 = oracle.drift_factor(OM, ai, 0.5, af, 0), oracle.drift_factor(OM, ai, 0.5, af, 1)
        k0, k1 = oracle.kick_factor(OM, ai, 0.5, af, 0), oracle.kick_factor(OM, ai, 0.5, af, 1)
        rel.append((abs(d0 / d1 - 1), abs(k0 / k1 - 1)))
    for j in range(2):
        assert rel[0][j] < 3e-3
        assert rel[1][j] / rel[0][j] == pytest.approx(0.25, rel=0.1)
        assert rel[2][j] / rel[1][j] == pytest.approx(0.25, rel=0.1)


def test_zeldovich_flow_is_reproduced_exactly(oracle):
    """A Zel'dovich flow x = q + D1 psi, p = Gf psi with its exact force f = 1.5 Om D1 psi is a
    fixed point of the kick-drift-kick scheme with the growth-factor operators (R4 derivation)."""
    psi, q = 0.37, 3.0
    a0, a1 = 0.2, 0.45
    ah = math.sqrt(a0 * a1)
    g0, g1 = oracle.growth(OM, a0), oracle.growth(OM, a1)
    x, p = q + g0["D1"] * psi, g0["Gf"] * psi
    p += 1.5 * OM * g0["D1"] * psi * oracle.kick_factor(OM, a0, a0, ah)
    x += p * oracle.drift_factor(OM, a0, ah, a1)
    p += 1.5 * OM * g1["D1"] * psi * oracle.kick_factor(OM, ah, a1, a1)
    assert x == pytest.approx(q + g1["D1"] * psi, rel=1e-10)
    assert p == pytest.approx(g1["Gf"] * psi, rel=1e-9)
