"""Pins for the oracle's emissivity, absorption and cross-sections (O3, O8)."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

HERE = os.path.dirname(__file__)
EE, CL, ME, HPL, SIGT = 4.80320680e-10, 2.99792458e10, 9.1093826e-28, 6.6260693e-27, 6.65245873e-25


def test_K2_against_scipy_and_paper_limit(olib):
    L = olib.L
    for th in (0.3, 0.5, 1.0, 3.7, 10.0, 55.0, 100.0):
        assert L.orc_K2_direct(th) == pytest.approx(special.kv(2, 1 / th), rel=1e-12)
        assert L.orc_K2_eval(th) == pytest.approx(special.kv(2, 1 / th), rel=2e-4)   # table interpolation
    # PAPER.md:61  K2(1/Theta) ~ 2 Theta^2 at large temperature
    for th in (100.001, 300.0, 1e3):
        assert L.orc_K2_eval(th) == 2 * th * th
        assert L.orc_K2_eval(th) == pytest.approx(special.kv(2, 1 / th), rel=3e-5)
    tab = olib.table(0)
    nodes = 0.3 * np.exp(np.arange(201) * math.log(100 / 0.3) / 200)
    assert np.allclose(tab, np.log(special.kv(2, 1 / nodes)), rtol=0, atol=1e-12)


def test_F_golden_values_and_asymptote(olib):
    L = olib.L
    asym = None
    for line in open(os.path.join(HERE, "golden", "F_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        a, b = line.split()
        if a == "asymptote":
            asym = float(b)
        else:
            assert L.orc_F_direct(float(a)) == pytest.approx(float(b), rel=2e-9)
    for K in (1e-9, 1e-12):
        assert L.orc_F_direct(K) / K ** (1 / 3) == pytest.approx(asym, rel=3e-3 if K > 1e-10 else 3e-4)
        assert L.orc_F_eval(K) / K ** (1 / 3) == pytest.approx(asym, rel=1e-9)
    # independent quadrature (scipy) of the same angle integral
    for K in (3e-5, 0.02, 7.0, 4e4):
        f = lambda t: math.sin(t) ** 2 * ((K / math.sin(t)) ** 0.5 + 2 ** (11 / 12) * (K / math.sin(t)) ** (1 / 6)) ** 2 \
            * math.exp(-(K / math.sin(t)) ** (1 / 3))
        want = 4 * math.pi * integrate.quad(f, 0, math.pi / 2, epsabs=0, epsrel=1e-12, limit=400)[0]
        assert L.orc_F_direct(K) == pytest.approx(want, rel=1e-9)
        assert L.orc_F_eval(K) == pytest.approx(want, rel=1.5e-3)   # log-log table interpolation error


def test_emissivity_total_power_fixes_the_prefactor(olib):
    """G1: int j_nu dnu dOmega = (4/3) sigma_T c U_B <gamma^2 beta^2> n_e (textbook synchrotron power)
    holds to the few-% accuracy of the Leung et al. fit only with sqrt(2)*pi in Eq. 3; the printed
    sqrt(2 pi) would give 0.57x."""
    L = olib.L
    ne, B = 1.0, 10.0
    for th in (3.0, 10.0, 30.0):
        nu0 = (2 / 9) * EE * B / (2 * math.pi * ME * CL) * th * th
        tot = integrate.quad(lambda ln: math.exp(ln) * L.orc_jnu_integrated(math.exp(ln), ne, th, B),
                             math.log(nu0 * 1e-6), math.log(nu0 * 1e6), epsrel=1e-8, limit=400)[0]
        g2b2 = integrate.quad(lambda g: (g * g - 1) * g * math.sqrt(g * g - 1) * math.exp(-(g - 1) / th), 1, 1 + 60 * th)[0] / \
            integrate.quad(lambda g: g * math.sqrt(g * g - 1) * math.exp(-(g - 1) / th), 1, 1 + 60 * th)[0]
        want = (4 / 3) * SIGT * CL * (B * B / (8 * math.pi)) * g2b2 * ne
        assert tot / want == pytest.approx(1.0, abs=0.04), (th, tot / want)
        assert abs(tot / want * math.sqrt(2 * math.pi) / (math.sqrt(2) * math.pi) - 1) > 0.3


def test_jnu_direct_matches_eq3_and_its_angle_integral(olib):
    L = olib.L
    nu, ne, th, B, sth = 2.3e11, 4e6, 12.0, 30.0, 0.8
    nus = (2 / 9) * EE * B / (2 * math.pi * ME * CL) * th * th * sth
    X = nu / nus
    want = math.sqrt(2) * math.pi * EE ** 2 * ne * nus / (3 * CL * special.kv(2, 1 / th)) * \
        (X ** 0.5 + 2 ** (11 / 12) * X ** (1 / 6)) ** 2 * math.exp(-X ** (1 / 3))
    assert L.orc_jnu(nu, ne, th, B, sth) == pytest.approx(want, rel=2e-4)
    ang = 4 * math.pi * integrate.quad(lambda t: math.sin(t) * L.orc_jnu(nu, ne, th, B, math.sin(t)), 0, math.pi / 2,
                                        epsrel=1e-10)[0]
    assert L.orc_jnu_integrated(nu, ne, th, B) == pytest.approx(ang, rel=2e-3)


def test_absorption_kirchhoff_and_paper_worked_value(olib):
    L = olib.L
    nu, ne, th, B = 1e9, 1e13, 100.0, 1.0
    j = L.orc_jnu(nu, ne, th, B, 1.0)
    Bnu = 2 * HPL * nu ** 3 / CL ** 2 / math.expm1(HPL * nu / (ME * CL * CL * th))
    na = L.orc_nu_alpha_abs(nu, ne, th, B, 1.0)
    assert na == pytest.approx(nu * j / Bnu, rel=1e-13)
    tau = na / nu * 1.0          # alpha_nu * L, L = 1 cm
    # "tau = alpha_nu L ~ 1e-4" for these numbers (order of magnitude only)
    assert 0.5e-4 < tau < 1e-3, tau


def _kn_textbook(e):
    # Rybicki & Lightman eq. 7.5 -- a different algebraic arrangement from PAPER.md Eq. 26
    l = math.log1p(2 * e)
    return 0.75 * ((1 + e) / e ** 3 * (2 * e * (1 + e) / (1 + 2 * e) - l) + l / (2 * e) - (1 + 3 * e) / (1 + 2 * e) ** 2)


def test_klein_nishina_total(olib):
    L = olib.L
    for e in (2e-3, 0.01, 0.3, 1.0, 7.0, 300.0, 1e5):
        assert L.orc_sigma_kn(e) == pytest.approx(_kn_textbook(e), rel=2e-8 if e > 5e-3 else 5e-6)
    for e in (1e-8, 1e-5, 9.99e-4):          # Eq. 27 regime
        assert L.orc_sigma_kn(e) == pytest.approx(1 - 2 * e, abs=6 * e * e)
    assert L.orc_sigma_kn(0.999e-3) == pytest.approx(L.orc_sigma_kn(1.001e-3), rel=1e-5)   # switch is continuous
    e = 1e6
    assert L.orc_sigma_kn(e) == pytest.approx(0.375 * (math.log(2 * e) + 0.5) / e, rel=1e-4)
    es = np.logspace(-6, 6, 200)
    v = np.array([L.orc_sigma_kn(x) for x in es])
    assert np.all(np.diff(v) < 0)


def test_hot_cross_section_limits_and_brute_force(olib):
    L = olib.L
    for e in (1e-3, 0.1, 3.0, 100.0):          # Theta -> 0  =>  sigma_KN(eps)
        assert L.orc_sigma_hot_direct(1e-6, e) == pytest.approx(L.orc_sigma_kn(e), rel=2e-5)
    for th in (0.01, 1.0, 30.0):               # eps -> 0 => sigma_T, since <1 - mu beta> = 1
        assert L.orc_sigma_hot_direct(th, 1e-11 / max(th, 1)) == pytest.approx(1.0, abs=1e-8)
    # brute-force Monte Carlo over an independently sampled Maxwell-Juttner distribution
    rng = np.random.default_rng(7)
    for th, e in ((0.5, 0.2), (4.0, 0.05), (10.0, 1.0), (100.0, 1e-3)):
        g = np.linspace(1, 1 + 80 * th, 400001)
        pdf = g * np.sqrt(g * g - 1) * np.exp(-(g - 1) / th)
        cdf = np.cumsum(pdf); cdf /= cdf[-1]
        gam = np.interp(rng.random(400000), cdf, g)
        beta = np.sqrt(1 - 1 / gam ** 2)
        mu = rng.uniform(-1, 1, gam.size)
        d = 1 - mu * beta
        vals = d * np.vectorize(_kn_textbook)(np.maximum(e * gam * d, 1e-9))
        mc, err = vals.mean(), vals.std() / math.sqrt(vals.size)
        assert abs(L.orc_sigma_hot_direct(th, e) - mc) < 4 * err + 2e-3 * mc, (th, e)
    # monotone decreasing in eps; table agrees with direct evaluation between nodes
    for th in (0.3, 4.0, 50.0):
        v = [L.orc_sigma_hot_direct(th, x) for x in (1e-4, 1e-2, 1.0, 100.0)]
        assert all(a > b for a, b in zip(v, v[1:]))
    for th, e in ((0.37, 0.011), (4.2, 3.3e-3), (11.0, 2.7), (230.0, 4.1e-5), (2e-3, 0.5)):
        assert L.orc_sigma_hot_eval(th, e) == pytest.approx(L.orc_sigma_hot_direct(th, e), rel=3e-3)
    assert L.orc_sigma_hot_eval(5.0, 1e-9) == 1.0             # Thomson shortcut
    assert L.orc_sigma_hot_eval(1e-5, 0.3) == L.orc_sigma_kn(0.3)
