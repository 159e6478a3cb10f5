"""Pins for the oracle's weights, per-zone counts and emission sampling (O4, O6; Eq. 2, 5-9)."""
import math

import numpy as np
import pytest
from scipy import integrate, special

from oracle_binding import Oracle, make_params
from paper_2602_13198_b200 import workloads as wl

EE, CL, ME, HPL = 4.80320680e-10, 2.99792458e10, 9.1093826e-28, 6.6260693e-27


def _jnu_eq3(nu, ne, th, B, s):
    """PAPER.md Eq. 3-4 retyped with scipy's K2 (prefactor sqrt(2) pi, G1)."""
    nus = (2 / 9) * EE * B / (2 * math.pi * ME * CL) * th * th * s
    X = nu / nus
    return math.sqrt(2) * math.pi * EE ** 2 * ne * nus / (3 * CL * special.kv(2, 1 / th)) * \
        (X ** 0.5 + 2 ** (11 / 12) * X ** (1 / 6)) ** 2 * math.exp(-X ** (1 / 3))


def _jnu_int(nu, ne, th, B):
    return 4 * math.pi * integrate.quad(lambda t: math.sin(t) * _jnu_eq3(nu, ne, th, B, math.sin(t)), 0, math.pi / 2,
                                        epsrel=1e-10)[0]


def test_expected_counts_sum_to_Ns_and_match_brute_force_quadrature_of_eq5():
    """Eq. 2 + Eq. 5 with G8: sum_i N_s,i = N_s when w_min = 0 (trapezoid on the same nodes => exact);
    one zone's N_s,i against scipy quadrature of Eq. 5 with Eq. 3 retyped above."""
    p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 4, 4, 5e4, 1, False, nu_min=1e9, nu_max=1e13)
    o = Oracle(p, prim)
    n = o.prepare()
    Nexp, qmax = o.zone_info()
    assert Nexp.sum() == pytest.approx(5e4, rel=1e-12)
    assert abs(n - 5e4) < 5 * math.sqrt(16 / 12) + 1            # integerisation adds < 1 per zone
    cnt = o.zone_counts()
    assert np.all((cnt == np.floor(Nexp)) | (cnt == np.floor(Nexp) + 1))
    nu_k, w_k = o.weight_table()
    lnw = lambda lnnu: np.interp(lnnu, np.log(nu_k), np.log(w_k))
    # zone (2,1): sqrt(-g) = r^3 pi sin(theta) in (ln r, x2, phi) coordinates
    i, j = 2, 1
    x1 = p["startx"][1] + (i + 0.5) * p["dx"][1]
    th = math.pi * (j + 0.5) * p["dx"][2]
    gdet = math.exp(3 * x1) * math.pi * math.sin(th)
    dV = p["dx"][1] * p["dx"][2] * p["dx"][3]
    dt = p["L_unit"] / CL
    f = lambda ln: _jnu_int(math.exp(ln), 1e13, 10.0, 1.0) / (HPL * math.exp(lnw(ln)))
    want = dt * gdet * dV * integrate.quad(f, math.log(1e9), math.log(1e13), epsrel=1e-8, limit=800,
                                            points=np.log(nu_k[1:-1:8]))[0]
    assert Nexp[i * 4 + j] == pytest.approx(want, rel=3e-3)      # trapezoid + table interpolation
    # Eq. 8 denominator is the maximum of F/w over the nodes
    assert qmax[i * 4 + j] > 0


def test_weight_is_eq2_at_a_node():
    p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 6, 6, 1e5, 1, False)
    o = Oracle(p, prim)
    o.prepare()
    nu_k, w_k = o.weight_table()
    k = 40
    x1 = p["startx"][1] + (np.arange(6) + 0.5) * p["dx"][1]
    th = math.pi * (np.arange(6) + 0.5) * p["dx"][2]
    vol = (np.exp(3 * x1)[:, None] * math.pi * np.sin(th)[None, :]).sum() * p["dx"][1] * p["dx"][2] * p["dx"][3]
    want = (p["L_unit"] / CL) * math.log(p["nu_max"] / p["nu_min"]) / (HPL * 1e5) * vol * _jnu_int(nu_k[k], 1e13, 10.0, 1.0)
    assert w_k[k] == pytest.approx(want, rel=2e-3)


def test_emitted_wavevector_is_null_with_the_sampled_energy_and_flat_counts_per_ln_nu(olib):
    p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 8, 8, 4e4, 3, False, nu_min=1e9, nu_max=1e12)
    o = Oracle(p, prim)
    n = o.prepare()
    P = make_params(p)
    lnnu, c2 = [], []
    for pid in range(0, n, 2):
        e = o.emit(pid)
        g = olib.gcov(P, e["x"])
        k = e["k"]
        assert abs(k @ g @ k) <= 1e-12 * k[0] ** 2
        eps = k[0]                                   # static fluid, flat space: -k.u = k^t
        assert e["E0"] == pytest.approx(eps, rel=1e-14)
        nu = eps * ME * CL * CL / HPL
        assert 1e9 <= nu <= 1e12
        lnnu.append(math.log(nu))
        # direction cosine to B (along z): physical components k_r = r k^1, k_th = r pi k^2
        r = math.exp(e["x"][1]); th = math.pi * e["x"][2]
        kz = r * k[1] * math.cos(th) - r * math.pi * k[2] * math.sin(th)
        c2.append((kz / eps) ** 2 if 3e10 < nu < 6e10 else np.nan)
    # Eq. 2's purpose: equal numbers per ln(nu) interval
    h, _ = np.histogram(lnnu, bins=12, range=(math.log(1e9), math.log(1e12)))
    chi2 = ((h - h.mean()) ** 2 / h.mean()).sum()
    assert chi2 < 35.0, (chi2, h)                    # 11 dof, p ~ 2e-4
    # Eq. 9: <cos^2> of the emission angle in a narrow band against quadrature of Eq. 3
    c2 = np.array(c2); c2 = c2[~np.isnan(c2)]
    nu_m = math.sqrt(3e10 * 6e10)
    num = integrate.quad(lambda t: math.sin(t) * math.cos(t) ** 2 * _jnu_eq3(nu_m, 1, 10.0, 1.0, math.sin(t)), 0, math.pi)[0]
    den = integrate.quad(lambda t: math.sin(t) * _jnu_eq3(nu_m, 1, 10.0, 1.0, math.sin(t)), 0, math.pi)[0]
    assert c2.mean() == pytest.approx(num / den, abs=4 * c2.std() / math.sqrt(c2.size) + 2e-3)


def test_tetrad_is_orthonormal_with_fixed_orientation(olib):
    a = 0.9375
    p = wl.default_params(); p.update(metric_kind=1, a_spin=a, hslope=0.3, r_max=1e3)
    P = make_params(p)
    rng = np.random.default_rng(5)
    for _ in range(30):
        x = np.array([0.0, math.log(rng.uniform(1.5, 30.0)), rng.uniform(0.03, 0.97), rng.uniform(0, 6)])
        g = olib.gcov(P, x)
        v = rng.normal(size=3) * 0.3 / np.sqrt(np.diag(g)[1:])
        # u^t from normalisation
        A = g[0, 0]; B = 2 * g[0, 1:] @ v; Cc = v @ g[1:, 1:] @ v + 1
        ut = (-B - math.sqrt(B * B - 4 * A * Cc)) / (2 * A)
        u = np.concatenate([[ut], v])
        trial = rng.normal(size=4)
        e = olib.tetrad(P, x, u, trial)
        eta = e @ g @ e.T
        assert np.allclose(eta, np.diag([-1, 1, 1, 1]), atol=1e-10)
        assert np.allclose(e[0], u)
        # e1 is the projected trial direction
        tp = trial + (trial @ g @ u) * u
        assert np.allclose(e[1], tp / math.sqrt(tp @ g @ tp), atol=1e-10)
        # fixed orientation (e3^m = eps^{mnrs} e0_n e1_r e2_s with eps^{0123} = -1/sqrt(-g)): det[e] sqrt(-g) = -1
        assert np.linalg.det(e) * olib.gdet(P, x) == pytest.approx(-1.0, abs=1e-9)
