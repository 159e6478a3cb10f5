"""Pins for the oracle's fluid -> plasma state map and interpolation (O2; G2-G5)."""
import math

import numpy as np
import pytest

from oracle_binding import Oracle, make_params
from paper_2602_13198_b200 import workloads as wl

ME, MP = 9.1093826e-28, 1.67262171e-24


def test_sphere_field_is_one_gauss_everywhere_and_fluid_static():
    """G5: with x1 = ln r the uniform field along z has B^x1 = B0 cos(th)/r, B^x2 = -B0 sin(th)/(r th');
    the plasma state must report |B| = 1 G, n_e = 1e13, Theta_e = 10 at any interior point."""
    p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 32, 16, 1e4, 1, False)
    o = Oracle(p, prim)
    rng = np.random.default_rng(0)
    for _ in range(40):
        x = [0.0, p["startx"][1] + rng.uniform(0.02, 0.98) * 3.0, rng.uniform(0.05, 0.95), rng.uniform(0, 6.28)]
        s = o.plasma_at(x)
        assert not s["vacuum"]
        # multilinear interpolation of B^i ~ cos(th)/r between centres is not exact: 1 % on this grid
        assert s["B"] == pytest.approx(1.0, rel=1.5e-2)
        assert s["ne"] == pytest.approx(1e13, rel=1e-12)
        assert s["thetae"] == 10.0
        assert np.allclose(s["ucon"], [1, 0, 0, 0], atol=1e-15)
    # at a zone centre the field strength is exact
    xc = [0.0, p["startx"][1] + 10.5 * p["dx"][1], 4.5 * p["dx"][2], 0.3]
    assert o.plasma_at(xc)["B"] == pytest.approx(1.0, rel=1e-12)
    # vacuum outside the x1 range
    assert o.plasma_at([0.0, p["startx"][1] + 3.0 + 1e-9, 0.5, 0.0])["vacuum"]
    assert o.plasma_at([0.0, p["startx"][1] - 1e-9, 0.5, 0.0])["vacuum"]


def test_torus_four_velocity_and_field_are_normalised(olib):
    p, prim = wl.torus(48, 48, 1, Ns=1e4)
    o = Oracle(p, prim)
    P = make_params(p)
    rng = np.random.default_rng(1)
    n_hot = 0
    for _ in range(200):
        x = [0.0, math.log(rng.uniform(2.0, 40.0)), rng.uniform(0.02, 0.98), 0.0]
        s = o.plasma_at(x)
        g = olib.gcov(P, x)
        u, b = s["ucon"], s["bcon"]
        assert u @ g @ u == pytest.approx(-1.0, abs=1e-11)
        assert abs(u @ g @ b) <= 1e-11 * max(1.0, math.sqrt(abs(b @ g @ b)))
        # B [gauss] = sqrt(b.b) * c sqrt(4 pi RHO_unit)
        Bunit = 2.99792458e10 * math.sqrt(4 * math.pi * p["M_unit"] / p["L_unit"] ** 3)
        assert s["B"] == pytest.approx(math.sqrt(max(b @ g @ b, 0.0)) * Bunit, rel=1e-12)
        n_hot += s["thetae"] > 0.3
    assert n_hot > 10


def test_thetae_modes_reduce_to_textbook_ideal_gas():
    """G3: mode 1 is k T_e = (gam-1) u/n /(1+Tp/Te) for a single-temperature-ratio ideal gas; mode 2 with
    R_high = R_low = R reduces to Theta_e = (mp/me)(2/3)(u/rho)/(2+R)."""
    p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 8, 8, 1e4, 1, False)
    prim[..., 1] = 2.5e-3 * prim[..., 0]
    x = [0.0, p["startx"][1] + 1.3, 0.4, 0.0]
    o = Oracle(dict(p, thetae_mode=1, trat=3.0, gam_ad=5.0 / 3.0), prim)
    assert o.plasma_at(x)["thetae"] == pytest.approx((MP / ME) * (2.0 / 3.0) * 2.5e-3 / 4.0, rel=1e-12)
    o = Oracle(dict(p, thetae_mode=2, R_low=7.0, R_high=7.0), prim)
    assert o.plasma_at(x)["thetae"] == pytest.approx((MP / ME) * (2.0 / 3.0) * 2.5e-3 / 9.0, rel=1e-12)
    o = Oracle(dict(p, thetae_mode=2, R_low=1.0, R_high=40.0, thetae_max=0.05), prim)
    assert o.plasma_at(x)["thetae"] == 0.05        # clamp


def test_interpolation_is_exact_for_multilinear_fields_and_periodic_in_x3():
    p = wl.default_params()
    n1, n2, n3 = 6, 5, 8
    p.update(n1=n1, n2=n2, n3=n3, startx=[0, 0.2, 0.0, 0.0], dx=[1, 0.25, 0.2, 2 * math.pi / n3], r_max=100.0,
             thetae_mode=1)
    x1 = 0.2 + (np.arange(n1) + 0.5) * 0.25
    x2 = (np.arange(n2) + 0.5) * 0.2
    x3 = (np.arange(n3) + 0.5) * 2 * math.pi / n3
    X1, X2, X3 = np.meshgrid(x1, x2, x3, indexing="ij")
    prim = np.zeros((n1, n2, n3, 8))
    prim[..., 0] = 1.0 + 2.0 * X1 + 3.0 * X2 + 0.5 * X1 * X2
    prim[..., 1] = 0.01 * prim[..., 0] * (1.0 + np.cos(X3))
    o = Oracle(p, prim)
    gam, trat = p["gam_ad"], p["trat"]
    for x in ([0, 0.9, 0.37, 1.0], [0, 1.33, 0.61, 4.0]):
        s = o.plasma_at(x)
        rho = 1.0 + 2.0 * x[1] + 3.0 * x[2] + 0.5 * x[1] * x[2]
        assert s["ne"] * (MP + ME) / (p["M_unit"] / p["L_unit"] ** 3) == pytest.approx(rho, rel=1e-13)
    # periodic wrap: x3 and x3 + 2 pi give the same state; between the last and first centre it interpolates
    a = o.plasma_at([0, 0.9, 0.37, 0.1])
    b = o.plasma_at([0, 0.9, 0.37, 0.1 + 2 * math.pi])
    assert a["thetae"] == pytest.approx(b["thetae"], rel=1e-12)
    lo, hi = o.plasma_at([0, 0.9, 0.37, x3[-1]]), o.plasma_at([0, 0.9, 0.37, x3[0]])
    mid = o.plasma_at([0, 0.9, 0.37, 0.0])
    uu = lambda s: s["thetae"] * s["ne"]          # proportional to interpolated u
    assert uu(mid) == pytest.approx(0.5 * (uu(lo) + uu(hi)), rel=1e-12)
    # clamped (constant) beyond the outermost centres in x2, reflected across the axis
    assert o.plasma_at([0, 0.9, 0.01, 1.0])["ne"] == pytest.approx(o.plasma_at([0, 0.9, 0.1, 1.0])["ne"], rel=1e-13)
    assert o.plasma_at([0, 0.9, -0.03, 1.0])["ne"] == pytest.approx(o.plasma_at([0, 0.9, 0.03, 1.0])["ne"], rel=1e-13)
