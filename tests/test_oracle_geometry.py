"""Pins for the oracle's metric, connection and geodesic integrator (O1, O7)."""
import math

import numpy as np
import pytest

from oracle_binding import make_params
from paper_2602_13198_b200 import workloads as wl


def _kerr(a=0.9375, hslope=0.3, **kw):
    p = wl.default_params()
    p.update(metric_kind=1, a_spin=a, hslope=hslope, r_max=1e3, r_horizon_stop=1.02 * (1 + math.sqrt(1 - a * a)))
    p.update(kw)
    return make_params(p)


def _flat(**kw):
    p = wl.default_params()
    p.update(metric_kind=0, hslope=1.0, r_max=1e3)
    p.update(kw)
    return make_params(p)


PTS = [(0.0, 0.4, 0.11, 0.3), (0.0, 1.7, 0.5, 1.0), (0.0, 3.0, 0.83, 5.0), (0.0, 0.9, 0.97, 2.0)]


@pytest.mark.parametrize("P", [_kerr(), _kerr(a=0.5, hslope=1.0), _flat()])
def test_inverse_and_determinant(olib, P):
    for x in PTS:
        g, gi = olib.gcov(P, x), olib.gcon(P, x)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-12)
        assert np.allclose(g, g.T)
        r = math.exp(x[1])
        th = math.pi * x[2] + 0.5 * (1 - P.hslope) * math.sin(2 * math.pi * x[2])
        dth = math.pi + (1 - P.hslope) * math.pi * math.cos(2 * math.pi * x[2])
        a = P.a_spin if P.metric_kind == 1 else 0.0
        closed = (r * r + a * a * math.cos(th) ** 2) * math.sin(th) * r * dth
        assert olib.gdet(P, x) == pytest.approx(closed, rel=1e-12)
        assert math.sqrt(-np.linalg.det(g)) == pytest.approx(closed, rel=1e-10)


def test_flat_limit_is_spherical_minkowski(olib):
    P = _flat()
    for x in PTS:
        r = math.exp(x[1]); th = math.pi * x[2]
        want = np.diag([-1.0, r * r, r * r * math.pi ** 2, r * r * math.sin(th) ** 2])
        assert np.allclose(olib.gcov(P, x), want, rtol=1e-14, atol=0)


def test_kerr_schild_textbook_components(olib):
    # independent retyping of the KS line element in (t,r,theta,phi), hslope=1 so that x2 = theta/pi
    a = 0.9375
    P = _kerr(a=a, hslope=1.0)
    x = (0.0, math.log(3.0), 0.3, 0.0)
    r, th = 3.0, math.pi * 0.3
    s, c = math.sin(th), math.cos(th)
    rho2 = r * r + a * a * c * c
    # ds^2 = -(1-2r/rho2)dt^2 + (4r/rho2)dt dr + (1+2r/rho2)dr^2 + rho2 dth^2
    #        + s^2[rho2 + a^2(1+2r/rho2)s^2]dphi^2 - (4 a r s^2/rho2) dt dphi - 2a(1+2r/rho2)s^2 dr dphi
    g = olib.gcov(P, x)
    J = np.array([1.0, r, math.pi, 1.0])
    gks = g / np.outer(J, J)
    assert gks[0, 0] == pytest.approx(-(1 - 2 * r / rho2))
    assert gks[0, 1] == pytest.approx(2 * r / rho2)
    assert gks[1, 1] == pytest.approx(1 + 2 * r / rho2)
    assert gks[2, 2] == pytest.approx(rho2)
    assert gks[3, 3] == pytest.approx(s * s * (rho2 + a * a * (1 + 2 * r / rho2) * s * s))
    assert gks[0, 3] == pytest.approx(-2 * a * r * s * s / rho2)
    assert gks[1, 3] == pytest.approx(-a * (1 + 2 * r / rho2) * s * s)


@pytest.mark.parametrize("P", [_kerr(), _flat()])
def test_analytic_metric_derivatives_vs_finite_differences(olib, P):
    d = 1e-4
    for x in PTS:
        dg = olib.dgcov(P, x)
        for al in range(4):
            def gat(s):
                y = list(x); y[al] += s
                return olib.gcov(P, y)
            fd = (-gat(2 * d) + 8 * gat(d) - 8 * gat(-d) + gat(-2 * d)) / (12 * d)
            scale = np.abs(olib.gcov(P, x)).max()
            assert np.allclose(dg[al], fd, atol=2e-10 * scale, rtol=1e-9)


def test_connection_definition_and_flat_textbook(olib):
    P = _kerr()
    x = PTS[1]
    G = olib.conn(P, x)
    assert np.allclose(G, np.transpose(G, (0, 2, 1)), atol=1e-14)
    gi, dg = olib.gcon(P, x), olib.dgcov(P, x)
    want = 0.5 * (np.einsum("mn,anb->mab", gi, dg) + np.einsum("mn,bna->mab", gi, dg) - np.einsum("mn,nab->mab", gi, dg))
    assert np.allclose(G, want, rtol=1e-12, atol=1e-14)
    # flat space in (ln r, theta/pi, phi): textbook spherical Christoffels transformed
    Pf = _flat()
    x = (0.0, 0.7, 0.31, 0.4)
    th = math.pi * 0.31
    Gf = olib.conn(Pf, x)
    assert Gf[1, 1, 1] == pytest.approx(1.0)                 # from r = e^x1
    assert Gf[1, 2, 2] == pytest.approx(-math.pi ** 2)       # Gamma^r_thth = -r  -> /r * pi^2
    assert Gf[1, 3, 3] == pytest.approx(-math.sin(th) ** 2)
    assert Gf[2, 1, 2] == pytest.approx(1.0)                 # Gamma^th_r th = 1/r -> * r
    assert Gf[2, 3, 3] == pytest.approx(-math.sin(th) * math.cos(th) / math.pi)
    assert Gf[3, 1, 3] == pytest.approx(1.0)
    assert Gf[3, 2, 3] == pytest.approx(math.pi * math.cos(th) / math.sin(th))
    assert abs(Gf[0]).max() == 0.0


def _null_k(olib, P, x, n3):
    """null k with unit coordinate-time component pointing along spatial coordinate direction n3"""
    g = olib.gcov(P, x)
    n = np.array(n3, dtype=float)
    A = g[0, 0]; B = 2 * g[0, 1:] @ n; Cc = n @ g[1:, 1:] @ n
    # A kt^2 + B kt + C = 0 ; future-directed root
    disc = B * B - 4 * A * Cc
    kt = (-B - math.sqrt(disc)) / (2 * A)
    return np.array([kt, *n])


def test_flat_space_rays_are_straight_lines(olib):
    P = _flat(r_max=50.0)
    x0 = np.array([0.0, math.log(2.0), 0.35, 0.3])
    k0 = _null_k(olib, P, x0, [0.3, 0.5, 0.9])
    tr = olib.geodesic(P, x0, k0)
    assert len(tr) > 50
    r = np.exp(tr[:, 1]); th = math.pi * tr[:, 2]; ph = tr[:, 3]
    X = np.stack([r * np.sin(th) * np.cos(ph), r * np.sin(th) * np.sin(ph), r * np.cos(th)], 1)
    d = X[-1] - X[0]; d /= np.linalg.norm(d)
    off = (X - X[0]) - np.outer((X - X[0]) @ d, d)
    assert np.abs(off).max() < 2e-3 * np.linalg.norm(X[-1] - X[0])
    # energy -k_t is exactly k^t here and must be conserved
    assert np.abs(tr[:, 4] / tr[0, 4] - 1).max() < 1e-3


def _drifts(olib, P, x0, n3, a):
    x0 = np.array(x0)
    k0 = _null_k(olib, P, x0, n3)
    tr = olib.geodesic(P, x0, k0)
    assert len(tr) > 100
    E, Lz, Q, KK = [], [], [], []
    for row in tr[:: max(1, len(tr) // 60)]:
        x, k = row[:4], row[4:]
        g = olib.gcov(P, x)
        kc = g @ k
        th = math.pi * x[2] + 0.35 * math.sin(2 * math.pi * x[2])
        dth = math.pi + 0.7 * math.pi * math.cos(2 * math.pi * x[2])
        kth = kc[2] / dth
        E.append(-kc[0]); Lz.append(kc[3]); KK.append((k @ kc) / (k[0] * k[0]))
        Q.append(kth ** 2 + math.cos(th) ** 2 * (kc[3] ** 2 / math.sin(th) ** 2 - a * a * kc[0] ** 2))
    E, Lz, Q, KK = map(np.array, (E, Lz, Q, KK))
    return (np.abs(E / E[0] - 1).max(), np.abs(Lz - Lz[0]).max() / max(abs(Lz[0]), abs(E[0])),
            np.abs(Q - Q[0]).max() / max(abs(Q[0]), E[0] ** 2), np.abs(KK).max())


def test_kerr_constants_of_motion(olib):
    """E = -k_t, L_z = k_phi, Carter's Q and k.k along integrated Kerr geodesics: conserved to the
    integrator's second-order truncation error -- small at the production step (energy, which
    sets the spectrum, to 2e-3), and shrinking ~4x per step halving (a wrong connection
    coefficient would not converge)."""
    a = 0.9375
    cases = (([0.2, 0.8, 1.5], [0.0, math.log(8.0), 0.45, 0.0]),
             ([-0.5, 0.1, 2.0], [0.0, math.log(6.0), 0.3, 1.0]),
             ([1.0, -0.4, -0.7], [0.0, math.log(12.0), 0.6, 2.0]))
    for n3, x0 in cases:
        d04 = _drifts(olib, _kerr(a=a, step_eps=0.04), x0, n3, a)
        d01 = _drifts(olib, _kerr(a=a, step_eps=0.01, verlet_tol=1e-8, verlet_maxit=30), x0, n3, a)
        d005 = _drifts(olib, _kerr(a=a, step_eps=0.005, verlet_tol=1e-9, verlet_maxit=30), x0, n3, a)
        assert d04[0] < 2e-3 and d04[1] < 5e-2 and d04[2] < 1e-1 and d04[3] < 3e-2, d04
        assert max(d01) < 3e-3, d01
        for hi, lo in zip(d01[1:], d005[1:]):
            assert lo < hi / 2.5 or hi < 1e-5, (d01, d005)


def test_push_is_second_order(olib):
    # halving the step must cut the one-step error by ~4x in x (Verlet position update)
    P = _kerr()
    x0 = np.array([0.0, math.log(7.0), 0.4, 0.0])
    k0 = _null_k(olib, P, x0, [0.5, 0.3, 0.4])
    G = olib.conn(P, x0)
    a0 = -np.einsum("mab,a,b->m", G, k0, k0)
    P.verlet_tol = 1e-13; P.verlet_maxit = 50

    def go(dl, n):
        x, k, a = x0, k0, a0
        for _ in range(n):
            x, k, a, it = olib.push(P, x, k, a, dl)
            assert it > 0
        return x
    ref = go(0.05 / 64, 64)
    e1 = np.abs(go(0.05, 1) - ref).max(); e2 = np.abs(go(0.025, 2) - ref).max()
    assert 3.0 < e1 / e2 < 5.5
