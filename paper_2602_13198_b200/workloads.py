"""Seeded synthetic input generators (fluid grids + parameter dictionaries).

This module serves BOTH the CUDA library and the CPU oracle and therefore holds
none of the method's arithmetic (no emissivity, no sampling, no geodesics, no
tally): it only writes the *inputs* of the problem -- a fluid grid
``prim[n1][n2][n3][8]`` (rho, u, u~1, u~2, u~3, B1, B2, B3 in code units,
zone-major fp64) and a plain ``dict`` of parameters whose keys are the fields of
``gm_params`` (include/gpumonty_b200.h).  Each binding marshals the dict into
its own struct.

The grids stand in for the paper's workloads:
  cfg 0  optically thin synchrotron sphere   PAPER.md:219-240 (section 4.1)
  cfg 1  scattering synchrotron sphere       PAPER.md:258-268 (section 4.2)
  cfg 2  2-D Fishbone-Moncrief Kerr torus    PAPER.md:284 (FM torus, a=0.9375)
  cfg 3  3-D GRMHD-shaped perturbed torus    PAPER.md:284 (288x128x128 snapshot, absent)
  cfg 4  cfg 2 with density x1e3             PAPER.md:302-316 (N_s sweep)

Coordinates: x = (t, x1 = ln r, x2, x3 = phi) with
theta(x2) = pi*x2 + 0.5*(1-hslope)*sin(2*pi*x2)   (reading G28).
"""
from __future__ import annotations

import json
import math
import os

import numpy as np

# CGS constants, used only to express the inputs in code units (G0).
MP = 1.67262171e-24
ME = 9.1093826e-28
CL = 2.99792458e10
GNEWT = 6.6742e-8
MSUN = 1.989e33
SIGMA_T = 6.65245873e-25

NPRIM = 8
_CALIB_PATH = os.path.join(os.path.dirname(__file__), "workloads_calibrated.json")


def calibrated() -> dict:
    """Values written by oracle/calibrate.py (M_unit, w_min, bias0 per config)."""
    with open(_CALIB_PATH) as f:
        return json.load(f)


def default_params() -> dict:
    return dict(
        abi_version=3, seed=1, Ns_target=1e5,
        metric_kind=0, a_spin=0.0, hslope=1.0,
        startx=[0.0, 0.0, 0.0, 0.0], dx=[1.0, 1.0, 1.0, 2.0 * math.pi],
        n1=1, n2=1, n3=1,
        L_unit=1.0, M_unit=1.0,
        thetae_mode=0, thetae_fixed=10.0, trat=3.0, R_low=1.0, R_high=40.0,
        gam_ad=4.0 / 3.0, thetae_min=0.3, thetae_max=1000.0,
        nu_min=1e8, nu_max=1e16, w_min=0.0,
        step_eps=0.04, verlet_tol=1e-3, verlet_maxit=8,
        r_max=1.0, r_horizon_stop=0.0, max_steps=200000,
        scattering_on=0, nsc_max=4, bias0=1.0, bias_p_theta=0, bias_q_nsc=0,
        roulette=1e4,
        n_th=1, n_nu=200, nu_lo=1e8, nu_hi=1e24, fold_theta=1,
        emit_mode=0, bias_tune=0, bias_target=1.0,
    )


def theta_of_x2(x2, hslope):
    return math.pi * x2 + 0.5 * (1.0 - hslope) * np.sin(2.0 * math.pi * x2)


def dtheta_dx2(x2, hslope):
    return math.pi + (1.0 - hslope) * math.pi * np.cos(2.0 * math.pi * x2)


# --------------------------------------------------------------------------
# cfg 0 / 1 : uniform synchrotron sphere in flat space
# --------------------------------------------------------------------------
def sphere(n_e=1e13, thetae=10.0, B_gauss=1.0, R=1e3, n1=32, n2=16,
           Ns=1e5, seed=1, scattering=False, r_out=None, partial_sub=0, **over):
    """Uniform sphere, radius R cm, static fluid, field along z (PAPER.md:221-229,
    with the G5 correction of Eq. 31 for x1 = ln r).

    r_out (default R): outer edge of the grid.  With r_out > R the sphere surface falls inside a radial zone, as
    it does on the paper's grid.  partial_sub = 0: abrupt cutoff (a zone holds gas if its
    centre lies inside R); partial_sub = m: the paper's partial-cell treatment -- each zone is divided into an
    m x m sub-grid and its density is scaled by the fraction of sub-cell centres inside R (m = 5 in the paper)."""
    p = default_params()
    L_unit = 1.0
    M_unit = (MP + ME) * L_unit ** 3          # => Ne_unit = 1, rho == n_e
    B_unit = CL * math.sqrt(4.0 * math.pi * M_unit / L_unit ** 3)
    x1_0 = math.log(R * math.exp(-3.0))
    x1_end = math.log(R if r_out is None else r_out)
    dx1 = 3.0 / n1 if r_out is None else (x1_end - x1_0) / n1
    dx2 = 1.0 / n2
    p.update(seed=seed, Ns_target=float(Ns), metric_kind=0, a_spin=0.0, hslope=1.0,
             startx=[0.0, x1_0, 0.0, 0.0], dx=[1.0, dx1, dx2, 2.0 * math.pi],
             n1=n1, n2=n2, n3=1, L_unit=L_unit, M_unit=M_unit,
             thetae_mode=0, thetae_fixed=float(thetae),
             r_max=3.0 * R, r_horizon_stop=0.0,
             scattering_on=int(bool(scattering)), nsc_max=4,
             n_th=1, n_nu=200, nu_lo=1e8, nu_hi=1e24)
    x1 = x1_0 + (np.arange(n1) + 0.5) * dx1
    x2 = (np.arange(n2) + 0.5) * dx2
    r = np.exp(x1)[:, None]
    th = theta_of_x2(x2, 1.0)[None, :]
    dth = dtheta_dx2(x2, 1.0)[None, :]
    B0 = B_gauss / B_unit
    prim = np.zeros((n1, n2, 1, NPRIM))
    prim[..., 0] = n_e
    if r_out is not None:
        m = max(1, int(partial_sub))
        # fraction of the m x m sub-cell centres (in x1, x2) of each zone that lie inside R; r depends on x1 only
        sub = x1_0 + (np.arange(n1)[:, None] + (np.arange(m)[None, :] + 0.5) / m) * dx1
        frac = (np.exp(sub) < R).mean(axis=1)
        prim[..., 0] = n_e * frac[:, None, None]
    prim[..., 1] = 1e-3 * prim[..., 0]         # unused in thetae_mode 0
    prim[:, :, 0, 5] = B0 * np.cos(th) / r
    prim[:, :, 0, 6] = -B0 * np.sin(th) / (r * dth)
    p.update(over)
    return p, np.ascontiguousarray(prim)


def config0(Ns=1e5, seed=1, **over):
    p, prim = sphere(1e13, 10.0, 1.0, 1e3, 32, 16, Ns, seed, False)
    p["w_min"] = calibrated()["cfg0"]["w_min_per_Ns1"] / float(Ns)
    p.update(over)
    return p, prim


def config1(Ns=1e6, seed=1, tau_T=1e-2, **over):
    R = 1e3
    n_e = tau_T / (SIGMA_T * R)
    p, prim = sphere(n_e, 4.0, 1.0, R, 32, 16, Ns, seed, True)
    p.update(bias0=0.25 / tau_T, bias_p_theta=0, bias_q_nsc=2, nsc_max=4)
    p["w_min"] = calibrated()["cfg1"]["w_min_per_Ns1"] / float(Ns)
    p.update(over)
    return p, prim


# --------------------------------------------------------------------------
# cfg 2-4 : Fishbone-Moncrief torus in (modified) Kerr-Schild coordinates
# --------------------------------------------------------------------------
def _ks_gcov(r, th, a):
    """Kerr-Schild covariant metric in (t,r,theta,phi); arrays broadcast."""
    s, c = np.sin(th), np.cos(th)
    Sig = r * r + a * a * c * c
    f = 2.0 * r / Sig
    g = np.zeros(np.broadcast(r, th).shape + (4, 4))
    g[..., 0, 0] = -1.0 + f
    g[..., 0, 1] = g[..., 1, 0] = f
    g[..., 0, 3] = g[..., 3, 0] = -f * a * s * s
    g[..., 1, 1] = 1.0 + f
    g[..., 1, 3] = g[..., 3, 1] = -a * s * s * (1.0 + f)
    g[..., 2, 2] = Sig
    g[..., 3, 3] = s * s * (Sig + a * a * s * s * (1.0 + f))
    return g


def _mks_gcov(x1, x2, a, hslope):
    r = np.exp(x1)
    th = theta_of_x2(x2, hslope)
    g = _ks_gcov(r, th, a)
    J = np.ones(np.broadcast(r, th).shape + (4,))
    J[..., 1] = r
    J[..., 2] = dtheta_dx2(x2, hslope)
    return g * J[..., :, None] * J[..., None, :]


def _fm_l(r, a):
    """u_phi*u^t of the circular equatorial Kerr geodesic at r (Bardeen 1972):
    the constant FM angular momentum that puts the pressure maximum at r."""
    sr = math.sqrt(r)
    den = r ** 0.75 * math.sqrt(r ** 1.5 - 3.0 * sr + 2.0 * a)
    ut = (r ** 1.5 + a) / den
    uphi = (r * r - 2.0 * a * sr + a * a) / den
    return ut * uphi


def _fm_lnh(r, th, a, l):
    s, c = np.sin(th), np.cos(th)
    Del = r * r - 2.0 * r + a * a
    A = (r * r + a * a) ** 2 - Del * a * a * s * s
    Sig = r * r + a * a * c * c
    q = np.sqrt(1.0 + 4.0 * l * l * Sig * Sig * Del / (A * A * s * s))
    return 0.5 * np.log((1.0 + q) / (Sig * Del / A)) - 0.5 * q - 2.0 * a * r * l / A


def fm_torus_fields(x1c, x2c, a, hslope, r_in=6.0, r_pmax=12.0, gam=4.0 / 3.0, kappa=1e-3):
    """rho, u (unnormalised) and KS-frame u^t, u^phi of the FM torus at the given
    (x1, x2) points (Fishbone & Moncrief 1976)."""
    r = np.exp(x1c)
    th = theta_of_x2(x2c, hslope)
    l = _fm_l(r_pmax, a)
    lnh = _fm_lnh(r, th, a, l) - _fm_lnh(np.float64(r_in), np.float64(0.5 * math.pi), a, l)
    inside = (lnh > 0.0) & (r >= r_in)
    h = np.exp(np.where(inside, lnh, 0.0))
    rho = np.where(inside, ((h - 1.0) * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0)), 0.0)
    u = kappa * rho ** gam / (gam - 1.0)
    s, c = np.sin(th), np.cos(th)
    Del = r * r - 2.0 * r + a * a
    A = (r * r + a * a) ** 2 - Del * a * a * s * s
    Sig = r * r + a * a * c * c
    ut2 = 0.5 * (-1.0 + np.sqrt(1.0 + 4.0 * l * l * Sig * Sig * Del / (A * A * s * s)))
    uphi = 2.0 * a * r * np.sqrt(1.0 + ut2) / np.sqrt(A * Sig * Del) + np.sqrt(Sig / A) * np.sqrt(ut2) / s
    return rho, u, uphi, inside, l


def _torus_grid(n1, n2, n3, a, hslope, r_out=100.0):
    r_h = 1.0 + math.sqrt(1.0 - a * a)
    x1_0 = math.log(0.98 * r_h)
    dx1 = (math.log(r_out) - x1_0) / n1
    dx2 = 1.0 / n2
    dx3 = 2.0 * math.pi / n3
    return x1_0, dx1, dx2, dx3, r_h


def torus(n1=256, n2=256, n3=1, a=0.9375, hslope=0.3, Ns=1e7, seed=1,
          beta_target=100.0, rho_scale=1.0, perturb=False, **over):
    """Fishbone-Moncrief torus + poloidal loop field on an MKS grid.

    perturb=True applies the cfg-3 recipe: seeded log-normal (sigma 0.5,
    correlation 4 cells) density/energy perturbation and 30 % random field
    perturbations, periodic in x3.
    """
    from scipy import ndimage  # input generation only

    gam = 4.0 / 3.0
    x1_0, dx1, dx2, dx3, r_h = _torus_grid(n1, n2, n3, a, hslope)
    x1 = x1_0 + (np.arange(n1) + 0.5) * dx1
    x2 = (np.arange(n2) + 0.5) * dx2
    X1, X2 = np.meshgrid(x1, x2, indexing="ij")
    r = np.exp(X1)
    rho, u, uphi, inside, l = fm_torus_fields(X1, X2, a, hslope, gam=gam)
    rho_max = rho.max()
    rho = rho / rho_max
    u = u / rho_max
    g = _mks_gcov(X1, X2, a, hslope)                       # [n1,n2,4,4]
    gdet = np.sqrt(-np.linalg.det(g))
    gcon = np.linalg.inv(g)
    # fluid 4-velocity (KS == MKS for t,phi components; u^1 = u^2 = 0)
    AA = g[..., 0, 0]
    BB = 2.0 * g[..., 0, 3] * uphi
    CC = 1.0 + g[..., 3, 3] * uphi * uphi
    disc = np.maximum(BB * BB - 4.0 * AA * CC, 0.0)
    ut = np.where(inside, (-BB - np.sqrt(disc)) / (2.0 * AA), 0.0)
    alpha2 = -1.0 / gcon[..., 0, 0]
    ucon = np.zeros(X1.shape + (4,))
    ucon[..., 0] = ut
    ucon[..., 3] = np.where(inside, uphi, 0.0)
    utilde = np.zeros(X1.shape + (3,))
    for i in range(3):
        utilde[..., i] = np.where(inside, ucon[..., i + 1] + alpha2 * ut * gcon[..., 0, i + 1], 0.0)
    # vector potential at zone corners from corner-averaged density
    rho_pad = np.pad(rho, 1, mode="edge")
    rho_c = 0.25 * (rho_pad[:-1, :-1] + rho_pad[1:, :-1] + rho_pad[:-1, 1:] + rho_pad[1:, 1:])
    Aphi = np.maximum(rho_c - 0.2, 0.0)                    # [n1+1, n2+1]
    B1 = -(Aphi[:-1, 1:] - Aphi[:-1, :-1] + Aphi[1:, 1:] - Aphi[1:, :-1]) / (2.0 * dx2 * gdet)
    B2 = (Aphi[1:, :-1] - Aphi[:-1, :-1] + Aphi[1:, 1:] - Aphi[:-1, 1:]) / (2.0 * dx1 * gdet)
    # floors (atmosphere at rest in the normal-observer frame)
    rho = np.maximum(rho, 1e-6 * r ** -1.5)
    u = np.maximum(u, 1e-8 * r ** -2.5)

    def bsq_of(B1_, B2_, B3_, ucon_, g_):
        Bv = np.stack([B1_, B2_, B3_], axis=-1)
        ucov = np.einsum("...mn,...n->...m", g_, ucon_)
        bt = np.einsum("...i,...i->...", Bv, ucov[..., 1:])
        bcon = np.zeros(ucon_.shape)
        bcon[..., 0] = bt
        bcon[..., 1:] = (Bv + bt[..., None] * ucon_[..., 1:]) / ucon_[..., :1]
        bcov = np.einsum("...mn,...n->...m", g_, bcon)
        return np.einsum("...m,...m->...", bcon, bcov)

    # full ucon including atmosphere (normal observer: u^t = 1/alpha, u^i = -alpha g^ti)
    gamma = np.sqrt(1.0 + np.einsum("...i,...ij,...j->...", utilde, g[..., 1:, 1:], utilde))
    alpha = np.sqrt(alpha2)
    ucon_full = np.zeros(X1.shape + (4,))
    ucon_full[..., 0] = gamma / alpha
    for i in range(3):
        ucon_full[..., i + 1] = utilde[..., i] - gamma * alpha * gcon[..., 0, i + 1]
    bsq = bsq_of(B1, B2, np.zeros_like(B1), ucon_full, g)
    pmax = ((gam - 1.0) * u).max()
    bsqmax = bsq.max()
    norm = math.sqrt(2.0 * pmax / (beta_target * bsqmax))
    B1 *= norm
    B2 *= norm

    prim = np.zeros((n1, n2, n3, NPRIM))
    prim[..., 0] = rho[:, :, None]
    prim[..., 1] = u[:, :, None]
    for i in range(3):
        prim[..., 2 + i] = utilde[:, :, None, i]
    prim[..., 5] = B1[:, :, None]
    prim[..., 6] = B2[:, :, None]

    if perturb:
        def gfield(sd):
            rng = np.random.Generator(np.random.PCG64(sd))
            w = rng.standard_normal((n1, n2, n3))
            w = ndimage.gaussian_filter(w, sigma=4.0, mode=("reflect", "reflect", "wrap"))
            return (w - w.mean()) / w.std()
        gg = gfield(3)
        fac = np.exp(0.5 * gg - 0.125)
        prim[..., 0] *= fac
        prim[..., 1] *= fac
        for k, sd in enumerate((4, 5, 6)):
            gi = gfield(sd)
            if k < 2:
                prim[..., 5 + k] *= (1.0 + 0.3 * gi)
            else:
                # toroidal component seeded from the poloidal strength
                bp = np.sqrt(g[..., 1, 1, None] * prim[..., 5] ** 2 + g[..., 2, 2, None] * prim[..., 6] ** 2)
                prim[..., 7] = 0.3 * gi * bp / np.sqrt(g[..., 3, 3, None])

    prim[..., 0] *= rho_scale
    prim[..., 1] *= rho_scale
    prim[..., 5:8] *= math.sqrt(rho_scale)     # keeps plasma beta fixed

    p = default_params()
    Mbh = 4.1e6 * MSUN
    L_unit = GNEWT * Mbh / (CL * CL)
    p.update(seed=seed, Ns_target=float(Ns), metric_kind=1, a_spin=a, hslope=hslope,
             startx=[0.0, x1_0, 0.0, 0.0], dx=[1.0, dx1, dx2, dx3], n1=n1, n2=n2, n3=n3,
             L_unit=L_unit, M_unit=1e19,
             thetae_mode=2, R_low=1.0, R_high=40.0, gam_ad=gam,
             r_max=1e3, r_horizon_stop=1.02 * r_h,
             scattering_on=1, nsc_max=8, bias0=1.0, bias_p_theta=2, bias_q_nsc=0,
             n_th=6, n_nu=200, nu_lo=1e8, nu_hi=1e24, fold_theta=1)
    p.update(over)
    return p, np.ascontiguousarray(prim)


def _apply_calib(p, key, Ns):
    c = calibrated()[key]
    p["M_unit"] = c["M_unit"]
    p["bias0"] = c["bias0"]
    p["w_min"] = c["w_min_per_Ns1"] / float(Ns)


def config2(Ns=1e7, seed=1, n1=256, n2=256, **over):
    p, prim = torus(n1, n2, 1, Ns=Ns, seed=seed)
    _apply_calib(p, "cfg2", Ns)
    p.update(over)
    return p, prim


def config3(Ns=1e7, seed=1, n1=192, n2=128, n3=128, **over):
    p, prim = torus(n1, n2, n3, Ns=Ns, seed=seed, perturb=True)
    _apply_calib(p, "cfg3", Ns)
    p.update(over)
    return p, prim


def config4(Ns=1e6, seed=1, n1=256, n2=256, **over):
    p, prim = torus(n1, n2, 1, Ns=Ns, seed=seed, rho_scale=1e3)
    _apply_calib(p, "cfg4", Ns)
    p.update(over)
    return p, prim


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}
