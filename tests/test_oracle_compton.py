"""Pins for the oracle's Compton event (O8; G24, G25)."""
import math

import numpy as np
import pytest
from scipy import integrate, special


def test_maxwell_juttner_sampler_moments(olib):
    """<gamma> = 3 Theta + K1(1/Theta)/K2(1/Theta); <gamma^2> by quadrature of gamma^2 beta exp(-gamma/Theta)."""
    n = 200000
    for th in (0.05, 0.5, 4.0, 30.0):
        g = olib.sample_mj(th, 11, n)
        assert np.all(g >= 1.0)
        want1 = 3 * th + special.kve(1, 1 / th) / special.kve(2, 1 / th)
        pdf = lambda x: x * math.sqrt(x * x - 1) * math.exp(-(x - 1) / th)
        hi = 1 + 80 * th
        want2 = integrate.quad(lambda x: x * x * pdf(x), 1, hi)[0] / integrate.quad(pdf, 1, hi)[0]
        assert g.mean() == pytest.approx(want1, abs=5 * g.std() / math.sqrt(n))
        assert (g * g).mean() == pytest.approx(want2, abs=5 * (g * g).std() / math.sqrt(n))


def test_scattered_photon_is_null_and_thomson_amplification(olib):
    """eps << 1/gamma: <eps_out/eps> = 1 + (4/3) <gamma^2 beta^2> (textbook inverse-Compton gain)."""
    n = 200000
    for th in (0.2, 2.0):
        e, c, kk = olib.compton_sample(th, 1e-9, 5, n)
        assert not np.isnan(e).any()
        assert np.max(np.abs(kk)) < 1e-10
        pdf = lambda x: x * math.sqrt(x * x - 1) * math.exp(-(x - 1) / th)
        hi = 1 + 80 * th
        g2b2 = integrate.quad(lambda x: (x * x - 1) * pdf(x), 1, hi)[0] / integrate.quad(pdf, 1, hi)[0]
        A = e / 1e-9
        assert A.mean() == pytest.approx(1 + 4 / 3 * g2b2, abs=5 * A.std() / math.sqrt(n))


def test_cold_electrons_reproduce_klein_nishina_and_thomson_angular_laws(olib):
    """Theta -> 0: electron at rest, so the event samples the differential Compton cross-section directly."""
    n = 200000
    # Thomson regime (eps' < 1e-4, G25): <mu> = 0, <mu^2> = 2/5, no energy change
    e, c, kk = olib.compton_sample(1e-10, 1e-6, 9, n)
    assert e / 1e-6 == pytest.approx(1.0, abs=1e-4)
    assert c.mean() == pytest.approx(0.0, abs=5 * c.std() / math.sqrt(n))
    assert (c * c).mean() == pytest.approx(0.4, abs=5 * (c * c).std() / math.sqrt(n))
    # Klein-Nishina: d sigma/d mu ~ r^2 (r + 1/r - 1 + mu^2), r = 1/(1 + eps (1 - mu))
    for eps in (0.3, 2.0, 50.0):
        e, c, kk = olib.compton_sample(1e-10, eps, 9, n)
        assert np.max(np.abs(kk)) < 1e-10
        # Compton formula ties energy to angle
        assert np.allclose(e, eps / (1 + eps * (1 - c)), rtol=5e-4)   # beta ~ sqrt(2 Theta) ~ 1e-5
        ds = lambda mu: (1 / (1 + eps * (1 - mu))) ** 2 * (1 / (1 + eps * (1 - mu)) + (1 + eps * (1 - mu)) - 1 + mu * mu)
        Z = integrate.quad(ds, -1, 1)[0]
        mu1 = integrate.quad(lambda m: m * ds(m), -1, 1)[0] / Z
        r1 = integrate.quad(lambda m: ds(m) / (1 + eps * (1 - m)), -1, 1)[0] / Z
        assert c.mean() == pytest.approx(mu1, abs=5 * c.std() / math.sqrt(n))
        assert (e / eps).mean() == pytest.approx(r1, abs=5 * (e / eps).std() / math.sqrt(n))


def test_event_rate_weighting_of_electron_direction(olib):
    """The electron direction cosine follows the pdf (1 - beta mu)/2 (the kernel of PAPER.md Eq. 23), whose mean is
    -beta/3.  For ultra-relativistic electrons and soft photons the scattered photon is beamed along the electron,
    so the lab-frame scattering cosine must average to -1/3 (an unweighted, isotropic electron would give 0)."""
    n = 200000
    e, c, kk = olib.compton_sample(60.0, 1e-12, 21, n)
    assert c.mean() == pytest.approx(-1.0 / 3.0, abs=5 * c.std() / math.sqrt(n) + 5e-3)
