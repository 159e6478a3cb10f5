// ORACLE (test infrastructure).  One Compton scattering event.
//
// "A plasma-frame orthonormal tetrad is constructed via a Gram-Schmidt orthogonalization
//  procedure, and the wave vector of the incoming superphoton is transformed to this frame.
//  The four-momentum of the scattering electron is sampled from the local electron distribution
//  function using a rejection-sampling method [...].  For each candidate electron-photon pair, a
//  second rejection step [samples] the scattered superphoton based on the differential Compton
//  scattering cross section, using the Thomson limit at low photon energies and the full
//  Klein-Nishina cross section otherwise.  [...] equivalent to the prescription of Canfield et
//  al. (1987) for isotropic thermal (Maxwell-Juttner) electron distributions.  The scattered
//  photon wave vector is finally constructed in the electron rest frame and boosted back."
//
// Readings: G24 (Maxwell-Juttner sampler: gamma = 1 + Theta y^2, four-component Gamma-mixture
// envelope), G25 (Thomson below eps' = 1e-4), canonical draw order (O8).
// Uniforms come from the TAG_SCAT stream keyed by (parent id, ordinal j of the event).
//
// Pins (tests/test_oracle_compton.py): <gamma>, <gamma^2> of the sampler vs K-Bessel closed
// forms; <mu> = -beta/3; scattered-photon nullity; mean energy amplification
// 1 + (4/3)<gamma^2 beta^2> in the Thomson regime; Klein-Nishina mean energy loss for
// cold electrons vs direct quadrature of the differential cross-section.
#include "oracle.hpp"
#include <cmath>

namespace orc {

// Maxwell-Juttner sample; consumes exactly 6 uniforms per trial
void sample_electron_mj(Stream& rs, double thetae, double* gamma_e, double* beta_e) {
  const double sp = std::sqrt(PI);
  double w2 = sp / 4.0;
  double w3 = 0.5 * std::sqrt(0.5 * thetae);
  double w4 = 3.0 * sp * thetae / 8.0;
  double w5 = thetae * std::sqrt(0.5 * thetae);
  double wt = w2 + w3 + w4 + w5;
  for (;;) {
    double us = rs.next();
    double u1 = rs.next(), u2 = rs.next(), u3 = rs.next(), u4 = rs.next();
    double ua = rs.next();
    double l1 = std::log(1.0 - u1), l2 = std::log(1.0 - u2), l3 = std::log(1.0 - u3);
    double y2;
    double sel = us * wt;
    if (sel < w2) {                       // y^2 ~ Gamma(3/2)
      double c = std::cos(2.0 * PI * u3);
      y2 = -l1 - l2 * c * c;
    } else if (sel < w2 + w3) {           // Gamma(2)
      y2 = -(l1 + l2);
    } else if (sel < w2 + w3 + w4) {      // Gamma(5/2)
      double c = std::cos(2.0 * PI * u4);
      y2 = -(l1 + l2) - l3 * c * c;
    } else {                              // Gamma(3)
      y2 = -(l1 + l2 + l3);
    }
    double y = std::sqrt(y2);
    double acc = std::sqrt(1.0 + 0.5 * thetae * y2) / (1.0 + y * std::sqrt(0.5 * thetae));
    if (ua < acc) {
      double t = thetae * y2;
      double gam = 1.0 + t;
      double gb = y * std::sqrt(thetae) * std::sqrt(2.0 + t);
      *gamma_e = gam;
      *beta_e = gb / gam;
      return;
    }
  }
}

bool compton_event(const Context& C, const Photon& p, const Geom& G, const Plasma& S, uint32_t j,
                   double kout[4]) {
  const Params& P = C.P;
  double kcov[4];
  lower(G.gcov, p.k, kcov);
  double eps = 0.0;
  for (int m = 0; m < 4; m++) eps -= kcov[m] * S.ucon[m];
  if (!(eps > 0.0) || !std::isfinite(eps)) return false;
  double econ[4][4];
  make_tetrad(G, S.ucon, p.k, econ);          // e1 along the photon: k^(a) = eps (1,1,0,0)

  Stream rs(P.seed, TAG_SCAT, p.id.i0, p.id.i1, p.id.i2, 0u, j);
  double gam, beta, mu, phie, epsp;
  for (;;) {
    sample_electron_mj(rs, S.thetae, &gam, &beta);
    double um = rs.next();
    double z = 2.0 * beta + beta * beta - 4.0 * beta * um;
    mu = -(2.0 + beta - 4.0 * um) / (1.0 + std::sqrt(1.0 + z));     // pdf ~ (1 - beta mu)
    phie = 2.0 * PI * rs.next();
    epsp = eps * gam * (1.0 - beta * mu);
    double uk = rs.next();
    if (uk < sigma_kn_over_T(epsp)) break;
  }
  if (mu > 1.0) mu = 1.0;
  if (mu < -1.0) mu = -1.0;
  double sm = std::sqrt(1.0 - mu * mu);
  double ne[3] = {mu, sm * std::cos(phie), sm * std::sin(phie)};   // electron direction, axes (1,2,3)

  // photon into the electron rest frame
  double pv[3] = {eps, 0.0, 0.0};
  double ndp = eps * mu;
  double fac = (gam - 1.0) * ndp - gam * beta * eps;
  double pp[3];
  for (int i = 0; i < 3; i++) pp[i] = pv[i] + fac * ne[i];
  double nn = std::sqrt(pp[0] * pp[0] + pp[1] * pp[1] + pp[2] * pp[2]);
  double np[3] = {pp[0] / nn, pp[1] / nn, pp[2] / nn};

  // scattering angle and energy in the electron frame
  double eout, mus;
  if (epsp > 1e-4) {                          // Klein-Nishina
    double elo = epsp / (1.0 + 2.0 * epsp);
    double fmax = (1.0 + 2.0 * epsp) + 1.0 / (1.0 + 2.0 * epsp);
    for (;;) {
      double up = rs.next(), ua = rs.next();
      eout = elo + up * (epsp - elo);
      mus = 1.0 + 1.0 / epsp - 1.0 / eout;
      double f = epsp / eout + eout / epsp - 1.0 + mus * mus;
      if (ua * fmax < f) break;
    }
  } else {                                    // Thomson
    for (;;) {
      double u1 = rs.next(), u2 = rs.next();
      mus = 2.0 * u1 - 1.0;
      if (2.0 * u2 < 1.0 + mus * mus) break;
    }
    eout = epsp;
  }
  if (mus > 1.0) mus = 1.0;
  if (mus < -1.0) mus = -1.0;
  double phis = 2.0 * PI * rs.next();

  // perpendicular pair about the incoming direction: least-aligned axis among (2),(3),(1)
  int cand[3] = {1, 2, 0};
  int ax = cand[0];
  for (int c = 1; c < 3; c++) if (std::fabs(np[cand[c]]) < std::fabs(np[ax])) ax = cand[c];
  double ep[3] = {0.0, 0.0, 0.0};
  ep[ax] = 1.0;
  double d = np[ax];
  for (int i = 0; i < 3; i++) ep[i] -= d * np[i];
  double en = std::sqrt(ep[0] * ep[0] + ep[1] * ep[1] + ep[2] * ep[2]);
  for (int i = 0; i < 3; i++) ep[i] /= en;
  double eq[3] = {np[1] * ep[2] - np[2] * ep[1], np[2] * ep[0] - np[0] * ep[2], np[0] * ep[1] - np[1] * ep[0]};
  double ss = std::sqrt(1.0 - mus * mus);
  double cs = std::cos(phis), sn = std::sin(phis);
  double po[3];
  for (int i = 0; i < 3; i++) po[i] = eout * (mus * np[i] + ss * (cs * ep[i] + sn * eq[i]));

  // back to the plasma frame (boost with -beta n_e)
  double ndpo = ne[0] * po[0] + ne[1] * po[1] + ne[2] * po[2];
  double k0 = gam * (eout + beta * ndpo);
  double fb = (gam - 1.0) * ndpo + gam * beta * eout;
  double kt[4] = {k0, po[0] + fb * ne[0], po[1] + fb * ne[1], po[2] + fb * ne[2]};
  for (int m = 0; m < 4; m++)
    kout[m] = econ[0][m] * kt[0] + econ[1][m] * kt[1] + econ[2][m] * kt[2] + econ[3][m] * kt[3];
  if (!(k0 > 0.0)) return false;
  for (int m = 0; m < 4; m++) if (!std::isfinite(kout[m])) return false;
  return true;
}

}  // namespace orc
