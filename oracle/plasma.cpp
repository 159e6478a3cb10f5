// ORACLE (test infrastructure).  Fluid grid -> local plasma state.
//
// The paper reads "plasma properties from GRMHD snapshots" and defines all
// plasma quantities in the fluid frame; it does not print the primitive ->
// four-velocity / field map, the electron temperature rule or the interpolation.  Readings:
// G2 (HARM convention u~, B^i), G3 (Theta_e modes), G4 (multilinear interpolation between
// zone centres, clamped in x1/x2, periodic in x3, vacuum outside the x1 range).
//
// Pins (tests/test_oracle_plasma.py): uniform grid -> constant; u.u = -1, u.b = 0;
// sphere field strength 1 G everywhere; bilinear exactness on a linear field.
#include "oracle.hpp"
#include <cmath>

namespace orc {

Units make_units(const Params& P) {
  Units u;
  u.L = P.L_unit;
  u.T = P.L_unit / CL;
  u.M = P.M_unit;
  u.RHO = P.M_unit / (P.L_unit * P.L_unit * P.L_unit);
  u.U = u.RHO * CL * CL;
  u.B = CL * std::sqrt(4.0 * PI * u.RHO);
  u.Ne = u.RHO / (MP + ME);
  return u;
}

// fractional zone-centre index, clamped so that the value is constant outside the
// outermost zone centres
static void axis_weights(double xx, double start, double d, int n, int* i0, int* i1, double* w1) {
  if (n == 1) { *i0 = 0; *i1 = 0; *w1 = 0.0; return; }
  double f = (xx - start) / d - 0.5;
  if (f < 0.0) f = 0.0;
  if (f > (double)(n - 1)) f = (double)(n - 1);
  int i = (int)std::floor(f);
  if (i > n - 2) i = n - 2;
  *i0 = i; *i1 = i + 1; *w1 = f - (double)i;
}

void interp_prim(const Params& P, const double* prim, const double x[4], double out[8], bool* inside) {
  double x1lo = P.startx[1], x1hi = P.startx[1] + P.n1 * P.dx[1];
  if (x[1] < x1lo || x[1] >= x1hi) {
    *inside = false;
    for (int q = 0; q < 8; q++) out[q] = 0.0;
    return;
  }
  *inside = true;
  int i0, i1, j0, j1, k0, k1;
  double wi, wj, wk;
  axis_weights(x[1], P.startx[1], P.dx[1], P.n1, &i0, &i1, &wi);
  double x2 = x[2];
  if (x2 < 0.0) x2 = -x2;            // across the polar axis: reflect
  if (x2 > 1.0) x2 = 2.0 - x2;
  axis_weights(x2, P.startx[2], P.dx[2], P.n2, &j0, &j1, &wj);
  if (P.n3 == 1) { k0 = k1 = 0; wk = 0.0; }
  else {
    double f = (x[3] - P.startx[3]) / P.dx[3] - 0.5;
    double fl = std::floor(f);
    wk = f - fl;
    long kk = (long)fl;
    long n3 = P.n3;
    k0 = (int)(((kk % n3) + n3) % n3);
    k1 = (int)((((kk + 1) % n3) + n3) % n3);
  }
  const long s1 = (long)P.n2 * P.n3 * 8, s2 = (long)P.n3 * 8, s3 = 8;
  for (int q = 0; q < 8; q++) {
    double v000 = prim[i0 * s1 + j0 * s2 + k0 * s3 + q], v001 = prim[i0 * s1 + j0 * s2 + k1 * s3 + q];
    double v010 = prim[i0 * s1 + j1 * s2 + k0 * s3 + q], v011 = prim[i0 * s1 + j1 * s2 + k1 * s3 + q];
    double v100 = prim[i1 * s1 + j0 * s2 + k0 * s3 + q], v101 = prim[i1 * s1 + j0 * s2 + k1 * s3 + q];
    double v110 = prim[i1 * s1 + j1 * s2 + k0 * s3 + q], v111 = prim[i1 * s1 + j1 * s2 + k1 * s3 + q];
    double v00 = v000 * (1.0 - wk) + v001 * wk, v01 = v010 * (1.0 - wk) + v011 * wk;
    double v10 = v100 * (1.0 - wk) + v101 * wk, v11 = v110 * (1.0 - wk) + v111 * wk;
    double v0 = v00 * (1.0 - wj) + v01 * wj, v1 = v10 * (1.0 - wj) + v11 * wj;
    out[q] = v0 * (1.0 - wi) + v1 * wi;
  }
}

// primitives (rho, u, u~^i, B^i) -> n_e, Theta_e, |B|, u^mu, b^mu   (G2, G3)
void plasma_from_prim(const Params& P, const Units& un, const Geom& G, const double pr[8], Plasma* S) {
  S->vacuum = false;
  S->rho = pr[0];
  S->uu = pr[1];
  const double* ut = &pr[2];   // u~^i
  const double* Bp = &pr[5];   // B^i
  double q = 0.0;
  for (int i = 1; i < 4; i++)
    for (int j = 1; j < 4; j++) q += G.gcov[i][j] * ut[i - 1] * ut[j - 1];
  double gamma = std::sqrt(1.0 + q);
  double alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
  S->ucon[0] = gamma / alpha;
  for (int i = 1; i < 4; i++) S->ucon[i] = ut[i - 1] - gamma * alpha * G.gcon[0][i];
  double ucov[4];
  lower(G.gcov, S->ucon, ucov);
  double bt = 0.0;
  for (int i = 1; i < 4; i++) bt += Bp[i - 1] * ucov[i];
  S->bcon[0] = bt;
  for (int i = 1; i < 4; i++) S->bcon[i] = (Bp[i - 1] + bt * S->ucon[i]) / S->ucon[0];
  double bsq = dot(G.gcov, S->bcon, S->bcon);
  if (bsq < 0.0) bsq = 0.0;
  S->B = std::sqrt(bsq) * un.B;
  S->ne = S->rho * un.Ne;
  double th;
  if (P.thetae_mode == 0) {
    th = P.thetae_fixed;
  } else if (P.thetae_mode == 1) {
    th = (MP / ME) * (P.gam_ad - 1.0) * (S->uu / S->rho) / (1.0 + P.trat);
  } else {
    double beta = (P.gam_ad - 1.0) * S->uu / (0.5 * bsq);   // p_gas / p_mag (inf if bsq = 0)
    double b2 = beta * beta;
    double R = std::isfinite(b2) ? (P.R_high * b2 / (1.0 + b2) + P.R_low / (1.0 + b2)) : P.R_high;
    th = (MP / ME) * (2.0 / 3.0) * (S->uu / S->rho) / (2.0 + R);
  }
  if (!(th > 0.0)) th = 0.0;
  if (th > P.thetae_max) th = P.thetae_max;
  S->thetae = th;
}

void plasma_at(const Params& P, const Units& un, const double* prim, const double x[4], const Geom& G,
               Plasma* S) {
  double pr[8];
  bool inside;
  interp_prim(P, prim, x, pr, &inside);
  if (!inside || !(pr[0] > 0.0)) {
    S->vacuum = true;
    S->ne = S->thetae = S->B = S->rho = S->uu = 0.0;
    for (int m = 0; m < 4; m++) S->ucon[m] = S->bcon[m] = 0.0;
    return;
  }
  plasma_from_prim(P, un, G, pr, S);
}

}  // namespace orc
