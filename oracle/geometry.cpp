// ORACLE (test infrastructure).  Coordinates, metric and connection.
//
// Coordinates x = (t, x1 = ln r, x2, x3 = phi), with
// theta(x2) = pi x2 + (1-hslope)/2 sin(2 pi x2)            (G28).
// Metric: Kerr-Schild in (t,r,theta,phi) with mass M = 1 (metric_kind 1) or M = 0
// (flat space, metric_kind 0: the same expressions with f = 0 give spherical-polar
// Minkowski), transformed with dr = r dx1, dtheta = theta'(x2) dx2.
// Connection: the plain definition under Eq. 10,
//   Gamma^m_ab = 1/2 g^{mn} (d_a g_nb + d_b g_na - d_n g_ab),
// with hand-derived analytic d_a g_mn and a generic 4x4 inverse.
//
// Pins (tests/test_oracle_geometry.py): g g^-1 = I; sqrt(-g) closed form; flat limit
// = diag(-1, r^2, r^2 th'^2, r^2 sin^2); analytic dg vs 4th-order central differences;
// conserved E, L_z, Carter Q and k.k along integrated geodesics; straight lines in flat space.
#include "oracle.hpp"
#include <cmath>

namespace orc {

double theta_of_x2(const Params& P, double x2) {
  return PI * x2 + 0.5 * (1.0 - P.hslope) * std::sin(2.0 * PI * x2);
}
double dtheta_dx2(const Params& P, double x2) {
  return PI + (1.0 - P.hslope) * PI * std::cos(2.0 * PI * x2);
}
static double d2theta_dx22(const Params& P, double x2) {
  return -2.0 * PI * PI * (1.0 - P.hslope) * std::sin(2.0 * PI * x2);
}

// Kerr-Schild metric in (t,r,theta,phi) and its r- and theta-derivatives.
static void ks_rtp(double M, double a, double r, double th, double g[4][4], double dgr[4][4],
                   double dgth[4][4]) {
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) g[m][n] = dgr[m][n] = dgth[m][n] = 0.0;
  double s = std::sin(th), c = std::cos(th);
  double s2 = s * s;
  double Sig = r * r + a * a * c * c;
  double f = 2.0 * M * r / Sig;
  double dSig_r = 2.0 * r, dSig_th = -2.0 * a * a * s * c;
  double df_r = 2.0 * M / Sig - 2.0 * M * r * dSig_r / (Sig * Sig);
  double df_th = -2.0 * M * r * dSig_th / (Sig * Sig);
  double ds2_th = 2.0 * s * c;

  g[0][0] = -1.0 + f;             dgr[0][0] = df_r;                 dgth[0][0] = df_th;
  g[0][1] = f;                    dgr[0][1] = df_r;                 dgth[0][1] = df_th;
  g[0][3] = -f * a * s2;          dgr[0][3] = -a * s2 * df_r;       dgth[0][3] = -a * (df_th * s2 + f * ds2_th);
  g[1][1] = 1.0 + f;              dgr[1][1] = df_r;                 dgth[1][1] = df_th;
  g[1][3] = -a * s2 * (1.0 + f);  dgr[1][3] = -a * s2 * df_r;       dgth[1][3] = -a * (ds2_th * (1.0 + f) + s2 * df_th);
  g[2][2] = Sig;                  dgr[2][2] = dSig_r;               dgth[2][2] = dSig_th;
  double W = Sig + a * a * s2 * (1.0 + f);
  double dW_r = dSig_r + a * a * s2 * df_r;
  double dW_th = dSig_th + a * a * (ds2_th * (1.0 + f) + s2 * df_th);
  g[3][3] = s2 * W;               dgr[3][3] = s2 * dW_r;            dgth[3][3] = ds2_th * W + s2 * dW_th;
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < m; n++) { g[m][n] = g[n][m]; dgr[m][n] = dgr[n][m]; dgth[m][n] = dgth[n][m]; }
}

void gcov_func(const Params& P, const double x[4], double gcov[4][4]) {
  double M = P.metric_kind == 1 ? 1.0 : 0.0;
  double a = P.metric_kind == 1 ? P.a_spin : 0.0;
  double r = std::exp(x[1]);
  double th = theta_of_x2(P, x[2]);
  double g[4][4], dr[4][4], dt[4][4];
  ks_rtp(M, a, r, th, g, dr, dt);
  double J[4] = {1.0, r, dtheta_dx2(P, x[2]), 1.0};
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) gcov[m][n] = J[m] * J[n] * g[m][n];
}

void dgcov_func(const Params& P, const double x[4], double dg[4][4][4]) {
  double M = P.metric_kind == 1 ? 1.0 : 0.0;
  double a = P.metric_kind == 1 ? P.a_spin : 0.0;
  double r = std::exp(x[1]);
  double th = theta_of_x2(P, x[2]);
  double g[4][4], gr[4][4], gt[4][4];
  ks_rtp(M, a, r, th, g, gr, gt);
  double dth = dtheta_dx2(P, x[2]);
  double J[4] = {1.0, r, dth, 1.0};
  double dJ1[4] = {0.0, r, 0.0, 0.0};                       // d/dx1 of J
  double dJ2[4] = {0.0, 0.0, d2theta_dx22(P, x[2]), 0.0};   // d/dx2 of J
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      dg[0][m][n] = 0.0;
      dg[3][m][n] = 0.0;
      dg[1][m][n] = dJ1[m] * J[n] * g[m][n] + J[m] * dJ1[n] * g[m][n] + J[m] * J[n] * gr[m][n] * r;
      dg[2][m][n] = dJ2[m] * J[n] * g[m][n] + J[m] * dJ2[n] * g[m][n] + J[m] * J[n] * gt[m][n] * dth;
    }
}

double det4(const double m[4][4]) {
  double a[4][4];
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) a[i][j] = m[i][j];
  double det = 1.0;
  for (int c = 0; c < 4; c++) {
    int p = c;
    for (int r = c + 1; r < 4; r++) if (std::fabs(a[r][c]) > std::fabs(a[p][c])) p = r;
    if (a[p][c] == 0.0) return 0.0;
    if (p != c) { for (int j = 0; j < 4; j++) { double t = a[c][j]; a[c][j] = a[p][j]; a[p][j] = t; } det = -det; }
    det *= a[c][c];
    for (int r = c + 1; r < 4; r++) {
      double fct = a[r][c] / a[c][c];
      for (int j = c; j < 4; j++) a[r][j] -= fct * a[c][j];
    }
  }
  return det;
}

bool invert4(const double m[4][4], double inv[4][4]) {
  double a[4][8];
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) { a[i][j] = m[i][j]; a[i][4 + j] = (i == j) ? 1.0 : 0.0; }
  for (int c = 0; c < 4; c++) {
    int p = c;
    for (int r = c + 1; r < 4; r++) if (std::fabs(a[r][c]) > std::fabs(a[p][c])) p = r;
    if (a[p][c] == 0.0) return false;
    if (p != c) for (int j = 0; j < 8; j++) { double t = a[c][j]; a[c][j] = a[p][j]; a[p][j] = t; }
    double piv = a[c][c];
    for (int j = 0; j < 8; j++) a[c][j] /= piv;
    for (int r = 0; r < 4; r++) if (r != c) {
      double fct = a[r][c];
      if (fct != 0.0) for (int j = 0; j < 8; j++) a[r][j] -= fct * a[c][j];
    }
  }
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) inv[i][j] = a[i][4 + j];
  return true;
}

void geom_func(const Params& P, const double x[4], Geom* G) {
  gcov_func(P, x, G->gcov);
  invert4(G->gcov, G->gcon);
  G->gdet = std::sqrt(std::fabs(det4(G->gcov)));
}

void conn_func(const Params& P, const double x[4], double conn[4][4][4]) {
  double g[4][4], gi[4][4], dg[4][4][4];
  gcov_func(P, x, g);
  invert4(g, gi);
  dgcov_func(P, x, dg);
  for (int m = 0; m < 4; m++)
    for (int a = 0; a < 4; a++)
      for (int b = 0; b < 4; b++) {
        double s = 0.0;
        for (int n = 0; n < 4; n++) s += gi[m][n] * (dg[a][n][b] + dg[b][n][a] - dg[n][a][b]);
        conn[m][a][b] = 0.5 * s;
      }
}

void lower(const double g[4][4], const double v[4], double out[4]) {
  for (int m = 0; m < 4; m++) {
    double s = 0.0;
    for (int n = 0; n < 4; n++) s += g[m][n] * v[n];
    out[m] = s;
  }
}

double dot(const double g[4][4], const double a[4], const double b[4]) {
  double s = 0.0;
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) s += g[m][n] * a[m] * b[n];
  return s;
}

}  // namespace orc
