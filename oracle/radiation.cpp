// ORACLE (test infrastructure).  Emissivity, absorption, cross sections and their tables.
//
//  jnu                 Eq. 3-4, prefactor sqrt(2)*pi (G1: the printed
//                      sqrt(2 pi) is a garble of the cited Leung et al. 2011 fit; pinned by the
//                      total-synchrotron-power identity).
//  K2                  "K2(1/Theta) ~ 2 Theta^2 in the large temperature limit";
//                      else a 201-node log-log table of std::cyl_bessel_k (G6).
//  F(K)                angle integral of Eq. 3 needed by Eqs. 2, 5, 6, tabulated (G7).
//  nu_alpha_abs        alpha_nu = j_nu/B_nu, in the invariant form nu*alpha_nu of Eq. 16/20.
//  sigma_kn_over_T     Eq. 26 and its small-eps limit Eq. 27 (G22).
//  sigma_hot_direct    Eq. 23 for a Maxwell-Juttner distribution.
//  sigma_hot_eval      "sigma_h is calculated a priori and stored in a lookup table" (G23).
//
// Pins (tests/test_oracle_radiation.py): K2 large-Theta limit and scipy.special.kv; three
// independently computed F(K) values + small-K asymptote; integral of j_nu over nu and Omega =
// (4/3) sigma_T c U_B <gamma^2 beta^2> n_e within the fit accuracy; sigma_KN series/closed-form
// overlap and the 3/8 (ln 2e + 1/2)/e ultra-relativistic limit; sigma_h -> sigma_KN (Theta -> 0),
// -> sigma_T (eps -> 0), brute-force Monte-Carlo average over a sampled MJ distribution.
#include "oracle.hpp"
#include <cmath>
#include <functional>

namespace orc {

// ---- adaptive Simpson --------------------------------------------------------
static double simpson_rec(const std::function<double(double)>& f, double a, double b, double fa, double fm,
                          double fb, double whole, double tol, int depth) {
  double m = 0.5 * (a + b);
  double lm = 0.5 * (a + m), rm = 0.5 * (m + b);
  double flm = f(lm), frm = f(rm);
  double left = (m - a) / 6.0 * (fa + 4.0 * flm + fm);
  double right = (b - m) / 6.0 * (fm + 4.0 * frm + fb);
  double delta = left + right - whole;
  // accept at the requested tolerance, or when the Richardson difference has reached the
  // rounding noise of the panel sum (otherwise an over-tight tolerance would recurse forever)
  double mag = (b - a) * (std::fabs(fa) + std::fabs(flm) + std::fabs(fm) + std::fabs(frm) + std::fabs(fb)) / 5.0;
  if (depth <= 0 || std::fabs(delta) <= 15.0 * tol || std::fabs(delta) <= 1e-14 * mag)
    return left + right + delta / 15.0;
  return simpson_rec(f, a, m, fa, flm, fm, left, 0.5 * tol, depth - 1) +
         simpson_rec(f, m, b, fm, frm, fb, right, 0.5 * tol, depth - 1);
}

// integrate f on [a,b]; the interval is first cut into npanel equal panels so that a
// narrow feature cannot be missed by the first three samples; abs tolerance = rel * |coarse|
static double integrate(const std::function<double(double)>& f, double a, double b, double rel, int npanel) {
  std::vector<double> fa(npanel + 1), fm(npanel);
  double h = (b - a) / npanel;
  for (int i = 0; i <= npanel; i++) fa[i] = f(a + i * h);
  for (int i = 0; i < npanel; i++) fm[i] = f(a + (i + 0.5) * h);
  double coarse = 0.0, coarse_abs = 0.0;
  for (int i = 0; i < npanel; i++) {
    double s = h / 6.0 * (fa[i] + 4.0 * fm[i] + fa[i + 1]);
    coarse += s;
    coarse_abs += std::fabs(s);
  }
  if (coarse_abs == 0.0) return 0.0;
  double tol = rel * coarse_abs / npanel;
  double sum = 0.0;
  for (int i = 0; i < npanel; i++) {
    double s = h / 6.0 * (fa[i] + 4.0 * fm[i] + fa[i + 1]);
    sum += simpson_rec(f, a + i * h, a + (i + 1) * h, fa[i], fm[i], fa[i + 1], s, tol, 30);
  }
  return sum;
}

// ---- Bessel K2 -------------------------------------------------------------------
double K2_direct(double thetae) { return std::cyl_bessel_k(2.0, 1.0 / thetae); }

// ---- angle-integrated emissivity shape ----------------------------------------------
// int j_nu dOmega = (sqrt2 pi e^2/(3c)) n_e nu_0 F(K)/K2,  nu_0 = (2/9) nu_c Theta^2, K = nu/nu_0,
// F(K) = 4 pi int_0^{pi/2} sin^2(th) (X^1/2 + 2^11/12 X^1/6)^2 exp(-X^1/3) dth,  X = K / sin(th).
static const double TWO_11_12 = std::pow(2.0, 11.0 / 12.0);
double F_direct(double K) {
  auto g = [K](double th) -> double {
    double s = std::sin(th);
    if (s <= 0.0) return 0.0;
    double X = K / s;
    double x13 = std::cbrt(X);
    double t = std::sqrt(X) + TWO_11_12 * std::sqrt(x13);
    return s * s * t * t * std::exp(-x13);
  };
  return 4.0 * PI * integrate(g, 0.0, 0.5 * PI, 1e-14, 64);
}
static double F_smallK(double K) {
  static const double c = 4.0 * PI * std::pow(2.0, 11.0 / 6.0) * 0.5 * std::sqrt(PI) *
                          std::tgamma(4.0 / 3.0) / std::tgamma(11.0 / 6.0);
  return c * std::cbrt(K);
}

// ---- Klein-Nishina total cross-section / sigma_T ---------------------------------------
double sigma_kn_over_T(double e) {
  if (e < 1e-3) return 1.0 - 2.0 * e + 5.2 * e * e;   // Eq. 27 (+ next term, G22)
  double l = std::log1p(2.0 * e);
  return 0.75 / (e * e) *
         (2.0 + e * e * (1.0 + e) / ((1.0 + 2.0 * e) * (1.0 + 2.0 * e)) + (e * e - 2.0 * e - 2.0) / (2.0 * e) * l);
}

// ---- hot cross-section, Eq. 23 for Maxwell-Juttner electrons ----------------------------
// sigma_h/sigma_T = 1/2 int dmu int dgamma f_MJ(gamma) (1 - mu beta) sigma_KN(eps gamma (1 - mu beta))/sigma_T,
// f_MJ = gamma^2 beta exp(-gamma/Theta)/(Theta K2(1/Theta)).  With gamma = 1 + Theta y^2,
// f_MJ dgamma is proportional to y^2 (1 + Theta y^2) sqrt(2 + Theta y^2) exp(-y^2) dy; the
// normalisation int f_MJ dgamma = 1 is imposed by dividing by the same integral without the
// cross-section factor (so K2(1/Theta), which underflows for small Theta, never appears).
double sigma_hot_direct(double thetae, double eps) {
  auto gy = [thetae](double y) -> double {
    double t = thetae * y * y;
    return y * y * (1.0 + t) * std::sqrt(2.0 + t) * std::exp(-y * y);
  };
  auto hy = [thetae, eps](double y) -> double {
    double t = thetae * y * y;
    double gam = 1.0 + t;
    double gb = y * std::sqrt(thetae) * std::sqrt(2.0 + t);   // gamma*beta
    double beta = gb / gam;
    auto fmu = [gam, beta, eps](double mu) -> double {
      double d = 1.0 - mu * beta;
      return d * sigma_kn_over_T(eps * gam * d);
    };
    return 0.5 * integrate(fmu, -1.0, 1.0, 1e-9, 8);
  };
  const double ymax = 10.0;
  double num = integrate([&](double y) { return gy(y) * hy(y); }, 0.0, ymax, 1e-8, 32);
  double den = integrate(gy, 0.0, ymax, 1e-13, 32);
  return num / den;
}

// ---- tables -----------------------------------------------------------------------------
void build_tables(Tables* T, bool with_sigh) {
  if (T->lnK2.empty()) {
    T->lnK2.resize(NK2 + 1);
    double l0 = std::log(K2_TMIN), dl = std::log(K2_TMAX / K2_TMIN) / NK2;
    for (int i = 0; i <= NK2; i++) T->lnK2[i] = std::log(K2_direct(std::exp(l0 + i * dl)));
    T->lnF.resize(NF + 1);
    double k0 = std::log(F_KMIN), dk = std::log(F_KMAX / F_KMIN) / NF;
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i <= NF; i++) T->lnF[i] = std::log(F_direct(std::exp(k0 + i * dk)));
  }
  if (with_sigh && !T->have_sigh) {
    T->lnSigH.resize((size_t)(NSE + 1) * (NST + 1));
    const double LN10 = std::log(10.0);
    double de = (SH_LE1 - SH_LE0) / NSE, dt = (SH_LT1 - SH_LT0) / NST;
#pragma omp parallel for collapse(2) schedule(dynamic, 8)
    for (int i = 0; i <= NSE; i++)
      for (int j = 0; j <= NST; j++) {
        double eps = std::exp(LN10 * (SH_LE0 + i * de));
        double th = std::exp(LN10 * (SH_LT0 + j * dt));
        T->lnSigH[(size_t)i * (NST + 1) + j] = std::log(sigma_hot_direct(th, eps));
      }
    T->have_sigh = true;
  }
}

double K2_eval(const Tables& T, double thetae) {
  if (thetae > K2_TMAX) return 2.0 * thetae * thetae;
  if (thetae < K2_TMIN) return K2_direct(thetae);         // not reached: emission gated at thetae_min >= 0.3
  double dl = std::log(K2_TMAX / K2_TMIN) / NK2;
  double f = (std::log(thetae) - std::log(K2_TMIN)) / dl;
  int i = (int)std::floor(f);
  if (i < 0) i = 0;
  if (i > NK2 - 1) i = NK2 - 1;
  double w = f - (double)i;
  return std::exp(T.lnK2[i] * (1.0 - w) + T.lnK2[i + 1] * w);
}

double F_eval(const Tables& T, double K) {
  if (K > F_KMAX) return 0.0;
  if (K < F_KMIN) return F_smallK(K);
  double dk = std::log(F_KMAX / F_KMIN) / NF;
  double f = (std::log(K) - std::log(F_KMIN)) / dk;
  int i = (int)std::floor(f);
  if (i < 0) i = 0;
  if (i > NF - 1) i = NF - 1;
  double w = f - (double)i;
  return std::exp(T.lnF[i] * (1.0 - w) + T.lnF[i + 1] * w);
}

double sigma_hot_eval(const Tables& T, double thetae, double eps) {
  double tmax = thetae > 1.0 ? thetae : 1.0;
  if (eps < 1e-12 || eps * tmax < 1e-6) return 1.0;       // Thomson regime
  if (thetae < 1e-4) return sigma_kn_over_T(eps);         // cold electrons
  double de = (SH_LE1 - SH_LE0) / NSE, dt = (SH_LT1 - SH_LT0) / NST;
  double fe = (std::log10(eps) - SH_LE0) / de;
  double ft = (std::log10(thetae) - SH_LT0) / dt;
  if (fe < 0.0) fe = 0.0;
  if (fe > (double)NSE) fe = (double)NSE;
  if (ft < 0.0) ft = 0.0;
  if (ft > (double)NST) ft = (double)NST;
  int i = (int)std::floor(fe), j = (int)std::floor(ft);
  if (i > NSE - 1) i = NSE - 1;
  if (j > NST - 1) j = NST - 1;
  double wi = fe - (double)i, wj = ft - (double)j;
  const double* t = T.lnSigH.data();
  const int s = NST + 1;
  double v = (1.0 - wi) * ((1.0 - wj) * t[i * s + j] + wj * t[i * s + j + 1]) +
             wi * ((1.0 - wj) * t[(i + 1) * s + j] + wj * t[(i + 1) * s + j + 1]);
  return std::exp(v);
}

// ---- emissivity and absorption --------------------------------------------------------------
static const double JPREF = std::sqrt(2.0) * PI * EE * EE / (3.0 * CL);   // G1

double jnu(const Tables& T, double nu, double ne, double thetae, double B, double sin_theta) {
  if (!(ne > 0.0) || !(B > 0.0) || !(sin_theta > 0.0) || !(thetae > 0.0)) return 0.0;
  double nuc = EE * B / (2.0 * PI * ME * CL);
  double nus = (2.0 / 9.0) * nuc * thetae * thetae * sin_theta;        // Eq. 4
  double X = nu / nus;
  double x13 = std::cbrt(X);
  double t = std::sqrt(X) + TWO_11_12 * std::sqrt(x13);
  return JPREF * ne * nus / K2_eval(T, thetae) * t * t * std::exp(-x13);   // Eq. 3
}

double jnu_angle_integrated(const Tables& T, double nu, double ne, double thetae, double B) {
  if (!(ne > 0.0) || !(B > 0.0) || !(thetae > 0.0)) return 0.0;
  double nuc = EE * B / (2.0 * PI * ME * CL);
  double nu0 = (2.0 / 9.0) * nuc * thetae * thetae;
  return JPREF * ne * nu0 / K2_eval(T, thetae) * F_eval(T, nu / nu0);
}

// nu * alpha_nu with alpha_nu = j_nu / B_nu, B_nu = 2 h nu^3/c^2 / expm1(h nu / k T_e)
double nu_alpha_abs(const Tables& T, double nu, double ne, double thetae, double B, double sin_theta) {
  double j = jnu(T, nu, ne, thetae, B, sin_theta);
  if (j == 0.0) return 0.0;
  double x = HPL * nu / (ME * CL * CL * thetae);
  double Bnu = 2.0 * HPL * nu * nu * nu / (CL * CL) / std::expm1(x);
  return nu * j / Bnu;
}

}  // namespace orc
