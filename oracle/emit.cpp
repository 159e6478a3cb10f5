// ORACLE (test infrastructure).  Superphoton weights, per-zone counts and emission sampling.
//
//  prepare        Eq. 2 (weight per frequency), Eq. 5 (expected count per zone,
//                 PAPER.md:65-67), Eq. 6 (dN/dln nu); readings G8 (Delta ln nu of
//                 Eq. 2 = ln(nu_max/nu_min)), G9 (trapezoid on the weight-table nodes), G10
//                 (stochastic integerisation with one uniform per zone).
//  emit_photon    Eq. 7-8 frequency rejection, Eq. 9 direction rejection
//                 (PAPER.md:83-85), emission in the plasma frame then "boosting back into the
//                 coordinate basis" through a Gram-Schmidt tetrad (G13);
//                 emission position = zone centre (G12).
//
// Pins (tests/test_oracle_emit.py): sum_i N_s,i = N_s when w_min = 0; per-zone count against a
// brute-force scipy quadrature of Eq. 5 on a 2x2 grid; k.k = 0 and -k.u = h nu/m_e c^2; tetrad
// orthonormality; accepted-frequency histogram vs F(K)/w; <cos^2 theta> vs quadrature of Eq. 3;
// thin-sphere spectrum vs Eq. 34 (tests/test_oracle_sphere.py).
#include "oracle.hpp"
#include <cmath>
#include <algorithm>

namespace orc {

static const double JPREF_E = std::sqrt(2.0) * PI * EE * EE / (3.0 * CL);

static void zone_centre(const Params& P, int i, int j, int k, double x[4]) {
  x[0] = 0.0;
  x[1] = P.startx[1] + (i + 0.5) * P.dx[1];
  x[2] = P.startx[2] + (j + 0.5) * P.dx[2];
  x[3] = P.startx[3] + (k + 0.5) * P.dx[3];
}

// Proper coordinate volume of zone (i,j,k): the integral of sqrt(-g) = (r^2 + a^2 cos^2 theta) sin(theta) r theta'(x2)
// over the zone, in closed form (dr = r dx1, dtheta = theta' dx2):
//   dphi * [ (r_hi^3 - r_lo^3)/3 (cos th_lo - cos th_hi) + a^2 (r_hi - r_lo) (cos^3 th_lo - cos^3 th_hi)/3 ].
// the paper smooths zone boundaries with 8192-32000 radial cells and partial cells; reading
// G31 (emit_mode 1) removes the midpoint-rule volume error of sqrt(-g)_centre dx1 dx2 dx3 instead.
double zone_volume(const Params& P, int i, int j, int k) {
  (void)k;
  double a = P.metric_kind == 1 ? P.a_spin : 0.0;
  double rlo = std::exp(P.startx[1] + i * P.dx[1]), rhi = std::exp(P.startx[1] + (i + 1) * P.dx[1]);
  double clo = std::cos(theta_of_x2(P, P.startx[2] + j * P.dx[2]));
  double chi = std::cos(theta_of_x2(P, P.startx[2] + (j + 1) * P.dx[2]));
  return P.dx[3] * ((rhi * rhi * rhi - rlo * rlo * rlo) / 3.0 * (clo - chi) +
                    a * a * (rhi - rlo) * (clo * clo * clo - chi * chi * chi) / 3.0);
}

// Position uniform in proper volume inside zone (i,j,k) (G31): rejection on sqrt(-g) from a uniform proposal in the
// zone's coordinate box.  Four uniforms per trial, in this order: x1, x2, x3, acceptance.  The bound is
// r_hi (r_hi^2 + a^2 max cos^2) max sin * max theta' over the zone (each factor is monotone between the zone edges,
// except sin which peaks at the equator), times 1 + 1e-12.
void sample_zone_position(const Params& P, int i, int j, int k, Stream& rs, double x[4]) {
  double a = P.metric_kind == 1 ? P.a_spin : 0.0;
  double x1lo = P.startx[1] + i * P.dx[1], x2lo = P.startx[2] + j * P.dx[2], x3lo = P.startx[3] + k * P.dx[3];
  double x2hi = P.startx[2] + (j + 1) * P.dx[2];
  double rhi = std::exp(P.startx[1] + (i + 1) * P.dx[1]);
  double tlo = theta_of_x2(P, x2lo), thi = theta_of_x2(P, x2hi);
  double clo = std::cos(tlo), chi = std::cos(thi);
  double c2 = clo * clo > chi * chi ? clo * clo : chi * chi;
  double slo = std::sin(tlo), shi = std::sin(thi);
  double smax = (tlo <= 0.5 * PI && thi >= 0.5 * PI) ? 1.0 : (slo > shi ? slo : shi);
  double dlo = dtheta_dx2(P, x2lo), dhi = dtheta_dx2(P, x2hi);
  double bound = rhi * (rhi * rhi + a * a * c2) * smax * (dlo > dhi ? dlo : dhi) * (1.0 + 1e-12);
  x[0] = 0.0;
  for (;;) {
    double ua = rs.next(), ub = rs.next(), uc = rs.next(), ud = rs.next();
    x[1] = x1lo + ua * P.dx[1];
    x[2] = x2lo + ub * P.dx[2];
    x[3] = x3lo + uc * P.dx[3];
    Geom G;
    geom_func(P, x, &G);
    if (ud * bound < G.gdet) return;
  }
}

double weight_of_nu(const Context& C, double nu) {
  const Params& P = C.P;
  double dl = std::log(P.nu_max / P.nu_min) / NW;
  double f = (std::log(nu) - std::log(P.nu_min)) / dl;
  int i = (int)std::floor(f);
  if (i < 0) i = 0;
  if (i > NW - 1) i = NW - 1;
  double t = f - (double)i;
  return std::exp(C.lnw[i] * (1.0 - t) + C.lnw[i + 1] * t);
}

void prepare(Context* C) {
  const Params& P = C->P;
  C->un = make_units(P);
  build_tables(&C->T, P.scattering_on != 0);
  const long nz = (long)P.n1 * P.n2 * P.n3;
  C->zones.assign(nz, ZoneInfo());
  const double Lam = std::log(P.nu_max / P.nu_min);
  const double Dl = Lam / NW;
  C->nu_nodes.resize(NW + 1);
  for (int k = 0; k <= NW; k++) C->nu_nodes[k] = P.nu_min * std::exp(k * Dl);
  const double dt = C->un.T;
  const double dV = P.dx[1] * P.dx[2] * P.dx[3] * P.L_unit * P.L_unit * P.L_unit;

  // per-zone plasma state at the zone centre
  std::vector<double> gdet(nz);
  for (int i = 0; i < P.n1; i++)
    for (int j = 0; j < P.n2; j++)
      for (int k = 0; k < P.n3; k++) {
        long z = ((long)i * P.n2 + j) * P.n3 + k;
        double x[4];
        zone_centre(P, i, j, k, x);
        Geom G;
        geom_func(P, x, &G);
        gdet[z] = G.gdet;
        ZoneInfo& Z = C->zones[z];
        const double* pr = &C->prim[z * 8];
        Z.A = 0.0; Z.nu0 = 0.0; Z.C = 0.0; Z.qmax = 0.0; Z.Nexp = 0.0; Z.n = 0;
        if (!(pr[0] > 0.0)) continue;
        Plasma S;
        plasma_from_prim(P, C->un, G, pr, &S);
        if (!(S.ne > 0.0) || !(S.B > 0.0) || !(S.thetae >= P.thetae_min)) continue;
        double nuc = EE * S.B / (2.0 * PI * ME * CL);
        Z.nu0 = (2.0 / 9.0) * nuc * S.thetae * S.thetae;
        Z.A = JPREF_E * S.ne * Z.nu0 / K2_eval(C->T, S.thetae);
        if (P.emit_mode == 1) gdet[z] = zone_volume(P, i, j, k) / (P.dx[1] * P.dx[2] * P.dx[3]);   // zone-averaged sqrt(-g) (G31)
        Z.C = dt * gdet[z] * dV * Z.A / HPL;
      }

  // Eq. 2: w(nu_k) = dt * Lambda/(h N_s) * sum_zones sqrt(-g) d3x int j_nu dOmega  (+ w_min floor)
  C->lnw.resize(NW + 1);
  std::vector<double> wk(NW + 1);
  for (int k = 0; k <= NW; k++) {
    double S = 0.0;
    for (long z = 0; z < nz; z++) {
      const ZoneInfo& Z = C->zones[z];
      if (Z.A > 0.0) S += gdet[z] * dV * Z.A * F_eval(C->T, C->nu_nodes[k] / Z.nu0);
    }
    wk[k] = dt * Lam / (HPL * P.Ns_target) * S + P.w_min;
    C->lnw[k] = wk[k] > 0.0 ? std::log(wk[k]) : -700.0;
  }

  // Eq. 5 discretised on the same nodes (trapezoid in ln nu), Eq. 8 denominator, integerisation
  C->offset.assign(nz + 1, 0);
  for (long z = 0; z < nz; z++) {
    ZoneInfo& Z = C->zones[z];
    if (Z.A > 0.0) {
      double sum = 0.0, qmax = 0.0;
      for (int k = 0; k <= NW; k++) {
        double q = wk[k] > 0.0 ? F_eval(C->T, C->nu_nodes[k] / Z.nu0) / wk[k] : 0.0;
        double ck = (k == 0 || k == NW) ? 0.5 : 1.0;
        sum = sum + ck * q;
        if (q > qmax) qmax = q;
      }
      Z.qmax = qmax;
      Z.Nexp = Z.C * (Dl * sum);
      double u0, u1;
      uniform_pair(P.seed, TAG_ZONE, (uint32_t)(z & 0xffffffff), (uint32_t)((uint64_t)z >> 32), 0u, 0u, &u0, &u1);
      double fl = std::floor(Z.Nexp);
      Z.n = (int32_t)fl + ((u0 < Z.Nexp - fl) ? 1 : 0);
    }
    C->offset[z + 1] = C->offset[z] + Z.n;
  }
  tally_init(P, &C->tally);
  C->stats = Stats();
  std::fill(C->gen_spawn.begin(), C->gen_spawn.end(), 0);
  std::fill(C->bias_fac.begin(), C->bias_fac.end(), 1.0);
  C->prepared = true;
}

// Gram-Schmidt tetrad (G13): e0 = u, e1 along `trial` (b for emission, the
// photon direction for scattering), e2 from the first of d_3, d_1, d_2 that keeps a quarter
// of its length after projection, e3 from the Levi-Civita tensor.
static void project_out(const Geom& G, double v[4], const double e[4], double sign_ee) {
  double ve = dot(G.gcov, v, e);
  for (int m = 0; m < 4; m++) v[m] -= sign_ee * ve * e[m];
}

void make_tetrad(const Geom& G, const double ucon[4], const double trial[4], double econ[4][4]) {
  for (int m = 0; m < 4; m++) econ[0][m] = ucon[m];
  double v[4];
  for (int m = 0; m < 4; m++) v[m] = trial[m];
  project_out(G, v, econ[0], -1.0);
  double n2 = dot(G.gcov, v, v);
  if (!(n2 > 0.0)) {
    v[0] = 0.0; v[1] = 1.0; v[2] = 0.0; v[3] = 0.0;
    project_out(G, v, econ[0], -1.0);
    n2 = dot(G.gcov, v, v);
  }
  double nrm = std::sqrt(n2);
  for (int m = 0; m < 4; m++) econ[1][m] = v[m] / nrm;

  const int order[3] = {3, 1, 2};
  double best[4] = {0, 0, 0, 0}, bestp = -1.0;
  bool found = false;
  for (int c = 0; c < 3 && !found; c++) {
    int ax = order[c];
    double t[4] = {0, 0, 0, 0};
    t[ax] = 1.0;
    project_out(G, t, econ[0], -1.0);
    project_out(G, t, econ[1], +1.0);
    double t2 = dot(G.gcov, t, t);
    double p = t2 / G.gcov[ax][ax];
    if (p > bestp) { bestp = p; for (int m = 0; m < 4; m++) best[m] = t[m]; }
    if (p >= 0.25) { for (int m = 0; m < 4; m++) best[m] = t[m]; found = true; }
  }
  double b2 = dot(G.gcov, best, best);
  double bn = std::sqrt(b2);
  for (int m = 0; m < 4; m++) econ[2][m] = best[m] / bn;

  double c0[4], c1[4], c2[4];
  lower(G.gcov, econ[0], c0);
  lower(G.gcov, econ[1], c1);
  lower(G.gcov, econ[2], c2);
  // e3^m = -(1/sqrt(-g)) [m n r s] e0_n e1_r e2_s
  static const int perm[24][4] = {
      {0, 1, 2, 3}, {0, 1, 3, 2}, {0, 2, 1, 3}, {0, 2, 3, 1}, {0, 3, 1, 2}, {0, 3, 2, 1},
      {1, 0, 2, 3}, {1, 0, 3, 2}, {1, 2, 0, 3}, {1, 2, 3, 0}, {1, 3, 0, 2}, {1, 3, 2, 0},
      {2, 0, 1, 3}, {2, 0, 3, 1}, {2, 1, 0, 3}, {2, 1, 3, 0}, {2, 3, 0, 1}, {2, 3, 1, 0},
      {3, 0, 1, 2}, {3, 0, 2, 1}, {3, 1, 0, 2}, {3, 1, 2, 0}, {3, 2, 0, 1}, {3, 2, 1, 0}};
  static const int sgn[24] = {+1, -1, -1, +1, +1, -1, -1, +1, +1, -1, -1, +1,
                              +1, -1, -1, +1, +1, -1, -1, +1, +1, -1, -1, +1};
  for (int m = 0; m < 4; m++) econ[3][m] = 0.0;
  for (int q = 0; q < 24; q++) {
    const int* p = perm[q];
    econ[3][p[0]] += sgn[q] * c0[p[1]] * c1[p[2]] * c2[p[3]];
  }
  for (int m = 0; m < 4; m++) econ[3][m] *= -1.0 / G.gdet;
}

static void accel(const Params& P, const double x[4], const double k[4], double a[4]) {
  double conn[4][4][4];
  conn_func(P, x, conn);
  for (int m = 0; m < 4; m++) {
    double s = 0.0;
    for (int al = 0; al < 4; al++)
      for (int be = 0; be < 4; be++) s += conn[m][al][be] * k[al] * k[be];
    a[m] = -s;
  }
}

void emit_photon(const Context& C, int64_t pid, Photon* ph) {
  const Params& P = C.P;
  // zone of this primary id: offset[z] <= pid < offset[z+1]
  long nz = (long)C.zones.size();
  long z = (long)(std::upper_bound(C.offset.begin(), C.offset.end(), pid) - C.offset.begin()) - 1;
  if (z < 0) z = 0;
  if (z >= nz) z = nz - 1;
  const ZoneInfo& Z = C.zones[z];
  int k3 = (int)(z % P.n3);
  int j2 = (int)((z / P.n3) % P.n2);
  int i1 = (int)(z / ((long)P.n3 * P.n2));
  ph->id.i0 = (uint32_t)((uint64_t)pid & 0xffffffffu);
  ph->id.i1 = (uint32_t)((uint64_t)pid >> 32);
  ph->id.i2 = 0u;
  Stream rs(P.seed, TAG_EMIT, ph->id.i0, ph->id.i1, ph->id.i2);

  double x[4];
  Geom G;
  Plasma S;
  if (P.emit_mode == 1) {
    // G31: position uniform in proper volume inside the zone (drawn first), plasma state interpolated there;
    // where the interpolated state does not emit (vacuum, Theta_e < thetae_min, B = 0) the zone's own state is kept
    sample_zone_position(P, i1, j2, k3, rs, x);
    geom_func(P, x, &G);
    plasma_at(P, C.un, C.prim.data(), x, G, &S);
    if (S.vacuum || !(S.ne > 0.0) || !(S.B > 0.0) || !(S.thetae >= P.thetae_min))
      plasma_from_prim(P, C.un, G, &C.prim[z * 8], &S);
  } else {
    zone_centre(P, i1, j2, k3, x);
    geom_func(P, x, &G);
    plasma_from_prim(P, C.un, G, &C.prim[z * 8], &S);
  }

  const double Lam = std::log(P.nu_max / P.nu_min);
  double nu = 0.0;
  for (;;) {                                   // Eq. 7-8
    double u1 = rs.next(), u2 = rs.next();
    nu = std::exp(u1 * Lam + std::log(P.nu_min));
    double q = F_eval(C.T, nu / Z.nu0) / weight_of_nu(C, nu);
    if (u2 < q / Z.qmax) break;
  }
  double cth = 0.0, sth = 0.0;
  double jmax = jnu(C.T, nu, S.ne, S.thetae, S.B, 1.0);
  for (;;) {                                   // Eq. 9
    double u3 = rs.next(), u4 = rs.next();
    cth = 2.0 * u3 - 1.0;
    sth = std::sqrt(1.0 - cth * cth);
    if (u4 < jnu(C.T, nu, S.ne, S.thetae, S.B, sth) / jmax) break;
  }
  double phi = 2.0 * PI * rs.next();

  double e0 = HPL * nu / (ME * CL * CL);
  double kt[4] = {e0, e0 * cth, e0 * sth * std::cos(phi), e0 * sth * std::sin(phi)};
  double econ[4][4];
  make_tetrad(G, S.ucon, S.bcon, econ);
  for (int m = 0; m < 4; m++) {
    ph->x[m] = x[m];
    ph->k[m] = econ[0][m] * kt[0] + econ[1][m] * kt[1] + econ[2][m] * kt[2] + econ[3][m] * kt[3];
  }
  accel(P, ph->x, ph->k, ph->a);
  ph->w = weight_of_nu(C, nu);
  ph->nsc = 0; ph->nstep = 0; ph->jscat = 0;
  opacities(C, ph->x, ph->k, G, S, &ph->nua_a, &ph->nua_s, &ph->bias, 0);
  double kcov[4];
  lower(G.gcov, ph->k, kcov);
  ph->E0 = -kcov[0];
}

}  // namespace orc
