// ORACLE (test infrastructure).  C entry points used by tests/, smoke() and bench.py's
// cpu_baseline / --impl reference legs through ctypes (tests/oracle_binding.py).
#include "oracle.hpp"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <omp.h>

using namespace orc;

static Tables g_tables;            // parameter-independent: built once per process
static std::mutex g_tables_mu;

static void ensure_tables(bool sigh) {
  std::lock_guard<std::mutex> lk(g_tables_mu);
  build_tables(&g_tables, sigh);
}

extern "C" {

int orc_sizeof_params() { return (int)sizeof(Params); }
int orc_sizeof_stats() { return (int)sizeof(Stats); }
int orc_sizeof_trace() { return (int)sizeof(TraceRec); }

void* orc_create(const Params* p, const double* prim, size_t n_doubles) {
  if (!p || !prim) return nullptr;
  size_t need = (size_t)p->n1 * p->n2 * p->n3 * 8;
  if (n_doubles != need) return nullptr;
  Context* C = new Context();
  C->P = *p;
  C->prim.assign(prim, prim + n_doubles);
  C->un = make_units(C->P);
  return C;
}
void orc_destroy(void* h) { delete (Context*)h; }

int orc_prepare(void* h, int64_t* n_primaries) {
  Context* C = (Context*)h;
  ensure_tables(C->P.scattering_on != 0);
  C->T = g_tables;
  prepare(C);
  if (C->P.bias_tune) tune_bias(C, omp_get_max_threads());     // G32: pilot on the first primaries, factors frozen after
  if (n_primaries) *n_primaries = C->offset.back();
  return 0;
}
// per-generation bias factors (G32) and spawn counts since the last reset: 64 entries each
int orc_get_bias_table(void* h, double* fac, int64_t* gen_spawn) {
  Context* C = (Context*)h;
  for (int g = 0; g < 64; g++) { if (fac) fac[g] = C->bias_fac[g]; if (gen_spawn) gen_spawn[g] = C->gen_spawn[g]; }
  return C->tune_iterations;
}
int orc_set_bias_table(void* h, const double* fac) {
  Context* C = (Context*)h;
  for (int g = 0; g < 64; g++) C->bias_fac[g] = fac[g];
  return 0;
}
int orc_get_zone_counts(void* h, int32_t* out) {
  Context* C = (Context*)h;
  for (size_t z = 0; z < C->zones.size(); z++) out[z] = C->zones[z].n;
  return 0;
}
int orc_get_zone_info(void* h, double* Nexp, double* qmax) {
  Context* C = (Context*)h;
  for (size_t z = 0; z < C->zones.size(); z++) { Nexp[z] = C->zones[z].Nexp; qmax[z] = C->zones[z].qmax; }
  return 0;
}
int orc_get_weight_table(void* h, double* nu, double* w) {
  Context* C = (Context*)h;
  for (int k = 0; k <= NW; k++) { nu[k] = C->nu_nodes[k]; w[k] = std::exp(C->lnw[k]); }
  return 0;
}
int orc_run(void* h, int64_t first, int64_t n, int nthreads) {
  Context* C = (Context*)h;
  if (!C->prepared) return -1;
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  run_range(C, first, n, nthreads);
  return nthreads;
}
int orc_reset_tally(void* h) {
  Context* C = (Context*)h;
  tally_init(C->P, &C->tally);
  C->stats = Stats();
  std::fill(C->gen_spawn.begin(), C->gen_spawn.end(), 0);
  return 0;
}
int orc_get_tally(void* h, double* A, double* Q, double* W, int64_t* n) {
  Context* C = (Context*)h;
  size_t nb = C->tally.A.size();
  std::memcpy(A, C->tally.A.data(), nb * 8);
  std::memcpy(Q, C->tally.Q.data(), nb * 8);
  std::memcpy(W, C->tally.W.data(), nb * 8);
  std::memcpy(n, C->tally.n.data(), nb * 8);
  return 0;
}
// nu L_nu [erg/s] per (theta, nu) bin, its Monte-Carlo sigma, and the superphoton count (O9)
int orc_get_spectrum(void* h, double* nuLnu, double* sigma, int64_t* nphot) {
  Context* C = (Context*)h;
  const Params& P = C->P;
  double db = std::log(P.nu_hi / P.nu_lo) / P.n_nu;
  double dt = C->un.T;
  for (int i = 0; i < P.n_th; i++) {
    double lo, hi, dOm;
    if (P.fold_theta) {
      lo = i * (0.5 * PI / P.n_th); hi = (i + 1) * (0.5 * PI / P.n_th);
      dOm = 4.0 * PI * (std::cos(lo) - std::cos(hi));
    } else {
      lo = i * (PI / P.n_th); hi = (i + 1) * (PI / P.n_th);
      dOm = 2.0 * PI * (std::cos(lo) - std::cos(hi));
    }
    double scale = ME * CL * CL / dt * (4.0 * PI / dOm) / db;
    for (int j = 0; j < P.n_nu; j++) {
      size_t b = (size_t)i * P.n_nu + j;
      nuLnu[b] = scale * C->tally.A[b];
      sigma[b] = scale * std::sqrt(C->tally.Q[b]);
      nphot[b] = C->tally.n[b];
    }
  }
  return 0;
}
int orc_get_stats(void* h, Stats* out) { *out = ((Context*)h)->stats; return 0; }

// state of a primary right after emission: x[4] k[4] a[4] w nua_a nua_s bias E0  (20 doubles)
int orc_emit(void* h, int64_t pid, double* out) {
  Context* C = (Context*)h;
  Photon ph;
  emit_photon(*C, pid, &ph);
  for (int m = 0; m < 4; m++) { out[m] = ph.x[m]; out[4 + m] = ph.k[m]; out[8 + m] = ph.a[m]; }
  out[12] = ph.w; out[13] = ph.nua_a; out[14] = ph.nua_s; out[15] = ph.bias; out[16] = ph.E0;
  return 0;
}
// final state of chosen primaries + sums over each primary's whole family
int orc_trace(void* h, const int64_t* pids, int n, TraceRec* out, double* fam_wE, int64_t* fam_n) {
  Context* C = (Context*)h;
#pragma omp parallel for schedule(dynamic, 16)
  for (int i = 0; i < n; i++) {
    Photon ph;
    emit_photon(*C, pids[i], &ph);
    Tally tl; tally_init(C->P, &tl);
    Stats st = Stats();
    track_history(*C, ph, &tl, &st, &out[i]);
    if (fam_wE) fam_wE[i] = st.sum_wE_rec;
    if (fam_n) fam_n[i] = st.n_spawned;
  }
  return 0;
}

// ---- bare functions for the pins -----------------------------------------------------------
void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void orc_uniform_pair(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t n, double* out) {
  uniform_pair(seed, tag, c0, c1, c2, n, &out[0], &out[1]);
}
void orc_stream(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, int n, double* out) {
  Stream s(seed, tag, c0, c1, c2);
  for (int i = 0; i < n; i++) out[i] = s.next();
}
// spawn keying (G11): ids of the children of n (parent id, event ordinal j) pairs; parents[n][3], j[n] -> out[n][3]
void orc_child_ids(uint64_t seed, const uint32_t* parents, const uint32_t* j, int64_t n, uint32_t* out) {
  for (int64_t i = 0; i < n; i++) {
    PhotonId par = {parents[3 * i], parents[3 * i + 1], parents[3 * i + 2]};
    PhotonId c = child_id(seed, par, j[i]);
    out[3 * i] = c.i0; out[3 * i + 1] = c.i1; out[3 * i + 2] = c.i2;
  }
}
double orc_K2_direct(double th) { return K2_direct(th); }
double orc_F_direct(double K) { return F_direct(K); }
double orc_sigma_kn(double e) { return sigma_kn_over_T(e); }
double orc_sigma_hot_direct(double th, double e) { return sigma_hot_direct(th, e); }
double orc_K2_eval(double th) { ensure_tables(false); return K2_eval(g_tables, th); }
double orc_F_eval(double K) { ensure_tables(false); return F_eval(g_tables, K); }
double orc_sigma_hot_eval(double th, double e) { ensure_tables(true); return sigma_hot_eval(g_tables, th, e); }
double orc_jnu(double nu, double ne, double th, double B, double sth) { ensure_tables(false); return jnu(g_tables, nu, ne, th, B, sth); }
double orc_jnu_integrated(double nu, double ne, double th, double B) { ensure_tables(false); return jnu_angle_integrated(g_tables, nu, ne, th, B); }
double orc_nu_alpha_abs(double nu, double ne, double th, double B, double sth) { ensure_tables(false); return nu_alpha_abs(g_tables, nu, ne, th, B, sth); }
int orc_get_table(int which, double* out, int n) {   // 0 lnK2, 1 lnF, 2 lnSigH
  ensure_tables(which == 2);
  const std::vector<double>& v = which == 0 ? g_tables.lnK2 : which == 1 ? g_tables.lnF : g_tables.lnSigH;
  if ((size_t)n != v.size()) return -(int)v.size();
  std::memcpy(out, v.data(), v.size() * 8);
  return 0;
}

void orc_gcov(const Params* P, const double* x, double* g) { gcov_func(*P, x, (double(*)[4])g); }
void orc_gcon(const Params* P, const double* x, double* g) { Geom G; geom_func(*P, x, &G); std::memcpy(g, G.gcon, 128); }
double orc_gdet(const Params* P, const double* x) { Geom G; geom_func(*P, x, &G); return G.gdet; }
void orc_dgcov(const Params* P, const double* x, double* dg) { dgcov_func(*P, x, (double(*)[4][4])dg); }
void orc_conn(const Params* P, const double* x, double* c) { conn_func(*P, x, (double(*)[4][4])c); }
double orc_step_size(const Params* P, const double* x, const double* k) { return step_size(*P, x, k); }
int orc_push(const Params* P, const double* x0, const double* k0, const double* a0, double dl, double* x1,
             double* k1, double* a1) {
  int it; bool cap;
  push_photon(*P, x0, k0, a0, dl, x1, k1, a1, &it, &cap);
  return cap ? -it : it;
}
// integrate a vacuum geodesic with the tracker's own step rule; traj[n][8] = x, k per step
int orc_geodesic(const Params* P, const double* x0, const double* k0, int nmax, double* traj) {
  double x[4], k[4], a[4], conn[4][4][4];
  for (int m = 0; m < 4; m++) { x[m] = x0[m]; k[m] = k0[m]; }
  conn_func(*P, x, conn);
  for (int m = 0; m < 4; m++) {
    double s = 0.0;
    for (int al = 0; al < 4; al++) for (int be = 0; be < 4; be++) s += conn[m][al][be] * k[al] * k[be];
    a[m] = -s;
  }
  int n = 0;
  for (; n < nmax; n++) {
    for (int m = 0; m < 4; m++) { traj[n * 8 + m] = x[m]; traj[n * 8 + 4 + m] = k[m]; }
    double r = std::exp(x[1]);
    if (r >= P->r_max || (P->metric_kind == 1 && r <= P->r_horizon_stop)) { n++; break; }
    double dl = step_size(*P, x, k);
    double x1[4], k1[4], a1[4]; int it; bool cap;
    push_photon(*P, x, k, a, dl, x1, k1, a1, &it, &cap);
    for (int m = 0; m < 4; m++) { x[m] = x1[m]; k[m] = k1[m]; a[m] = a1[m]; }
  }
  return n;
}
void orc_tetrad(const Params* P, const double* x, const double* ucon, const double* trial, double* econ) {
  Geom G; geom_func(*P, x, &G);
  make_tetrad(G, ucon, trial, (double(*)[4])econ);
}
// plasma state at x: out = ne, thetae, B, ucon[4], bcon[4], vacuum flag  (12 doubles)
void orc_plasma_at(void* h, const double* x, double* out) {
  Context* C = (Context*)h;
  Geom G; geom_func(C->P, x, &G);
  Plasma S; plasma_at(C->P, C->un, C->prim.data(), x, G, &S);
  out[0] = S.ne; out[1] = S.thetae; out[2] = S.B;
  for (int m = 0; m < 4; m++) { out[3 + m] = S.ucon[m]; out[7 + m] = S.bcon[m]; }
  out[11] = S.vacuum ? 1.0 : 0.0;
}
// fluid-frame photon energy and field angle at x for wavevector k: out = eps, cos(theta_B), nu*alpha_abs,
// nu*alpha_scat, bias (n_sc = nsc), vacuum flag  (6 doubles)
void orc_fluid_frame(void* h, const double* x, const double* k, int nsc, double* out) {
  Context* C = (Context*)h;
  if (C->T.lnK2.empty() || (C->P.scattering_on && !C->T.have_sigh)) { ensure_tables(C->P.scattering_on != 0); C->T = g_tables; }
  Geom G; geom_func(C->P, x, &G);
  Plasma S; plasma_at(C->P, C->un, C->prim.data(), x, G, &S);
  for (int i = 0; i < 6; i++) out[i] = 0.0;
  out[5] = S.vacuum ? 1.0 : 0.0;
  if (S.vacuum) return;
  fluid_frame(*C, k, G, S, &out[0], &out[1]);
  opacities(*C, x, k, G, S, &out[2], &out[3], &out[4], nsc);
}
double orc_zone_volume(const Params* P, int i, int j, int k) { return zone_volume(*P, i, j, k); }
// n positions drawn in zone (i,j,k) with emit_mode 1 (stream TAG_EMIT of ids 0..n-1): out[n][4]
void orc_sample_positions(const Params* P, int i, int j, int k, int n, double* out) {
  for (int q = 0; q < n; q++) {
    Stream rs(P->seed, TAG_EMIT, (uint32_t)q, 0u, 0u);
    sample_zone_position(*P, i, j, k, rs, out + 4 * q);
  }
}
void orc_sample_mj(double thetae, uint64_t seed, int n, double* gamma_out) {
  for (int i = 0; i < n; i++) {
    Stream rs(seed, TAG_SCAT, (uint32_t)i, 0u, 0u);
    double g, b;
    sample_electron_mj(rs, thetae, &g, &b);
    gamma_out[i] = g;
  }
}
// n independent Compton events of a photon of plasma-frame energy eps (units m_e c^2) moving along
// +x1 through static plasma of temperature thetae in flat space: returns scattered plasma-frame energy
// and cosine of the lab scattering angle, plus k'.k' for the nullity pin
void orc_compton_sample(double thetae, double eps, uint64_t seed, int n, double* eps_out, double* cos_out,
                        double* kk_out) {
  ensure_tables(false);
  Context C;
  std::memset(&C.P, 0, sizeof(Params));
  C.P.metric_kind = 0; C.P.hslope = 1.0; C.P.seed = seed;
  C.T = g_tables;
  double x[4] = {0.0, 0.3, 0.37, 0.2};
  Geom G; geom_func(C.P, x, &G);
  Plasma S; S.vacuum = false; S.ne = 1.0; S.thetae = thetae; S.B = 0.0;
  for (int m = 0; m < 4; m++) { S.ucon[m] = 0.0; S.bcon[m] = 0.0; }
  S.ucon[0] = 1.0;
  for (int i = 0; i < n; i++) {
    Photon p;
    for (int m = 0; m < 4; m++) { p.x[m] = x[m]; p.k[m] = 0.0; }
    p.k[0] = eps; p.k[1] = eps / std::sqrt(G.gcov[1][1]);
    p.id.i0 = (uint32_t)i; p.id.i1 = 7u; p.id.i2 = 0u;
    double ko[4];
    bool ok = compton_event(C, p, G, S, 0u, ko);
    if (!ok) { eps_out[i] = cos_out[i] = kk_out[i] = NAN; continue; }
    eps_out[i] = ko[0];
    cos_out[i] = ko[1] * std::sqrt(G.gcov[1][1]) / ko[0];
    kk_out[i] = dot(G.gcov, ko, ko) / (ko[0] * ko[0]);
  }
}

}  // extern "C"
