// ORACLE (test infrastructure).  Geodesic tracking with absorption, biased scattering and tally.
//
//  push_photon    velocity-Verlet with fixed-point iteration on k, Eqs. 11-15;
//                 G17 (Eq. 11 needs dlambda^2 on its last term), G18 (Eq. 15 as an L1 ratio).
//  step_size      [parity unpinned] the paper never states its step rule; G16.
//  opacities      nu*alpha_nu, nu*n_e*sigma_h (Eq. 24-25).
//  track_history  per-step order of operations: stop tests (r_max), minimum
//                 weight / roulette [parity unpinned, G15], push, Eq. 20 and 25
//                 optical depths, scatter test "b dtau_scat > x1 = -log(rand)",
//                 weight split w(1-1/b) / w/b, Eq. 19 attenuation; scattered
//                 photons are kept on an explicit stack (no recursion).
//  record         detector binning; G26, G27.
//
// Pins (tests/test_oracle_geometry.py, test_oracle_sphere.py, test_oracle_pins.py): straight lines in flat space,
// E / L_z / Carter constant / k.k conservation in Kerr; absorbing uniform sphere closed form;
// weight conservation with absorption off; bias-independence of the scattered spectrum;
// N_s^-1/2 convergence.
#include "oracle.hpp"
#include <algorithm>
#include <cmath>
#include <vector>
#include <omp.h>

namespace orc {

// [parity unpinned] G16
double step_size(const Params& P, const double x[4], const double k[4]) {
  double d2 = x[2] < 1.0 - x[2] ? x[2] : 1.0 - x[2];
  double den = std::fabs(k[1]) + std::fabs(k[2]) / d2 + std::fabs(k[3]) + 1e-300;
  return P.step_eps / den;
}

static void accel_with(const double conn[4][4][4], const double k[4], double a[4]) {
  for (int m = 0; m < 4; m++) {
    double s = 0.0;
    for (int al = 0; al < 4; al++)
      for (int be = 0; be < 4; be++) s += conn[m][al][be] * k[al] * k[be];
    a[m] = -s;
  }
}

void push_photon(const Params& P, const double x0[4], const double k0[4], const double a0[4], double dl,
                 double x1[4], double k1[4], double a1[4], int* iters, bool* capped) {
  for (int m = 0; m < 4; m++) x1[m] = x0[m] + k0[m] * dl + 0.5 * a0[m] * dl * dl;   // Eq. 11 (G17)
  double kp[4];
  for (int m = 0; m < 4; m++) kp[m] = k0[m] + a0[m] * dl;                            // Eq. 12
  double conn[4][4][4];
  conn_func(P, x1, conn);
  int it = 0;
  bool conv = false;
  while (it < P.verlet_maxit) {
    it++;
    accel_with(conn, kp, a1);                                                         // Eq. 13
    double num = 0.0, den = 0.0;
    for (int m = 0; m < 4; m++) {
      k1[m] = k0[m] + 0.5 * (a0[m] + a1[m]) * dl;                                     // Eq. 14
      num += std::fabs(k1[m] - kp[m]);
      den += std::fabs(k1[m]);
    }
    for (int m = 0; m < 4; m++) kp[m] = k1[m];     // "uses Eq. 14 to evaluate Eq. 12"
    if (num < P.verlet_tol * den) { conv = true; break; }                             // Eq. 15 (G18)
  }
  *iters = it;
  *capped = !conv;
}

// [parity unpinned] G21: b = max(1, bias0 * fac * Theta_e^p * (n_sc+1)^q), integer p, q; fac = the tuned factor of
// generation n_sc (G32), 1 without tuning
double bias_func(const Params& P, double thetae, int nsc, double fac) {
  double b = P.bias0 * fac;
  for (int i = 0; i < P.bias_p_theta; i++) b *= thetae;
  for (int i = 0; i < P.bias_q_nsc; i++) b *= (double)(nsc + 1);
  return b > 1.0 ? b : 1.0;
}

// eps = -k.u and cos(theta_B) = k.b/(eps |b|) in the fluid frame; false when eps is not a
// positive finite number.  cos_b is 0 when the field vanishes.
bool fluid_frame(const Context& C, const double k[4], const Geom& G, const Plasma& S, double* eps_out, double* cos_b) {
  double kcov[4];
  lower(G.gcov, k, kcov);
  double eps = 0.0, kb = 0.0;
  for (int m = 0; m < 4; m++) { eps -= kcov[m] * S.ucon[m]; kb += kcov[m] * S.bcon[m]; }
  *eps_out = eps; *cos_b = 0.0;
  if (!(eps > 0.0) || !std::isfinite(eps)) return false;
  if (S.B > 0.0) {
    double bnorm = S.B / C.un.B;
    double c = kb / (eps * bnorm);
    if (c > 1.0) c = 1.0;
    if (c < -1.0) c = -1.0;
    *cos_b = c;
  }
  return true;
}

void opacities(const Context& C, const double x[4], const double k[4], const Geom& G, const Plasma& S,
               double* nua_a, double* nua_s, double* bias, int nsc) {
  (void)x;
  *nua_a = 0.0; *nua_s = 0.0; *bias = 1.0;
  if (S.vacuum) return;
  const Params& P = C.P;
  double eps, c;
  if (!fluid_frame(C, k, G, S, &eps, &c)) return;
  double nu = eps * ME * CL * CL / HPL;
  if (S.thetae >= P.thetae_min && S.B > 0.0) {
    double s = std::sqrt(1.0 - c * c);
    *nua_a = nu_alpha_abs(C.T, nu, S.ne, S.thetae, S.B, s);
  }
  if (P.scattering_on) {
    *nua_s = nu * S.ne * SIGMA_THOMSON * sigma_hot_eval(C.T, S.thetae, eps);
    *bias = bias_func(P, S.thetae, nsc, C.bias_fac[nsc < 63 ? nsc : 63]);
  }
}

void tally_init(const Params& P, Tally* tl) {
  size_t n = (size_t)P.n_th * P.n_nu;
  tl->A.assign(n, 0.0); tl->Q.assign(n, 0.0); tl->W.assign(n, 0.0); tl->n.assign(n, 0);
}

// returns true if recorded in range
static bool record(const Params& P, const Photon& p, const Geom& G, Tally* tl, int* ith, int* inu, double* Einf) {
  double kcov[4];
  lower(G.gcov, p.k, kcov);
  double E = -kcov[0];
  *Einf = E;
  double nu = E * ME * CL * CL / HPL;
  double db = std::log(P.nu_hi / P.nu_lo) / P.n_nu;
  *ith = -1; *inu = -1;
  if (!(E > 0.0) || !std::isfinite(E)) return false;
  double fj = std::floor(std::log(nu / P.nu_lo) / db);
  if (fj < 0.0 || fj >= (double)P.n_nu) return false;
  double th = theta_of_x2(P, p.x[2]);
  th = std::fmod(th, 2.0 * PI);
  if (th < 0.0) th += 2.0 * PI;
  if (th > PI) th = 2.0 * PI - th;
  int it;
  if (P.fold_theta) {
    double tf = th < PI - th ? th : PI - th;
    it = (int)std::floor(tf / (0.5 * PI / P.n_th));
  } else {
    it = (int)std::floor(th / (PI / P.n_th));
  }
  if (it < 0) it = 0;
  if (it > P.n_th - 1) it = P.n_th - 1;
  *ith = it; *inu = (int)fj;
  size_t b = (size_t)it * P.n_nu + (size_t)fj;
  double wE = p.w * E;
  tl->A[b] += wE; tl->Q[b] += wE * wE; tl->W[b] += p.w; tl->n[b] += 1;
  return true;
}

static void fill_trace(TraceRec* tr, const Photon& p, int fate, double Einf, int ith, int inu) {
  if (!tr) return;
  for (int m = 0; m < 4; m++) { tr->x[m] = p.x[m]; tr->k[m] = p.k[m]; }
  tr->w = p.w; tr->E_inf = Einf; tr->nstep = p.nstep; tr->fate = fate; tr->nsc = p.nsc;
  tr->ith = ith; tr->inu = inu; tr->jscat = p.jscat; tr->pad_ = 0;
}

static void track_one(const Context& C, Photon p, std::vector<Photon>* stack, Tally* tl, Stats* st, TraceRec* tr,
                      int64_t* gen_spawn) {
  const Params& P = C.P;
  const double Cfac = HPL * P.L_unit / (ME * CL * CL);
  for (;;) {
    if (p.x[2] < 0.0) { p.x[2] = -p.x[2]; p.k[2] = -p.k[2]; p.a[2] = -p.a[2]; p.x[3] += PI; }
    if (p.x[2] > 1.0) { p.x[2] = 2.0 - p.x[2]; p.k[2] = -p.k[2]; p.a[2] = -p.a[2]; p.x[3] += PI; }
    double r = std::exp(p.x[1]);
    if (r >= P.r_max) {
      Geom G; geom_func(P, p.x, &G);
      int ith, inu; double E;
      bool ok = record(P, p, G, tl, &ith, &inu, &E);
      if (ok) { st->n_recorded++; st->sum_w_rec += p.w; st->sum_wE_rec += p.w * E; }
      else { st->n_outofrange++; st->sum_w_outofrange += p.w; }
      fill_trace(tr, p, ok ? F_RECORDED : F_OUTOFRANGE, E, ith, inu);
      return;
    }
    if (P.metric_kind == 1 && r <= P.r_horizon_stop) {
      st->n_horizon++; st->sum_w_horizon += p.w;
      fill_trace(tr, p, F_HORIZON, 0.0, -1, -1);
      return;
    }
    if ((int64_t)p.nstep >= P.max_steps) {
      st->n_maxstep++; st->sum_w_maxstep += p.w;
      fill_trace(tr, p, F_MAXSTEP, 0.0, -1, -1);
      return;
    }
    double ux, ur;
    uniform_pair(P.seed, TAG_STEP, p.id.i0, p.id.i1, p.id.i2, p.nstep, &ux, &ur);
    if (p.w < P.w_min) {                       // [parity unpinned] G15
      if (ur < 1.0 / P.roulette) {
        st->n_roulette_survived++; st->sum_w_roulette_gain += p.w * (P.roulette - 1.0);
        p.w *= P.roulette;
      } else {
        st->n_roulette_killed++; st->sum_w_roulette_killed += p.w;
        fill_trace(tr, p, F_ROULETTE, 0.0, -1, -1);
        return;
      }
    }
    double dl = step_size(P, p.x, p.k);
    double x1[4], k1[4], a1[4];
    int it; bool cap;
    push_photon(P, p.x, p.k, p.a, dl, x1, k1, a1, &it, &cap);
    st->n_verlet_iters += it; if (cap) st->n_verlet_capped++;
    Geom G1; geom_func(P, x1, &G1);
    Plasma S1; plasma_at(P, C.un, C.prim.data(), x1, G1, &S1);
    double na1, ns1, b1;
    opacities(C, x1, k1, G1, S1, &na1, &ns1, &b1, p.nsc);
    double tau_a = 0.5 * (p.nua_a + na1) * Cfac * dl;      // Eq. 20
    double tau_s = 0.5 * (p.nua_s + ns1) * Cfac * dl;      // Eq. 25
    double b = 0.5 * (p.bias + b1);                        // G19
    bool scattered = false;
    if (P.scattering_on && p.nsc < P.nsc_max && tau_s > 0.0) {
      double xr = -std::log(1.0 - ux);
      if (b * tau_s > xr && p.w / b >= P.w_min) {
        double f = xr / (b * tau_s);
        double xe[4], ke[4], ae[4];
        push_photon(P, p.x, p.k, p.a, f * dl, xe, ke, ae, &it, &cap);
        Geom Ge; geom_func(P, xe, &Ge);
        Plasma Se; plasma_at(P, C.un, C.prim.data(), xe, Ge, &Se);
        if (!Se.vacuum && Se.ne > 0.0) {
          scattered = true;
          st->n_verlet_iters += it; if (cap) st->n_verlet_capped++;
          double w0 = p.w;
          p.w = w0 * std::exp(-f * tau_a);                 // Eq. 19 up to the event
          st->sum_w_absorbed += w0 - p.w;
          for (int m = 0; m < 4; m++) { p.x[m] = xe[m]; p.k[m] = ke[m]; p.a[m] = ae[m]; }
          // child
          Photon c;
          double kout[4];
          bool ok = compton_event(C, p, Ge, Se, p.jscat, kout);
          double wc = p.w / b;
          if (ok) {
            for (int m = 0; m < 4; m++) { c.x[m] = xe[m]; c.k[m] = kout[m]; }
            double conn[4][4][4];
            conn_func(P, xe, conn);
            accel_with(conn, c.k, c.a);
            c.w = wc; c.nsc = p.nsc + 1; c.nstep = 0; c.jscat = 0;
            c.id = child_id(P.seed, p.id, p.jscat);
            opacities(C, c.x, c.k, Ge, Se, &c.nua_a, &c.nua_s, &c.bias, c.nsc);
            double kc[4]; lower(Ge.gcov, c.k, kc); c.E0 = -kc[0];
            stack->push_back(c);
            st->n_spawned++; st->sum_w_spawned += wc;
            if (gen_spawn) gen_spawn[p.nsc < 63 ? p.nsc : 63]++;
          } else {
            st->n_bad_scatter++; st->sum_w_bad += wc;
          }
          p.w = p.w - wc;                                  // w (1 - 1/b)
          p.jscat++;
          opacities(C, p.x, p.k, Ge, Se, &p.nua_a, &p.nua_s, &p.bias, p.nsc);
          p.nstep++;
          st->n_steps_total++;
          if (!(p.w > 0.0)) {                              // analog limit b = 1
            st->n_analog_killed++;
            fill_trace(tr, p, F_ANALOG, 0.0, -1, -1);
            return;
          }
        }
      }
    }
    if (!scattered) {
      double w0 = p.w;
      p.w = w0 * std::exp(-tau_a);                         // Eq. 19
      st->sum_w_absorbed += w0 - p.w;
      for (int m = 0; m < 4; m++) { p.x[m] = x1[m]; p.k[m] = k1[m]; p.a[m] = a1[m]; }
      p.nua_a = na1; p.nua_s = ns1; p.bias = b1;
      p.nstep++;
      st->n_steps_total++;
    }
  }
}

void track_history(const Context& C, Photon ph, Tally* tl, Stats* st, TraceRec* root_trace, int64_t* gen_spawn) {
  std::vector<Photon> stack;
  st->n_primary++; st->sum_w_emit += ph.w; st->sum_wE_emit += ph.w * ph.E0;
  track_one(C, ph, &stack, tl, st, root_trace, gen_spawn);
  while (!stack.empty()) {
    Photon c = stack.back();
    stack.pop_back();
    track_one(C, c, &stack, tl, st, nullptr, gen_spawn);
  }
}

static void stats_add(Stats* a, const Stats& b) {
  a->n_primary += b.n_primary; a->n_spawned += b.n_spawned; a->n_recorded += b.n_recorded;
  a->n_horizon += b.n_horizon; a->n_roulette_killed += b.n_roulette_killed;
  a->n_roulette_survived += b.n_roulette_survived; a->n_maxstep += b.n_maxstep;
  a->n_outofrange += b.n_outofrange; a->n_steps_total += b.n_steps_total;
  a->n_verlet_iters += b.n_verlet_iters; a->n_verlet_capped += b.n_verlet_capped;
  a->n_bad_scatter += b.n_bad_scatter; a->n_analog_killed += b.n_analog_killed;
  a->sum_w_emit += b.sum_w_emit; a->sum_w_rec += b.sum_w_rec; a->sum_w_horizon += b.sum_w_horizon;
  a->sum_w_roulette_killed += b.sum_w_roulette_killed; a->sum_w_roulette_gain += b.sum_w_roulette_gain;
  a->sum_w_outofrange += b.sum_w_outofrange; a->sum_w_maxstep += b.sum_w_maxstep;
  a->sum_w_absorbed += b.sum_w_absorbed; a->sum_wE_emit += b.sum_wE_emit; a->sum_wE_rec += b.sum_wE_rec;
  a->sum_w_bad += b.sum_w_bad; a->sum_w_spawned += b.sum_w_spawned;
}

void run_range(Context* C, int64_t first, int64_t n, int nthreads) {
  if (nthreads < 1) nthreads = 1;
  std::vector<Tally> tls(nthreads);
  std::vector<Stats> sts(nthreads);
  std::vector<std::vector<int64_t>> gens(nthreads, std::vector<int64_t>(64, 0));
  for (int t = 0; t < nthreads; t++) { tally_init(C->P, &tls[t]); sts[t] = Stats(); }
  const int64_t chunk = 1024;
  const int64_t nchunks = (n + chunk - 1) / chunk;
#pragma omp parallel for num_threads(nthreads) schedule(static, 1)
  for (int64_t c = 0; c < nchunks; c++) {
    int t = omp_get_thread_num();
    int64_t lo = first + c * chunk, hi = lo + chunk;
    if (hi > first + n) hi = first + n;
    for (int64_t pid = lo; pid < hi; pid++) {
      Photon ph;
      emit_photon(*C, pid, &ph);
      track_history(*C, ph, &tls[t], &sts[t], nullptr, gens[t].data());
    }
  }
  size_t nb = C->tally.A.size();
  for (int t = 0; t < nthreads; t++) {
    for (size_t b = 0; b < nb; b++) {
      C->tally.A[b] += tls[t].A[b]; C->tally.Q[b] += tls[t].Q[b];
      C->tally.W[b] += tls[t].W[b]; C->tally.n[b] += tls[t].n[b];
    }
    stats_add(&C->stats, sts[t]);
    for (int g = 0; g < 64; g++) C->gen_spawn[g] += gens[t][g];
  }
}

// On-the-fly bias tuning (PAPER.md:369 names it as future work; the bias is there "to prevent
// the number of generated superphotons from becoming excessive", 7-10x N_s in the GRMHD run).  Reading G32: the
// separate scattered-superphoton generations give the counts for free, so one factor per generation is tuned on a
// PILOT -- the first min(n, 32768) primaries and all their descendants, tracked into a scratch tally that is thrown
// away -- until every generation with at least 200 parents spawns bias_target scattered superphotons per parent
// within 5 % (|ln(ratio/target)| < 0.05).  Per generation and iteration, with r = spawned/parents:
//   spawned < 50 (too few to steer by):  fac x 16; if the count has not grown three times running, the factor the
//                                        climb started from is restored and the generation is frozen;
//   else, closer to the target than ever: fac x clamp(target/r, 1/4, 4);
//   else:                                 the best factor so far is restored and the generation is frozen.
// (The ratio is not monotone in the bias: the gate w/b >= w_min removes children that a larger bias makes lighter, so
// a generation can saturate below the target.)  A generation with fewer than 200 parents takes the factor of the one
// before it.  At most 2 nsc_max + 8 iterations.  The factors are then frozen: the run proper does not depend on how it
// is batched or sharded, and any bias leaves the spectrum unbiased
// (test_scattered_spectrum_is_independent_of_the_bias).
void tune_bias(Context* C, int nthreads) {
  const Params& P = C->P;
  std::fill(C->bias_fac.begin(), C->bias_fac.end(), 1.0);
  C->tune_iterations = 0;
  if (!P.bias_tune || !P.scattering_on || P.nsc_max < 1) return;
  const int64_t n_all = C->offset.back();
  const int64_t n_pilot = n_all < 32768 ? n_all : 32768;
  if (n_pilot < 200) return;
  const int G = P.nsc_max < 63 ? P.nsc_max : 63;           // generations 0 .. G-1 can scatter
  Tally keep_t = C->tally; Stats keep_s = C->stats; std::vector<int64_t> keep_g = C->gen_spawn;
  std::vector<double> best_fac(64, 1.0), best_err(64, 1e300), low_base(64, 1.0);
  std::vector<int64_t> last_spawned(64, -1);
  std::vector<int> low_fail(64, 0), in_low(64, 0);
  std::vector<char> frozen(64, 0);
  for (int iter = 0; iter < 2 * G + 8; iter++) {
    tally_init(P, &C->tally); C->stats = Stats(); std::fill(C->gen_spawn.begin(), C->gen_spawn.end(), 0);
    run_range(C, 0, n_pilot, nthreads);
    C->tune_iterations = iter + 1;
    bool done = true;
    int64_t parents = n_pilot;
    for (int g = 0; g < G; g++) {
      const int64_t spawned = C->gen_spawn[g];
      if (parents >= 200) {
        if (!frozen[g]) {
          const double r = (double)spawned / (double)parents;
          const double err = spawned > 0 ? std::fabs(std::log(r / P.bias_target)) : 1e30;
          if (!(err < 0.05)) {
            done = false;
            if (spawned < 50) {
              if (!in_low[g]) { in_low[g] = 1; low_base[g] = C->bias_fac[g]; low_fail[g] = 0; last_spawned[g] = -1; }
              low_fail[g] = spawned > last_spawned[g] ? 0 : low_fail[g] + 1;
              last_spawned[g] = spawned;
              if (low_fail[g] >= 3) { C->bias_fac[g] = low_base[g]; frozen[g] = 1; }
              else C->bias_fac[g] *= 16.0;
            } else if (err < best_err[g]) {
              in_low[g] = 0;
              best_err[g] = err; best_fac[g] = C->bias_fac[g];
              double f = P.bias_target / r;
              if (f > 4.0) f = 4.0;
              if (f < 0.25) f = 0.25;
              C->bias_fac[g] *= f;
            } else {
              C->bias_fac[g] = best_fac[g]; frozen[g] = 1;    // one more pass runs with the restored factor
            }
          }
        }
      } else if (g > 0 && !frozen[g]) {
        C->bias_fac[g] = C->bias_fac[g - 1];
      }
      parents = spawned;
    }
    if (done) break;
  }
  C->tally = keep_t; C->stats = keep_s; C->gen_spawn = keep_g;
}

}  // namespace orc
