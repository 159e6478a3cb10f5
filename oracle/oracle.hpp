// ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-history-at-a-time CPU implementation (fp64) of the
// superphoton transport path of GPUmonty (arxiv 2602.13198, /root/reference/PAPER.md),
// written from the paper's equations in the paper's order.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call anything in this directory.  It shares no code, header,
// table or constant generator with paper_2602_13198_b200/csrc (the CUDA path).
//
// Every function cites the PAPER.md passage it follows; where the paper is silent
// or garbled the reading is the numbered "G#" item in DESIGN.md.
//
// Pins (tests/test_oracle_*.py, -m "not gpu") are listed per function in DESIGN.md
// section "Oracle pins".  Functions whose behaviour rests on a reading that no
// external fact fixes are marked  [parity unpinned]  below and in DESIGN.md:
//   step_size (G16), roulette (G15), tetrad axis choice (G13), bias law (G21),
//   KN/Thomson switch thresholds (G22/G25).
#pragma once
#include <cstdint>
#include <cstddef>
#include <vector>

namespace orc {

// ---- CGS constants (G0) -----------------------------------------
constexpr double EE = 4.80320680e-10;
constexpr double CL = 2.99792458e10;
constexpr double ME = 9.1093826e-28;
constexpr double MP = 1.67262171e-24;
constexpr double HPL = 6.6260693e-27;
constexpr double KBOL = 1.3806505e-16;
constexpr double SIGMA_THOMSON = 6.65245873e-25;
constexpr double PI = 3.14159265358979323846;

// ---- parameters: mirrors the dict of workloads.py (own declaration) --------
struct Params {
  double Ns_target;
  double a_spin, hslope;
  double startx[4], dx[4];
  double L_unit, M_unit;
  double thetae_fixed, trat, R_low, R_high, gam_ad, thetae_min, thetae_max;
  double nu_min, nu_max, w_min;
  double step_eps, verlet_tol;
  double r_max, r_horizon_stop;
  double bias0, roulette;
  double nu_lo, nu_hi;
  uint64_t seed;
  int64_t max_steps;
  int32_t metric_kind;  // 0 flat (M=0), 1 Kerr-Schild (M=1)
  int32_t n1, n2, n3;
  int32_t thetae_mode;  // 0 fixed, 1 constant Tp/Te, 2 R_low/R_high
  int32_t verlet_maxit;
  int32_t scattering_on, nsc_max, bias_p_theta, bias_q_nsc;
  int32_t n_th, n_nu, fold_theta;
  int32_t emit_mode;    // 0: emission at the zone centre (G12); 1: uniform in proper volume inside the zone (G31)
  double bias_target;   // on-the-fly bias tuning (G32): target scattered superphotons per parent and generation
  int32_t bias_tune;    // 0 off, 1: tune the per-generation bias factors in prepare()
  int32_t pad_;
};

// ---- Philox4x32-10 (O5 / G11) -------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
enum Tag : uint32_t { TAG_ZONE = 0x5a4f4e45u, TAG_EMIT = 0x454d4954u, TAG_STEP = 0x53544550u,
                      TAG_SCAT = 0x53434154u, TAG_SPAWN = 0x5350574eu };
struct PhotonId { uint32_t i0, i1, i2; };
// sequential uniform stream: block n of (id, tag) yields two doubles
struct Stream {
  uint32_t ctr[4]; uint32_t key[2]; double buf[2]; int have;
  Stream(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t n0 = 0,
         uint32_t key1_xor = 0);   // key = (seed_lo ^ tag, seed_hi ^ key1_xor)
  double next();
};
void uniform_pair(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t n,
                  double* u0, double* u1);
PhotonId child_id(uint64_t seed, PhotonId parent, uint32_t j);

// ---- geometry (O1) ----------------------------
struct Geom { double gcov[4][4], gcon[4][4], gdet; };
double theta_of_x2(const Params& P, double x2);
double dtheta_dx2(const Params& P, double x2);
void gcov_func(const Params& P, const double x[4], double gcov[4][4]);
void dgcov_func(const Params& P, const double x[4], double dg[4][4][4]);  // dg[a][m][n] = d_a g_mn
bool invert4(const double m[4][4], double inv[4][4]);
double det4(const double m[4][4]);
void geom_func(const Params& P, const double x[4], Geom* G);
void conn_func(const Params& P, const double x[4], double conn[4][4][4]);  // conn[m][a][b]
void lower(const double g[4][4], const double v[4], double out[4]);
double dot(const double g[4][4], const double a[4], const double b[4]);

// ---- fluid / plasma state (O2) --------------------------------------
struct Units { double L, T, M, RHO, U, B, Ne; };
Units make_units(const Params& P);
struct Plasma {
  bool vacuum;       // outside the grid in x1
  double ne, thetae, B;       // cgs: cm^-3, dimensionless, gauss
  double ucon[4], bcon[4];    // code units
  double rho, uu;             // interpolated primitives (code)
};
void interp_prim(const Params& P, const double* prim, const double x[4], double out[8], bool* inside);
void plasma_from_prim(const Params& P, const Units& un, const Geom& G, const double pr[8], Plasma* S);
void plasma_at(const Params& P, const Units& un, const double* prim, const double x[4], const Geom& G, Plasma* S);

// ---- radiation processes (O3, O8) ----------
struct Tables {
  // K2: ln K2 at 201 log-uniform Theta nodes on [0.3, 100]
  std::vector<double> lnK2;
  // F(K): ln F at NF+1 log-uniform K nodes on [1e-6, 1e7]
  std::vector<double> lnF;
  // hot cross-section: ln(sigma_h/sigma_T) at (221 eps) x (81 Theta) nodes
  std::vector<double> lnSigH;
  bool have_sigh = false;
};
constexpr int NK2 = 200, NF = 260, NSE = 220, NST = 80, NW = 200;
constexpr double K2_TMIN = 0.3, K2_TMAX = 100.0;
constexpr double F_KMIN = 1e-6, F_KMAX = 1e7;
constexpr double SH_LE0 = -12.0, SH_LE1 = 6.0, SH_LT0 = -4.0, SH_LT1 = 4.0;
double K2_direct(double thetae);                 // std::cyl_bessel_k(2, 1/Theta)
double F_direct(double K);                       // adaptive quadrature of the angle integral
double sigma_kn_over_T(double eps);              // Eq. 26 / Eq. 27
double sigma_hot_direct(double thetae, double eps);  // Eq. 23 by nested adaptive quadrature, / sigma_T
void build_tables(Tables* T, bool with_sigh);
double K2_eval(const Tables& T, double thetae);
double F_eval(const Tables& T, double K);
double sigma_hot_eval(const Tables& T, double thetae, double eps);   // / sigma_T
double jnu(const Tables& T, double nu, double ne, double thetae, double B, double sin_theta);  // Eq. 3
double jnu_angle_integrated(const Tables& T, double nu, double ne, double thetae, double B);
double nu_alpha_abs(const Tables& T, double nu, double ne, double thetae, double B, double sin_theta);

// ---- context ---------------------------------------------------------------
struct ZoneInfo { double A, nu0, C, qmax, Nexp; int32_t n; };
struct Stats {
  int64_t n_primary, n_spawned, n_recorded, n_horizon, n_roulette_killed, n_roulette_survived,
      n_maxstep, n_outofrange, n_steps_total, n_verlet_iters, n_verlet_capped, n_bad_scatter,
      n_analog_killed;
  double sum_w_emit, sum_w_rec, sum_w_horizon, sum_w_roulette_killed, sum_w_roulette_gain,
      sum_w_outofrange, sum_w_maxstep, sum_w_absorbed, sum_wE_emit, sum_wE_rec, sum_w_bad,
      sum_w_spawned;   // total weight w/b handed to scattered superphotons; diagnostic of the Eq. 24-25 pin
};
struct Tally {
  std::vector<double> A, Q, W;  // sum wE, sum (wE)^2, sum w, per [n_th][n_nu]
  std::vector<int64_t> n;
};
struct Photon {
  double x[4], k[4], a[4];   // position, wavevector (units m_e c^2), dk/dlambda at x
  double w;                  // weight
  double nua_a, nua_s, bias; // invariant opacities and bias at x (the "n" values of Eq. 20/25)
  PhotonId id; int32_t nsc; uint32_t nstep; uint32_t jscat;
  double E0;                 // -k_t at creation (diagnostic)
};
struct TraceRec {
  double x[4], k[4], w, E_inf; int64_t nstep; int32_t fate, nsc, ith, inu; uint32_t jscat; uint32_t pad_;
};
enum Fate : int32_t { F_ALIVE = 0, F_RECORDED = 1, F_HORIZON = 2, F_ROULETTE = 3, F_MAXSTEP = 4,
                      F_OUTOFRANGE = 5, F_ANALOG = 6 };

struct Context {
  Params P; Units un; Tables T;
  std::vector<double> prim;
  std::vector<double> nu_nodes, lnw;   // 201 weight-table nodes: nu_k and ln w_k
  std::vector<ZoneInfo> zones;
  std::vector<int64_t> offset;          // exclusive scan of zone counts, size zones+1
  Tally tally; Stats stats;
  // on-the-fly bias tuning (G32): one factor per scattering generation multiplying bias0, and the number of
  // scattered superphotons each generation has spawned (index = n_sc of the parent) since the last reset
  std::vector<double> bias_fac = std::vector<double>(64, 1.0);
  std::vector<int64_t> gen_spawn = std::vector<int64_t>(64, 0);
  int tune_iterations = 0;
  bool prepared = false;
};
void tune_bias(Context* C, int nthreads);

// weights / counts / emission (O4, O6)
void prepare(Context* C);
double zone_volume(const Params& P, int i, int j, int k);     // coordinate volume integral of sqrt(-g) over a zone
void sample_zone_position(const Params& P, int i, int j, int k, Stream& rs, double x[4]);   // G31
double weight_of_nu(const Context& C, double nu);
void make_tetrad(const Geom& G, const double ucon[4], const double trial[4], double econ[4][4]);
void emit_photon(const Context& C, int64_t pid, Photon* ph);

// transport (O7)
double step_size(const Params& P, const double x[4], const double k[4]);
void push_photon(const Params& P, const double x0[4], const double k0[4], const double a0[4], double dl,
                 double x1[4], double k1[4], double a1[4], int* iters, bool* capped);
double bias_func(const Params& P, double thetae, int nsc, double fac = 1.0);
// fluid-frame photon energy eps = -k_mu u^mu (units m_e c^2) and cosine of the angle between the photon and
// the magnetic field in that frame, (k.b)/(eps |b|) (all plasma quantities are fluid-frame)
bool fluid_frame(const Context& C, const double k[4], const Geom& G, const Plasma& S, double* eps, double* cos_b);
void opacities(const Context& C, const double x[4], const double k[4], const Geom& G, const Plasma& S,
               double* nua_a, double* nua_s, double* bias, int nsc);
// Compton event (O8)
bool compton_event(const Context& C, const Photon& parent_at_event, const Geom& G, const Plasma& S,
                   uint32_t j, double kout[4]);
void sample_electron_mj(Stream& rs, double thetae, double* gamma_e, double* beta_e);  // for pins
// history driver: tracks photon and all its descendants; tallies
void track_history(const Context& C, Photon ph, Tally* tl, Stats* st, TraceRec* root_trace, int64_t* gen_spawn = nullptr);
void tally_init(const Params& P, Tally* tl);
void run_range(Context* C, int64_t first, int64_t n, int nthreads);

}  // namespace orc
