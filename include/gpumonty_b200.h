/* gpumonty_b200.h -- C-ABI boundary of the B200-native superphoton transport library.
 *
 * The library computes the hot path of the grmonty-style Monte Carlo radiative transfer
 * method described in GPUmonty (arxiv 2602.13198; PAPER.md = /root/reference/PAPER.md):
 * input  = fluid grid + metric/units + sampling/bias/bin parameters + N_s
 *          (PAPER.md:45, 188, 221, 233, 284-286),
 * output = nu L_nu per (theta, nu) detector bin plus per-bin diagnostics.
 * Every step runs in CUDA kernels for sm_100a (paper_2602_13198_b200/csrc); there is no CPU
 * fallback: every entry point returns GM_ERR_CUDA when no usable device is present.
 *
 * Conventions
 *  - Plain C, no exceptions cross the boundary.  Every function returns 0 (GM_OK) or a
 *    negative error code; gm_last_error(ctx) gives a NUL-terminated message owned by ctx
 *    (valid until the next call on that ctx).  A context is not thread-safe.
 *  - The caller owns every pointer it passes and every output buffer.  Unless a parameter
 *    says "device", pointers are HOST pointers.  `cuda_stream` is a cudaStream_t passed as
 *    void* (NULL = the legacy default stream); all work of the call is enqueued on it and the
 *    gm_get_* / gm_trace calls synchronise it before they return.
 *  - Layouts are C order, fp64 unless stated.  Coordinates x = (t, x1 = ln r, x2, x3 = phi)
 *    (PAPER.md:221); theta(x2) = pi x2 + (1-hslope)/2 sin(2 pi x2) (G28).
 *  - Nothing is dropped silently: an internal queue that fills makes gm_run shrink its batch
 *    and redo it (tallies restored), or fail with GM_ERR_OVERFLOW.
 */
#ifndef GPUMONTY_B200_H
#define GPUMONTY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GM_ABI_VERSION 3u

enum {
  GM_OK = 0,
  GM_ERR_PARAM = -1,    /* invalid parameter / NULL pointer / wrong size */
  GM_ERR_STATE = -2,    /* call order (e.g. gm_run before gm_prepare)    */
  GM_ERR_CUDA = -3,     /* CUDA runtime error, or no device              */
  GM_ERR_OVERFLOW = -4, /* scattered-superphoton queue cannot hold one batch of minimum size */
  GM_ERR_GRID = -5,     /* non-finite value in the fluid grid            */
  GM_ERR_BOUND = -6     /* a cold-pass upper bound was exceeded by the exact value (gm_stats.n_bound_violations): the run's tally is void */
};

/* POD parameter block, copied at gm_create.  Field meaning: the comments below and DESIGN.md section 2 (readings G0-G33);
 * the values of the five configs: DESIGN.md section 4.  Same field names as the dict produced by paper_2602_13198_b200.workloads. */
typedef struct gm_params {
  uint32_t abi_version;      /* must equal GM_ABI_VERSION                                            */
  int32_t metric_kind;       /* 0 flat (Kerr-Schild form with M = 0), 1 Kerr-Schild M = 1            */
  uint64_t seed;             /* Philox key (north_star: counter-based RNG keyed per superphoton)     */
  double Ns_target;          /* N_s of Eq. 2                                        */
  double a_spin, hslope;     /* |a| < 1; theta map parameter (G28)                                   */
  double startx[4], dx[4];   /* grid origin and zone size in (t,x1,x2,x3); x2 in [0,1]               */
  int32_t n1, n2, n3;        /* zones; n3 == 1 => axisymmetric                                       */
  int32_t thetae_mode;       /* 0 fixed, 1 constant Tp/Te, 2 R_low/R_high (G3)                       */
  double L_unit, M_unit;     /* cm, g                                            */
  double thetae_fixed, trat, R_low, R_high, gam_ad;
  double thetae_min, thetae_max; /* emission/absorption only for Theta_e >= thetae_min (>= 0.3)      */
  double nu_min, nu_max;     /* sampled frequency range of Eq. 7               */
  double w_min;              /* "minimum weight": floor of Eq. 2, roulette threshold  */
  double step_eps;           /* geodesic step parameter (G16)                                        */
  double verlet_tol;         /* Eq. 15 tolerance, paper default 1e-3                  */
  double r_max;              /* record when r >= r_max                           */
  double r_horizon_stop;     /* Kerr only: kill when r <= this                                       */
  double bias0;              /* b = max(1, bias0 Theta_e^p (n_sc+1)^q) (G21) */
  double roulette;           /* survival gain of the weight roulette (G15)                           */
  double nu_lo, nu_hi;       /* detector frequency range                         */
  int64_t max_steps;         /* per-superphoton step cap (counted, must stay ~0)                     */
  int32_t verlet_maxit;      /* cap on Eq. 12-14 iterations                                          */
  int32_t scattering_on, nsc_max, bias_p_theta, bias_q_nsc;
  int32_t n_th, n_nu, fold_theta; /* detector bins; fold_theta: theta and pi-theta share a bin (G27) */
  int32_t emit_mode;         /* 0: superphotons are born at the zone centre (G12); 1: uniform in proper volume inside
                                the zone, zone volumes exact (G31)             */
  double bias_target;        /* bias tuning (G32): target scattered superphotons per parent, per
                                scattering generation                                                             */
  int32_t bias_tune;         /* 0: b from bias0 alone; 1: gm_prepare tunes one factor per generation on a pilot   */
  int32_t pad_;
} gm_params;

/* Run counters (PAPER.md:316 counts emitted + scattered superphotons; invariants of DESIGN.md O7). */
typedef struct gm_stats {
  int64_t n_primary, n_spawned, n_recorded, n_horizon, n_roulette_killed, n_roulette_survived,
      n_maxstep, n_outofrange, n_steps_total, n_verlet_iters, n_verlet_capped, n_bad_scatter,
      n_analog_killed,
      n_steps_free,   /* of n_steps_total: steps taken in free flight beyond the grid (escape kernel) */
      n_reentered,    /* superphotons that came back into the grid from free flight                  */
      n_bound_violations; /* records whose exact scattering opacity / bias / Theta_e exceeded the per-cell upper bound the cold
                             pass had decided a step with; any non-zero value makes gm_run fail (GM_ERR_BOUND) */
  double sum_w_emit, sum_w_rec, sum_w_horizon, sum_w_roulette_killed, sum_w_roulette_gain,
      sum_w_outofrange, sum_w_maxstep, sum_w_absorbed, sum_wE_emit, sum_wE_rec, sum_w_bad,
      sum_w_spawned;  /* total weight w/b given to scattered superphotons                       */
} gm_stats;

/* Final state of one primary superphoton and sums over its family (primary + descendants). */
typedef struct gm_trace_rec {
  double x[4], k[4];     /* position / wavevector (units m_e c^2) where the primary stopped           */
  double w, E_inf;       /* final weight; -k_t when recorded, else 0                                   */
  int64_t nstep;         /* steps taken by the primary                                                 */
  int32_t fate;          /* GM_FATE_*                                                                  */
  int32_t nsc;           /* scattering generation (0 for a primary)                                    */
  int32_t ith, inu;      /* detector bin, or -1                                                        */
  uint32_t jscat;        /* scattering events the primary underwent                                    */
  uint32_t pad_;
  double fam_wE;         /* sum of w * E_inf over every recorded member of the family                 */
  int64_t fam_nspawn;    /* scattered superphotons spawned in the family                               */
} gm_trace_rec;

enum { GM_FATE_ALIVE = 0, GM_FATE_RECORDED = 1, GM_FATE_HORIZON = 2, GM_FATE_ROULETTE = 3,
       GM_FATE_MAXSTEP = 4, GM_FATE_OUTOFRANGE = 5, GM_FATE_ANALOG = 6 };

/* State of a primary right after emission sampling (Eq. 7-9). */
typedef struct gm_emit_rec {
  double x[4], k[4], a[4]; /* a = dk/dlambda = -Gamma k k (Eq. 10)                        */
  double w, nua_a, nua_s, bias, E0; /* weight, nu*alpha_abs, nu*alpha_scat, bias, -k_t                 */
} gm_emit_rec;

enum { GM_TABLE_LNK2 = 0,   /* 201 : ln K2(1/Theta), Theta log-uniform on [0.3,100] (G6)  */
       GM_TABLE_LNF = 1,    /* 261 : ln F(K), K log-uniform on [1e-6,1e7] (angle integral of Eq. 3; G7) */
       GM_TABLE_LNSIGH = 2, /* 221x81 : ln(sigma_h/sigma_T)(eps, Theta) (Eq. 23; G23) */
       GM_TABLE_LNW = 3,    /* 201 : ln w(nu_k) of Eq. 2 (after gm_prepare)                            */
       GM_TABLE_NEXP = 4,   /* zones : expected superphotons per zone, Eq. 5 (after gm_prepare)        */
       GM_TABLE_QMAX = 5    /* zones : max_k dN/dln nu / C_i, Eq. 8 denominator (after gm_prepare)     */ };

enum { GM_EVAL_ACCEL = 0,   /* in x[4],k[4]            -> out a[4] = -Gamma^m_ab k^a k^b (Eq. 10)       */
       GM_EVAL_GEOM = 1,    /* in x[4]                 -> out gcov[16], gcon[16], sqrt(-g)  (33)        */
       GM_EVAL_PLASMA = 2,  /* in x[4]                 -> out ne,thetae,B,ucon[4],bcon[4],vacuum (12)   */
       GM_EVAL_OPAC = 3,    /* in x[4],k[4]            -> out nu*alpha_abs, nu*alpha_scat, bias (nsc=0) */
       GM_EVAL_PUSH = 4,    /* in x[4],k[4],a[4],dl    -> out x[4],k[4],a[4],iters (Eq. 11-15)          */
       GM_EVAL_RAD = 5,     /* in nu,ne,thetae,B,sin   -> out j_nu (Eq. 3), nu*alpha (Eq. 16/20), sigma_h/sigma_T(thetae, h nu/m c^2) */
       GM_EVAL_NB = 6,      /* in x                    -> out the hot loop's branch-free 1/x, sqrt(x), exp(x) */
       GM_EVAL_BOUND = 7    /* in x[4],k[4] (after gm_prepare) -> out k^t S, Theta_B of the point's interpolation cell (the cold
                               pass's upper bounds), then the exact nu*alpha_scat, Theta_e, bias(Theta_B),
                               bias(Theta_e) at the point (nsc = 0) */ };

typedef struct gm_ctx gm_ctx; /* opaque; owned by the library */

/* Validate and copy the parameters, select the current CUDA device, build the parameter-free
 * device tables (K2, F, sigma_h if scattering_on).  *out is NULL on failure (message via
 * gm_last_error(NULL)). */
int gm_create(gm_ctx** out, const gm_params* p);
void gm_destroy(gm_ctx* ctx);
/* (Re)build the parameter-free device tables K2, F and (if scattering_on) sigma_h on `cuda_stream`
 * (PAPER.md:166, 188).  gm_create calls it once; a benchmark may call it per step. */
int gm_build_tables(gm_ctx* ctx, void* cuda_stream);
/* Message of the last failing call on ctx (ctx == NULL: of the last failing context-free call, i.e. gm_create,
 * gm_fp64_peak or gm_scan_counts_static). */
const char* gm_last_error(const gm_ctx* ctx);

/* Fluid grid prim[n1][n2][n3][8] = rho, u, u~1, u~2, u~3, B1, B2, B3 in code units, zone-major fp64
 * (PAPER.md:188, 284).  `prim` is a host pointer (on_device = 0) or a device pointer (on_device = 1);
 * n_bytes must equal n1*n2*n3*8*sizeof(double).  The library copies it (device to device when
 * on_device) on `cuda_stream`; the caller's buffer may be released once the stream has drained. */
int gm_set_grid(gm_ctx* ctx, const double* prim, int on_device, size_t n_bytes, void* cuda_stream);

/* Weights w(nu_k) (Eq. 2), per-zone expected and integer counts (Eq. 5; one Philox draw per zone),
 * Eq. 8 maxima and the exclusive prefix sum of the counts.  *n_primaries_out (may be NULL) receives
 * the number of primary superphotons; ids 0..n-1 are assigned in zone order.  Resets the tally. */
int gm_prepare(gm_ctx* ctx, void* cuda_stream, int64_t* n_primaries_out);

int gm_get_zone_counts(gm_ctx* ctx, int32_t* counts /* [n1*n2*n3] */);
/* The exclusive prefix sum gm_prepare formed from those counts: offsets[z] = id of the first primary of zone z,
 * offsets[n1*n2*n3] = number of primaries.  `offsets` is a HOST array of n1*n2*n3 + 1 values. */
int gm_get_zone_offsets(gm_ctx* ctx, int64_t* offsets /* [n1*n2*n3 + 1] */);

/* The same prefix sum (zone counts -> which zone a primary id belongs to) as a
 * stand-alone call that allocates nothing -- no cudaMalloc / cudaFree, no allocating library routine, no context.
 *
 * Who needs it: code that is not allowed to ask the CUDA allocator for memory at the point where it wants the scan.
 * Typical cases are a module hosted by an application whose own pool has reserved the device and forbids outside
 * allocations, and a latency-bound loop that cannot afford cudaMalloc's implicit device-wide synchronisation.  Such a
 * caller cannot use gm_create / gm_prepare (they allocate); it brings its own buffers and calls this instead.
 *
 *   d_counts   DEVICE, n_zones int32 values >= 0 (the caller's; read only)
 *   d_offsets  DEVICE, n_zones + 1 int64 values (the caller's): d_offsets[z] = sum of d_counts[0..z), the last
 *              one the total.  Bit-identical to what gm_prepare computes (gm_get_zone_offsets).
 *   n_zones    0 .. GM_SCAN_STATIC_MAX_ZONES.  Anything larger is refused with GM_ERR_PARAM and a message naming the
 *              limit; nothing is launched.  The limit exists because the partial sums between the phases of the scan
 *              (one int64 per 1024 zones) sit in a fixed 32 KiB array compiled into the library.  Every GPU that loads
 *              the library carries that array until the process ends, used or not; it cannot be resized or released.
 *
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device current)
 * and makes CUDA load the kernels; make that first call outside any stream capture.  Later calls only enqueue three
 * small kernels on `cuda_stream` and return without synchronising.
 * All calls on one device share the one array.  It keeps whatever the previous call left there; that is harmless
 * (each call overwrites every element it later reads), but two calls that can run on the GPU at the same time --
 * different streams, or different host threads on different streams -- overwrite each other's partial sums and return
 * garbage.  Keep calls on one stream, or order them with events.
 * Errors: GM_ERR_PARAM (NULL pointer, n_zones out of range), GM_ERR_CUDA (no device, look-up or launch failed); the text
 * is available from gm_last_error(NULL). */
#define GM_SCAN_STATIC_MAX_ZONES 4194304 /* 4096 tiles of 1024 zones; cfg3's 192x128x128 grid has 3,145,728 */
int gm_scan_counts_static(const int32_t* d_counts, int64_t n_zones, int64_t* d_offsets, void* cuda_stream);
/* Copy a table to `out`; n must equal the table's length (else GM_ERR_PARAM). */
int gm_get_table(gm_ctx* ctx, int which, double* out, size_t n);

/* Emit and transport primaries first_id .. first_id+n_ids-1 and all their descendants, adding to
 * the tally.  Asynchronous on `cuda_stream` except for one overflow check per internal batch. */
int gm_run(gm_ctx* ctx, int64_t first_id, int64_t n_ids, void* cuda_stream);
/* Upper bound on primaries per internal batch and capacity of the scattered-superphoton queue
 * (records).  0 keeps the default.  Call before the first gm_run. */
int gm_set_batch(gm_ctx* ctx, int64_t batch_primaries, int64_t queue_records);
/* Tracker schedule (a tuning knob; no result depends on it).  Absorption (PAPER.md:114-140,
 * Eq. 16-20) is evaluated only where Theta_e >= thetae_min, and the scattering test can be decided far
 * from the torus with per-cell upper bounds; each scattering generation can therefore be tracked in `pairs` hot/cold
 * pass pairs: a hot pass (the full step) hands a superphoton over after `k_cold` consecutive quiet steps (not in hot
 * plasma, b tau_s < 1/64), a cold pass takes only steps its bounds decide and hands everything else back, a last
 * mixed pass does everything in place.  pairs = 0: one mixed pass; pairs > 0 is honoured for metric_kind = 1 only;
 * pairs < 0 (default): automatic -- none for batches below 5e5 primaries or a uniform Theta_e; otherwise the first
 * hot pass of the first batch of >= 1e6 primaries after gm_prepare is run, and 3 pairs are used from then on if it
 * handed over >= 0.35 of its primaries, else none.  k_cold >= 1.  Call before the first gm_run (run buffers are
 * re-allocated). */
int gm_set_phase_passes(gm_ctx* ctx, int pairs, int k_cold);

/* Bias tuning (262-264, 304; G32).  With gm_params.bias_tune = 1, gm_prepare tunes one factor per
 * scattering generation, b = max(1, bias0 fac[n_sc] Theta_e^p (n_sc+1)^q), on a pilot (the first min(n, 32768) primaries
 * and their descendants, scratch tally) until each generation with >= 200 parents spawns gm_params.bias_target scattered
 * superphotons per parent within 5 %; the factors are then frozen, so a run does not depend on its batching or sharding.
 * gm_get_bias_table: fac[64] (may be NULL), gen_spawn[64] = scattered superphotons spawned by each generation since the
 * last gm_reset_tally / gm_prepare (may be NULL), *pilot_passes (may be NULL).  gm_set_bias_table: install 64 factors
 * (e.g. those another context tuned); gm_prepare resets them to 1 (or tunes them again). */
int gm_get_bias_table(gm_ctx* ctx, double* fac, int64_t* gen_spawn, int* pilot_passes);
int gm_set_bias_table(gm_ctx* ctx, const double* fac);

/* nu L_nu [erg/s], its Monte Carlo sigma [erg/s] and the number of superphotons per [n_th][n_nu]
 * bin (O9).  Any of the three may be NULL. */
int gm_get_spectrum(gm_ctx* ctx, double* nuLnu, double* sigma, int64_t* nphot);
/* Same scaling written to caller-owned DEVICE buffers [n_th][n_nu] on `cuda_stream`, no synchronisation. */
int gm_spectrum_device(gm_ctx* ctx, double* d_nuLnu, double* d_sigma, void* cuda_stream);
/* Raw accumulators per bin: sum wE, sum (wE)^2, sum w, count.  Any may be NULL. */
int gm_get_tally(gm_ctx* ctx, double* A, double* Q, double* W, int64_t* n);
int gm_get_stats(gm_ctx* ctx, gm_stats* out);
int gm_reset_tally(gm_ctx* ctx);

/* Diagnostics for parity tests: state of chosen primaries after emission; final state of chosen
 * primaries with family sums (runs those histories into a scratch tally; the main tally is untouched). */
int gm_emit(gm_ctx* ctx, const int64_t* ids, int n, gm_emit_rec* out);
int gm_trace(gm_ctx* ctx, const int64_t* ids, int n, gm_trace_rec* out);
/* Evaluate one device function of the path on n inputs (GM_EVAL_*): `in` and `out` are HOST arrays
 * of n rows with the row lengths listed at GM_EVAL_*. */
int gm_eval(gm_ctx* ctx, int what, const double* in, int n, double* out);

/* Per-kernel device times.  Returns, per category GM_T_*, the summed CUDA-event duration [ms] and the
 * number of kernel launches since the previous gm_timing call, then clears the record and switches
 * recording on (enable != 0) or off.  Synchronises the device.  ms_out / launches_out: [GM_T_COUNT]. */
enum { GM_T_TABLES = 0, GM_T_PREPARE = 1, GM_T_EMIT = 2, GM_T_TRACK = 3, GM_T_COMPTON = 4, GM_T_SPECTRUM = 5,
       GM_T_ESCAPE = 6, GM_T_COUNT = 7 };
int gm_timing(gm_ctx* ctx, int enable, double* ms_out, int64_t* launches_out);

/* sizeof(gm_params), sizeof(gm_stats), sizeof(gm_trace_rec), sizeof(gm_emit_rec): lets a binding check its
 * struct layouts against the library's. */
void gm_abi_sizes(int out[4]);

/* DFMA-chain microbenchmark: FP64 FLOP/s of the plain FP64 pipe of the current device (the
 * roofline denominator of the tracker). */
int gm_fp64_peak(double* flops_out, double* sm_clock_mhz_out);

#ifdef __cplusplus
}
#endif
#endif /* GPUMONTY_B200_H */
