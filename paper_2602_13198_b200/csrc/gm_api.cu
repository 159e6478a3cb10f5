// C-ABI of the library (include/gpumonty_b200.h): context, validation, device memory, the batch
// driver (S13; N_s is split into serial batches sized to memory, only the tallies
// persist) and the getters.  No torch types, no CPU fallback.
#include "gm_host.h"
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace gm;

struct gm_ctx {
  gm_params p;
  DevParams P;
  int device = 0, n_sm = 0;
  long nz = 0;
  // device memory
  double* d_prim = nullptr;
  double2* d_cellB = nullptr;                     // per-cell bounds of the cold pass (nz entries)
  double *d_lnK2 = nullptr, *d_lnF = nullptr, *d_lnSigH = nullptr, *d_lnw = nullptr;
  ZoneArrays Z{};
  int n_weight_blocks = 0;
  Tally tally{}; Tally tally_snap{};
  DevStats *d_stats = nullptr, *d_stats_snap = nullptr;
  double *d_spec = nullptr;          // [2][nb]
  int* d_counters = nullptr;         // 72 ints, layout in run_batch
  Photon *d_prim_ph = nullptr, *d_qA = nullptr, *d_qB = nullptr, *d_esc = nullptr;
  Photon *d_parkA = nullptr, *d_parkB = nullptr;   // hot/cold pass hand-over queues (esc_records each)
  Photon* d_wstack = nullptr;                      // per-warp event stacks of the cascade pass (track_wstack_records)
  bool cascade_overflowed = false, cascade_skip = false;   // the free-flight queue overflowed in a cascade: redo that batch without
  int cascade_max = -1;                            // a generation with fewer input records starts the cascade (0: never; default: half the
                                                   // tracker's resident lanes, set in gm_create); GPUMONTY_B200_CASCADE overrides
  int phase_pairs = -1, k_cold = 4;                // -1: automatic (decided by a pilot batch, see gm_run)
  int auto_pairs = -1;                             // the pilot's decision (-1: not taken yet)
  int carry_lanes = 4;                             // straggler hand-over threshold (0: off); GPUMONTY_B200_CARRY overrides
  double pilot_cold_fraction = -1.0;
  int tune_iterations = 0;                         // bias tuning (G32): pilot passes of the last gm_prepare
  long long esc_records = 0;
  long long batch_primaries = 0, queue_records = 0;   // allocated sizes
  long long want_batch = 0, want_queue = 0;
  bool batch_limited_by_memory = false;
  bool have_grid = false, prepared = false;
  long long n_primaries = 0;
  std::string err;
  // per-kernel timing: event pairs recorded around every launch (categories GM_T_*)
  std::vector<cudaEvent_t> ev_pool;
  std::vector<int> ev_cat;       // category of pair i (events 2i, 2i+1)
  size_t ev_used = 0;
  bool timing = false;
};

static void t_begin(gm_ctx* c, int cat, cudaStream_t st) {
  if (!c->timing) return;
  if (c->ev_used + 2 > c->ev_pool.size()) {
    if (c->ev_pool.size() >= 16384) return;
    for (int i = 0; i < 256; i++) { cudaEvent_t e; cudaEventCreate(&e); c->ev_pool.push_back(e); }
  }
  c->ev_cat.push_back(cat);
  cudaEventRecord(c->ev_pool[c->ev_used], st);
  c->ev_used += 1;
}
static void t_end(gm_ctx* c, cudaStream_t st) {
  if (!c->timing || (c->ev_used & 1) == 0) return;
  cudaEventRecord(c->ev_pool[c->ev_used], st);
  c->ev_used += 1;
}
#define TIMED(cat, st, call) do { t_begin(ctx, cat, st); cudaError_t e__ = (call); t_end(ctx, st); \
    if (e__ != cudaSuccess) return fail(ctx, GM_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e__)); } while (0)

static std::string g_create_err;

static int fail(gm_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (c) c->err = buf; else g_create_err = buf;
  return code;
}
#define CK(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) return fail(ctx, GM_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

static void free_run_buffers(gm_ctx* c) {
  cudaFree(c->d_prim_ph); cudaFree(c->d_qA); cudaFree(c->d_qB); cudaFree(c->d_esc);
  cudaFree(c->d_parkA); cudaFree(c->d_parkB); cudaFree(c->d_wstack);
  c->d_prim_ph = c->d_qA = c->d_qB = c->d_esc = c->d_parkA = c->d_parkB = c->d_wstack = nullptr;
  c->batch_primaries = c->queue_records = c->esc_records = 0;
}

static void free_all(gm_ctx* c) {
  if (!c) return;
  free_run_buffers(c);
  cudaFree(c->d_prim); cudaFree(c->d_cellB); cudaFree(c->d_lnK2); cudaFree(c->d_lnF); cudaFree(c->d_lnSigH); cudaFree(c->d_lnw);
  cudaFree(c->Z.A); cudaFree(c->Z.nu0); cudaFree(c->Z.vol); cudaFree(c->Z.Nexp); cudaFree(c->Z.qmax);
  cudaFree(c->Z.n); cudaFree(c->Z.offset); cudaFree(c->Z.partial); cudaFree(c->Z.nu_nodes); cudaFree(c->Z.wk);
  cudaFree(c->Z.blocksum); cudaFree(c->Z.bad);
  cudaFree(c->tally.A); cudaFree(c->tally_snap.A);
  cudaFree(c->d_stats); cudaFree(c->d_stats_snap); cudaFree(c->d_spec); cudaFree(c->d_counters);
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  c->ev_pool.clear();
}

static bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

static int validate(const gm_params* p) {
  if (p->abi_version != GM_ABI_VERSION) return fail(nullptr, GM_ERR_PARAM, "abi_version %u != %u", p->abi_version, GM_ABI_VERSION);
  if (p->metric_kind != 0 && p->metric_kind != 1) return fail(nullptr, GM_ERR_PARAM, "metric_kind must be 0 or 1");
  if (p->n1 < 1 || p->n2 < 1 || p->n3 < 1) return fail(nullptr, GM_ERR_PARAM, "n1,n2,n3 must be >= 1");
  if (!finite_pos(p->Ns_target)) return fail(nullptr, GM_ERR_PARAM, "Ns_target must be > 0");
  if (p->metric_kind == 1 && !(std::fabs(p->a_spin) < 1.0)) return fail(nullptr, GM_ERR_PARAM, "|a_spin| must be < 1");
  if (!(p->hslope > 0.0 && p->hslope <= 1.0)) return fail(nullptr, GM_ERR_PARAM, "hslope must be in (0,1]");
  for (int i = 1; i < 4; i++)
    if (!finite_pos(p->dx[i]) || !std::isfinite(p->startx[i])) return fail(nullptr, GM_ERR_PARAM, "bad startx/dx[%d]", i);
  if (!finite_pos(p->L_unit) || !finite_pos(p->M_unit)) return fail(nullptr, GM_ERR_PARAM, "L_unit, M_unit must be > 0");
  if (p->thetae_mode < 0 || p->thetae_mode > 2) return fail(nullptr, GM_ERR_PARAM, "thetae_mode must be 0, 1 or 2");
  if (!(p->thetae_min >= 0.3)) return fail(nullptr, GM_ERR_PARAM, "thetae_min must be >= 0.3 (range of the K2 table and of Eq. 3)");
  if (!(p->thetae_max >= p->thetae_min)) return fail(nullptr, GM_ERR_PARAM, "thetae_max < thetae_min");
  if (p->thetae_mode == 0 && !finite_pos(p->thetae_fixed)) return fail(nullptr, GM_ERR_PARAM, "thetae_fixed must be > 0");
  if (!finite_pos(p->nu_min) || !(p->nu_max > p->nu_min)) return fail(nullptr, GM_ERR_PARAM, "need 0 < nu_min < nu_max");
  if (!(p->w_min >= 0.0)) return fail(nullptr, GM_ERR_PARAM, "w_min must be >= 0");
  if (!finite_pos(p->step_eps) || !finite_pos(p->verlet_tol) || p->verlet_maxit < 1) return fail(nullptr, GM_ERR_PARAM, "bad step_eps / verlet_tol / verlet_maxit");
  if (!finite_pos(p->r_max)) return fail(nullptr, GM_ERR_PARAM, "r_max must be > 0");
  if (p->max_steps < 1) return fail(nullptr, GM_ERR_PARAM, "max_steps must be >= 1");
  if (p->scattering_on && (!(p->bias0 > 0.0) || p->nsc_max < 0 || p->nsc_max > 60 || p->bias_p_theta < 0 || p->bias_q_nsc < 0 || !(p->roulette > 1.0)))
    return fail(nullptr, GM_ERR_PARAM, "bad scattering parameters");
  if (!(p->roulette > 1.0)) return fail(nullptr, GM_ERR_PARAM, "roulette must be > 1");
  if (p->n_th < 1 || p->n_nu < 1 || !finite_pos(p->nu_lo) || !(p->nu_hi > p->nu_lo)) return fail(nullptr, GM_ERR_PARAM, "bad detector bins");
  if (p->emit_mode != 0 && p->emit_mode != 1) return fail(nullptr, GM_ERR_PARAM, "emit_mode must be 0 or 1");
  if (p->bias_tune != 0 && p->bias_tune != 1) return fail(nullptr, GM_ERR_PARAM, "bias_tune must be 0 or 1");
  if (p->bias_tune && !(p->bias_target > 0.0 && p->bias_target < 100.0)) return fail(nullptr, GM_ERR_PARAM, "bias_target must be in (0, 100)");
  return GM_OK;
}

static void fill_dev_params(gm_ctx* c) {
  const gm_params& p = c->p;
  DevParams& P = c->P;
  memset(&P, 0, sizeof(P));
  P.a_spin = p.metric_kind == 1 ? p.a_spin : 0.0;
  P.hslope = p.hslope;
  P.startx1 = p.startx[1]; P.startx2 = p.startx[2]; P.startx3 = p.startx[3];
  P.dx1 = p.dx[1]; P.dx2 = p.dx[2]; P.dx3 = p.dx[3];
  P.inv_dx1 = 1.0 / p.dx[1]; P.inv_dx2 = 1.0 / p.dx[2]; P.inv_dx3 = 1.0 / p.dx[3];
  P.x1lo = p.startx[1]; P.x1hi = p.startx[1] + p.n1 * p.dx[1];
  P.cell_c1 = -p.startx[1] * P.inv_dx1 - 0.5; P.cell_c2 = -p.startx[2] * P.inv_dx2 - 0.5; P.cell_c3 = -p.startx[3] * P.inv_dx3 - 0.5;
  P.n1 = p.n1; P.n2 = p.n2; P.n3 = p.n3; P.metric_kind = p.metric_kind;
  P.L_unit = p.L_unit;
  P.T_unit = p.L_unit / C_CL;
  const double RHO = p.M_unit / (p.L_unit * p.L_unit * p.L_unit);
  P.B_unit = C_CL * std::sqrt(4.0 * C_PI * RHO);
  P.Ne_unit = RHO / (C_MP + C_ME);
  P.Cfac = C_HPL * p.L_unit / C_MEC2;
  P.thetae_mode = p.thetae_mode;
  P.thetae_fixed = p.thetae_fixed; P.trat = p.trat; P.R_low = p.R_low; P.R_high = p.R_high; P.gam_ad = p.gam_ad;
  P.thetae_min = p.thetae_min; P.thetae_max = p.thetae_max;
  P.nu_min = p.nu_min; P.lnnu_min = std::log(p.nu_min); P.Lam = std::log(p.nu_max / p.nu_min);
  P.inv_Dlw = (double)NW / P.Lam; P.w_min = p.w_min; P.Ns_target = p.Ns_target;
  P.dV = p.dx[1] * p.dx[2] * p.dx[3] * p.L_unit * p.L_unit * p.L_unit;
  P.step_eps = p.step_eps; P.verlet_tol = p.verlet_tol; P.r_max = p.r_max; P.r_horizon_stop = p.r_horizon_stop;
  P.lnr_max = std::log(p.r_max);
  P.lnr_hor = p.r_horizon_stop > 0.0 ? std::log(p.r_horizon_stop) : -1e300;
  P.max_steps = p.max_steps; P.verlet_maxit = p.verlet_maxit;
  P.scattering_on = p.scattering_on; P.nsc_max = p.nsc_max; P.bias_p = p.bias_p_theta; P.bias_q = p.bias_q_nsc;
  P.bias0 = p.bias0; P.roulette = p.roulette; P.inv_roulette = 1.0 / p.roulette;
  for (int g = 0; g < 64; g++) P.bias_fac[g] = 1.0;
  P.n_th = p.n_th; P.n_nu = p.n_nu; P.fold_theta = p.fold_theta; P.emit_mode = p.emit_mode;
  P.nu_lo = p.nu_lo; P.db = std::log(p.nu_hi / p.nu_lo) / p.n_nu; P.inv_db = 1.0 / P.db;
  P.seed_lo = (uint32_t)(p.seed & 0xffffffffu); P.seed_hi = (uint32_t)(p.seed >> 32);
  P.cellB = c->d_cellB;
  P.bound_debug_scale = 1.0;
  if (const char* e = getenv("GPUMONTY_B200_BOUND_SCALE")) { const double v = atof(e); if (v > 0.0 && std::isfinite(v)) P.bound_debug_scale = v; }
  P.prim = c->d_prim; P.lnK2 = c->d_lnK2; P.lnF = c->d_lnF; P.lnSigH = c->d_lnSigH; P.lnw = c->d_lnw;
}

namespace gm {
void note_global_error(const char* msg) { g_create_err = msg ? msg : ""; }
}  // namespace gm

extern "C" {

static int tune_bias(gm_ctx* ctx, cudaStream_t st);

const char* gm_last_error(const gm_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

int gm_create(gm_ctx** out, const gm_params* p) {
  if (!out) return fail(nullptr, GM_ERR_PARAM, "out is NULL");
  *out = nullptr;
  if (!p) return fail(nullptr, GM_ERR_PARAM, "params is NULL");
  int v = validate(p);
  if (v != GM_OK) return v;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0)
    return fail(nullptr, GM_ERR_CUDA, "no CUDA device (%s): this library has no CPU path", cudaGetErrorString(e));
  gm_ctx* ctx = new gm_ctx();
  ctx->p = *p;
  ctx->nz = (long)p->n1 * p->n2 * p->n3;
  cudaDeviceProp prop;
  if (cudaGetDevice(&ctx->device) != cudaSuccess || cudaGetDeviceProperties(&prop, ctx->device) != cudaSuccess) {
    delete ctx;
    return fail(nullptr, GM_ERR_CUDA, "cannot query the CUDA device");
  }
  if (prop.major < 10) {
    int maj = prop.major, mnr = prop.minor;
    delete ctx;
    return fail(nullptr, GM_ERR_CUDA, "device is sm_%d%d; this library is built for sm_100a only", maj, mnr);
  }
  ctx->n_sm = prop.multiProcessorCount;
  const long nz = ctx->nz;
  const int nb = p->n_th * p->n_nu;
  const int nblk = (int)((nz + 255) / 256), ntile = (int)((nz + 1023) / 1024);
  ctx->n_weight_blocks = nblk;
  auto A = [&](void** ptr, size_t bytes) { return cudaMalloc(ptr, bytes ? bytes : 8); };
  bool ok = true;
  ok = ok && A((void**)&ctx->d_prim, nz * 8 * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_cellB, nz * sizeof(double2)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_lnK2, (NK2 + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_lnF, (NF + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_lnSigH, (size_t)(NSE + 1) * (NST + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_lnw, (NW + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.A, nz * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.nu0, nz * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.vol, nz * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.Nexp, nz * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.qmax, nz * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.n, nz * sizeof(int32_t)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.offset, (nz + 1) * sizeof(long long)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.partial, (size_t)nblk * (NW + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.nu_nodes, (NW + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.wk, (NW + 1) * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.blocksum, (size_t)ntile * sizeof(long long)) == cudaSuccess;
  ok = ok && A((void**)&ctx->Z.bad, sizeof(int)) == cudaSuccess;
  // tally: A, Q, W, n contiguous so that snapshot/restore is one copy
  ok = ok && A((void**)&ctx->tally.A, (size_t)nb * 4 * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->tally_snap.A, (size_t)nb * 4 * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_stats, sizeof(DevStats)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_stats_snap, sizeof(DevStats)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_spec, (size_t)nb * 2 * sizeof(double)) == cudaSuccess;
  ok = ok && A((void**)&ctx->d_counters, 72 * sizeof(int)) == cudaSuccess;
  if (!ok) {
    std::string m = cudaGetErrorString(cudaGetLastError());
    free_all(ctx); delete ctx;
    return fail(nullptr, GM_ERR_CUDA, "device allocation failed: %s", m.c_str());
  }
  ctx->tally.Q = ctx->tally.A + nb; ctx->tally.W = ctx->tally.A + 2 * nb;
  ctx->tally.n = (unsigned long long*)(ctx->tally.A + 3 * nb);
  ctx->tally_snap.Q = ctx->tally_snap.A + nb; ctx->tally_snap.W = ctx->tally_snap.A + 2 * nb;
  ctx->tally_snap.n = (unsigned long long*)(ctx->tally_snap.A + 3 * nb);
  fill_dev_params(ctx);
  {
    cudaError_t oe = track_kernel_optin();       // per device: a second context on another GPU needs it again
    if (oe != cudaSuccess) {
      std::string m = cudaGetErrorString(oe);
      free_all(ctx); delete ctx;
      return fail(nullptr, GM_ERR_CUDA, "cudaFuncSetAttribute(track_kernel, max dynamic shared memory): %s", m.c_str());
    }
  }
  ctx->cascade_max = ctx->n_sm * 192;              // half of n_sm x 3 CTAs x 128 lanes: a generation that cannot fill the machine
  if (const char* e = getenv("GPUMONTY_B200_CASCADE")) ctx->cascade_max = atoi(e) < 0 ? 0 : atoi(e);
  if (const char* e = getenv("GPUMONTY_B200_CARRY")) ctx->carry_lanes = atoi(e) < 0 ? 0 : (atoi(e) > 32 ? 32 : atoi(e));
  // parameter-free tables (S0)
  cudaError_t te = gm_build_tables(ctx, nullptr) == GM_OK ? cudaSuccess : cudaErrorUnknown;
  if (te == cudaSuccess) te = cudaMemset(ctx->tally.A, 0, (size_t)nb * 4 * sizeof(double));
  if (te == cudaSuccess) te = cudaMemset(ctx->d_stats, 0, sizeof(DevStats));
  if (te == cudaSuccess) te = cudaDeviceSynchronize();
  if (te != cudaSuccess) {
    std::string m = cudaGetErrorString(te);
    free_all(ctx); delete ctx;
    return fail(nullptr, GM_ERR_CUDA, "table build failed: %s", m.c_str());
  }
  *out = ctx;
  return GM_OK;
}

int gm_build_tables(gm_ctx* ctx, void* cuda_stream) {
  if (!ctx) return GM_ERR_PARAM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TIMED(GM_T_TABLES, st, build_K2_table(ctx->d_lnK2, st));
  TIMED(GM_T_TABLES, st, build_F_table(ctx->d_lnF, st));
  if (ctx->p.scattering_on) TIMED(GM_T_TABLES, st, build_sigh_table(ctx->d_lnSigH, st));
  return GM_OK;
}

void gm_destroy(gm_ctx* ctx) {
  if (!ctx) return;
  cudaDeviceSynchronize();
  free_all(ctx);
  delete ctx;
}

int gm_set_grid(gm_ctx* ctx, const double* prim, int on_device, size_t n_bytes, void* cuda_stream) {
  if (!ctx) return GM_ERR_PARAM;
  if (!prim) return fail(ctx, GM_ERR_PARAM, "prim is NULL");
  if (n_bytes != (size_t)ctx->nz * 8 * sizeof(double))
    return fail(ctx, GM_ERR_PARAM, "n_bytes %zu != n1*n2*n3*8*8 = %zu", n_bytes, (size_t)ctx->nz * 64);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CK(cudaMemcpyAsync(ctx->d_prim, prim, n_bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
  ctx->have_grid = true; ctx->prepared = false;
  return GM_OK;
}

int gm_reset_tally(gm_ctx* ctx) {
  if (!ctx) return GM_ERR_PARAM;
  const int nb = ctx->p.n_th * ctx->p.n_nu;
  CK(cudaMemset(ctx->tally.A, 0, (size_t)nb * 4 * sizeof(double)));
  CK(cudaMemset(ctx->d_stats, 0, sizeof(DevStats)));
  return GM_OK;
}

int gm_prepare(gm_ctx* ctx, void* cuda_stream, int64_t* n_primaries_out) {
  if (!ctx) return GM_ERR_PARAM;
  if (!ctx->have_grid) return fail(ctx, GM_ERR_STATE, "gm_prepare before gm_set_grid");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double nu_nodes[NW + 1];
  const double Dl = ctx->P.Lam / NW;
  for (int k = 0; k <= NW; k++) nu_nodes[k] = ctx->p.nu_min * std::exp(k * Dl);
  CK(cudaMemcpyAsync(ctx->Z.nu_nodes, nu_nodes, sizeof(nu_nodes), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(ctx->Z.bad, 0, sizeof(int), st));
  TIMED(GM_T_PREPARE, st, launch_prepare(ctx->P, ctx->Z, ctx->d_lnw, ctx->nz, st));
  long long total = 0;
  int bad = 0;
  CK(cudaMemcpyAsync(&total, ctx->Z.offset + ctx->nz, sizeof(long long), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(&bad, ctx->Z.bad, sizeof(int), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (bad) return fail(ctx, GM_ERR_GRID, "non-finite value in the fluid grid");
  ctx->n_primaries = total;
  ctx->prepared = true;
  ctx->auto_pairs = -1;
  int r = gm_reset_tally(ctx);
  if (r != GM_OK) return r;
  r = tune_bias(ctx, st);                                   // G32: no-op unless bias_tune
  if (r != GM_OK) return r;
  if (n_primaries_out) *n_primaries_out = total;
  return GM_OK;
}

int gm_get_zone_counts(gm_ctx* ctx, int32_t* counts) {
  if (!ctx || !counts) return GM_ERR_PARAM;
  if (!ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  CK(cudaMemcpy(counts, ctx->Z.n, ctx->nz * sizeof(int32_t), cudaMemcpyDeviceToHost));
  return GM_OK;
}

int gm_get_zone_offsets(gm_ctx* ctx, int64_t* offsets) {
  if (!ctx || !offsets) return GM_ERR_PARAM;
  if (!ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  static_assert(sizeof(long long) == sizeof(int64_t), "offset type");
  CK(cudaMemcpy(offsets, ctx->Z.offset, (ctx->nz + 1) * sizeof(long long), cudaMemcpyDeviceToHost));
  return GM_OK;
}

int gm_get_table(gm_ctx* ctx, int which, double* out, size_t n) {
  if (!ctx || !out) return GM_ERR_PARAM;
  const double* src = nullptr;
  size_t len = 0;
  switch (which) {
    case GM_TABLE_LNK2: src = ctx->d_lnK2; len = NK2 + 1; break;
    case GM_TABLE_LNF: src = ctx->d_lnF; len = NF + 1; break;
    case GM_TABLE_LNSIGH:
      if (!ctx->p.scattering_on) return fail(ctx, GM_ERR_STATE, "sigma_h table is built only when scattering_on");
      src = ctx->d_lnSigH; len = (size_t)(NSE + 1) * (NST + 1); break;
    case GM_TABLE_LNW: src = ctx->d_lnw; len = NW + 1; break;
    case GM_TABLE_NEXP: src = ctx->Z.Nexp; len = ctx->nz; break;
    case GM_TABLE_QMAX: src = ctx->Z.qmax; len = ctx->nz; break;
    default: return fail(ctx, GM_ERR_PARAM, "unknown table %d", which);
  }
  if (which >= GM_TABLE_LNW && !ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  if (n != len) return fail(ctx, GM_ERR_PARAM, "table %d has %zu entries, caller passed %zu", which, len, n);
  CK(cudaMemcpy(out, src, len * sizeof(double), cudaMemcpyDeviceToHost));
  return GM_OK;
}

int gm_set_batch(gm_ctx* ctx, int64_t batch_primaries, int64_t queue_records) {
  if (!ctx) return GM_ERR_PARAM;
  if (batch_primaries < 0 || queue_records < 0 || batch_primaries > (1ll << 30) || queue_records > (1ll << 30))
    return fail(ctx, GM_ERR_PARAM, "batch sizes must be in [0, 2^30]");
  ctx->want_batch = batch_primaries; ctx->want_queue = queue_records;
  cudaDeviceSynchronize();
  free_run_buffers(ctx);
  return GM_OK;
}

// number of hot/cold pass pairs per generation (gm_set_phase_passes)
static int phase_pairs_of(const gm_ctx* ctx) {
  if (ctx->p.metric_kind != 1) return 0;                 // instantiated for the Kerr workloads only
  if (ctx->phase_pairs >= 0) return ctx->phase_pairs;
  if (ctx->p.thetae_mode == 0) return 0;                 // a uniform Theta_e has no cold phase
  return ctx->auto_pairs >= 0 ? ctx->auto_pairs : 3;
}

int gm_set_phase_passes(gm_ctx* ctx, int pairs, int k_cold) {
  if (!ctx) return GM_ERR_PARAM;
  if (pairs > 8 || k_cold < 1 || k_cold > 1000000) return fail(ctx, GM_ERR_PARAM, "pairs must be <= 8 and k_cold in [1, 1e6]");
  ctx->phase_pairs = pairs < 0 ? -1 : pairs; ctx->k_cold = k_cold; ctx->auto_pairs = -1;
  cudaDeviceSynchronize();
  free_run_buffers(ctx);
  return GM_OK;
}

static int ensure_run_buffers(gm_ctx* ctx, long long n_ids) {
  // buffers sized for an earlier, smaller request (a gm_trace of a few thousand ids, a small first gm_run) are
  // re-allocated when a larger id range arrives and the caller did not fix the batch size himself
  const long long default_batch = 1ll << 22;
  if (ctx->d_prim_ph) {
    const bool grow = !ctx->want_batch && ctx->batch_primaries < default_batch && n_ids > ctx->batch_primaries &&
                      !ctx->batch_limited_by_memory;
    if (!grow) return GM_OK;
    CK(cudaDeviceSynchronize());
    free_run_buffers(ctx);
  }
  size_t free_b = 0, total_b = 0;
  CK(cudaMemGetInfo(&free_b, &total_b));
  long long batch = ctx->want_batch ? ctx->want_batch : default_batch;
  if (batch > n_ids && !ctx->want_batch) {
    batch = 1024;
    while (batch < n_ids) batch <<= 1;           // power of two >= n_ids
  }
  // scattered-superphoton queues: 8 records per primary by default (7-10x N_s are generated in
  // total, spread over the scattering generations); the escape queue must hold one whole tracker input
  const bool sc = ctx->p.scattering_on != 0;
  // (without scattering the queue only ever holds re-entrants from free flight: none in flat space)
  const bool kerr = ctx->p.metric_kind == 1;
  auto queue_for = [&](long long b) { return ctx->want_queue ? ctx->want_queue : (sc ? 8 * b : (kerr ? b : 1)); };
  long long queue = queue_for(batch);
  // size the batch from the free device memory (at most half of it)
  const int pairs = phase_pairs_of(ctx);
  const bool want_wstack = ctx->p.scattering_on && ctx->cascade_max > 0;
  auto bytes = [&](long long b, long long q) {      // everything allocated below, the cascade's event stacks included
    return (size_t)(b + 2 * q + (pairs > 0 ? 3 : 1) * (b > q ? b : q) + (want_wstack ? track_wstack_records(ctx->n_sm) : 0)) * sizeof(Photon);
  };
  ctx->batch_limited_by_memory = false;
  while (bytes(batch, queue) > free_b / 2 && batch > 1024) { batch >>= 1; queue = queue_for(batch); ctx->batch_limited_by_memory = true; }
  const long long esc = batch > queue ? batch : queue;
  cudaError_t e = cudaMalloc((void**)&ctx->d_prim_ph, (size_t)batch * sizeof(Photon));
  if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_qA, (size_t)queue * sizeof(Photon));
  if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_qB, (size_t)queue * sizeof(Photon));
  if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_esc, (size_t)esc * sizeof(Photon));
  if (e == cudaSuccess && pairs > 0) e = cudaMalloc((void**)&ctx->d_parkA, (size_t)esc * sizeof(Photon));
  if (e == cudaSuccess && pairs > 0) e = cudaMalloc((void**)&ctx->d_parkB, (size_t)esc * sizeof(Photon));
  if (e == cudaSuccess && want_wstack)
    e = cudaMalloc((void**)&ctx->d_wstack, (size_t)track_wstack_records(ctx->n_sm) * sizeof(Photon));
  if (e != cudaSuccess) {                        // leave no half-allocated state behind (batch_primaries stays 0)
    free_run_buffers(ctx);
    return fail(ctx, GM_ERR_CUDA, "run buffers (%lld primaries, %lld queue records): %s", batch, queue, cudaGetErrorString(e));
  }
  ctx->batch_primaries = batch; ctx->queue_records = queue; ctx->esc_records = esc;
  return GM_OK;
}

// one batch: emit -> per scattering generation [track -> compton (events -> scattered superphotons) -> escape
// (free flight of the leavers; re-entrants are appended behind the scattered superphotons)].  Returns the
// largest queue occupancy seen (device counters may exceed the capacity: overflow).
static int run_batch(gm_ctx* ctx, long long first, int n, const long long* d_ids, TraceBuf trace, bool with_root,
                     Tally tally, DevStats* stats, cudaStream_t st, int* max_queue) {
  // [0] primaries, [1] work counter, [2] free-flight queue (reset per round), [3 + round] queue filled by that round,
  // [64], [65] hand-over queues of the hot/cold passes, [66] count of the null queue, [67] sticky overflow flags set
  // by the consumer kernels (1: a tracker input, 2: the free-flight queue was filled past its capacity)
  int* cnt = ctx->d_counters;
  const int NCNT = 72, MAXROUND = 64 - 3;
  int* oflow = cnt + 67;
  // a generation's own input (primaries, or the scattered queue of the previous round) may overflow legitimately:
  // that case is seen through the queue counts and makes the caller redo the batch in smaller pieces
  int* oflow_in = cnt + 68;
  CK(cudaMemsetAsync(cnt, 0, 72 * sizeof(int), st));
  TIMED(GM_T_EMIT, st, launch_emit(ctx->P, ctx->Z, ctx->nz, first, n, d_ids, ctx->d_prim_ph, cnt + 0, stats, nullptr, with_root, st));
  const int qcap = (int)ctx->queue_records;
  const Photon* in = ctx->d_prim_ph;
  const int* in_count = cnt + 0;
  int in_cap = (int)ctx->batch_primaries;
  const int layers = ctx->p.scattering_on ? ctx->p.nsc_max : 0;
  Queue esc{ctx->d_esc, cnt + 2, (int)ctx->esc_records};
  // automatic schedule: every pass ends with a tail of few long histories, so the passes pay only when a
  // generation fills the machine many times over (measured: profiles/r01c, break-even near 5e5 primaries)
  const bool small_batch = ctx->phase_pairs < 0 && n < (ctx->auto_pairs < 0 ? 1000000 : 500000);
  int pairs = (ctx->d_parkA && !small_batch) ? phase_pairs_of(ctx) : 0;
  // Automatic schedule, decided once per gm_prepare on the first batch of >= 1e6 primaries: the passes pay when the
  // superphotons outlive the hot plasma they start in (configs 2-3: 0.47-0.61 of the primaries are handed over by
  // the first hot pass) and cost when most histories end there (config 4, optically thick with analog
  // scattering: 0.24-0.27; profiles/r01e).  The first hot pass is run, its hand-over count read back, and the
  // generation continues with either schedule.
  bool deciding = ctx->phase_pairs < 0 && ctx->auto_pairs < 0 && pairs > 0 && n >= 1000000;
  Queue nopark{nullptr, cnt + 66, 0};
  Queue parkA{ctx->d_parkA, cnt + 64, (int)ctx->esc_records}, parkB{ctx->d_parkB, cnt + 65, (int)ctx->esc_records};
  int h_counts[NCNT];
  int mq = 0, round = 0;
  bool cascaded = false;
  for (;;) {
    // generations 0..layers are enqueued back to back; the only host round trips inside this block are the schedule
    // pilot (once per gm_prepare) and, for Kerr workloads with scattering, ONE 4-byte read-back per generation from
    // generation 1 on that decides when the cascade pass starts (so gm_run is not asynchronous within a batch);
    // afterwards rounds continue only while re-entrants keep a queue non-empty
    // first block: the nominal generations; afterwards one round per host check (re-entrants from free flight and
    // the descendants of stragglers that were carried into the last nominal round)
    const bool first_block = round == 0;
    const int last = first_block ? layers : round;
    for (; round <= last && round < MAXROUND; round++) {
      Queue out{(round & 1) ? ctx->d_qB : ctx->d_qA, cnt + 3 + round, qcap};
      // stragglers of every generation but the last nominal one continue in the next generation's launch
      const int carry = (ctx->carry_lanes > 0 && first_block && round < last) ? ctx->carry_lanes : 0;
      CK(cudaMemsetAsync(esc.count, 0, sizeof(int), st));
      if (pairs == 0) {
        TIMED(GM_T_TRACK, st, launch_track(ctx->P, 0, in, in_count, in_cap, cnt + 1, out, esc, nopark, 0, carry, tally, stats, trace, oflow_in, ctx->n_sm, st));
      } else {
        // hot pass (in -> parkA), cold pass (parkA -> parkB), hot pass (parkB -> parkA), ... ; the last cold
        // pass handles hot plasma in place.  Every queue is fully consumed before it is refilled.
        const Photon* pin = in; const int* pcount = in_count; int pcap = in_cap;
        for (int pp = 0; pp < pairs; pp++) {
          CK(cudaMemsetAsync(parkA.count, 0, sizeof(int), st));
          TIMED(GM_T_TRACK, st, launch_track(ctx->P, 1, pin, pcount, pcap, cnt + 1, out, esc, parkA, ctx->k_cold, carry, tally, stats, trace, pp == 0 ? oflow_in : oflow, ctx->n_sm, st));
          if (deciding) {
            int parked = 0;
            CK(cudaMemcpyAsync(&parked, parkA.count, sizeof(int), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            ctx->pilot_cold_fraction = (double)parked / (double)n;
            ctx->auto_pairs = ctx->pilot_cold_fraction >= 0.35 ? 3 : 0;
            if (getenv("GPUMONTY_B200_DEBUG"))
              fprintf(stderr, "[gpumonty_b200] %.3f of the primaries leave the first hot pass alive -> %d pass pairs\n",
                      ctx->pilot_cold_fraction, ctx->auto_pairs);
            deciding = false;
            if (ctx->auto_pairs == 0) pairs = 1;           // finish this generation with the mixed pass, then none
          }
          if (pp >= pairs - 1) {
            // what the last hot pass handed over is mostly quiet: one more cold pass takes the steps its bounds decide,
            // the mixed pass finishes the rest in place
            if (pairs > 1) {
              CK(cudaMemsetAsync(parkB.count, 0, sizeof(int), st));
              TIMED(GM_T_TRACK, st, launch_track(ctx->P, 2, parkA.buf, parkA.count, parkA.capacity, cnt + 1, out, esc, parkB, 0, carry, tally, stats, trace, oflow, ctx->n_sm, st));
              TIMED(GM_T_TRACK, st, launch_track(ctx->P, 0, parkB.buf, parkB.count, parkB.capacity, cnt + 1, out, esc, nopark, 0, carry, tally, stats, trace, oflow, ctx->n_sm, st));
            } else
            TIMED(GM_T_TRACK, st, launch_track(ctx->P, 0, parkA.buf, parkA.count, parkA.capacity, cnt + 1, out, esc, nopark, 0, carry, tally, stats, trace, oflow, ctx->n_sm, st));
          } else {
            CK(cudaMemsetAsync(parkB.count, 0, sizeof(int), st));
            TIMED(GM_T_TRACK, st, launch_track(ctx->P, 2, parkA.buf, parkA.count, parkA.capacity, cnt + 1, out, esc, parkB, 0, carry, tally, stats, trace, oflow, ctx->n_sm, st));
            pin = parkB.buf; pcount = parkB.count; pcap = parkB.capacity;
          }
        }
        if (ctx->phase_pairs < 0 && ctx->auto_pairs == 0) pairs = 0;
      }
      TIMED(GM_T_COMPTON, st, launch_compton(ctx->P, out, stats, trace, ctx->n_sm, st));
      TIMED(GM_T_ESCAPE, st, launch_escape(ctx->P, esc, cnt + 1, out, tally, stats, trace, oflow, ctx->n_sm, st));
      in = out.buf; in_count = out.count; in_cap = qcap;
      // Cascade (PHASE_CASCADE): once a generation's input is small, all remaining generations are tracked in one
      // launch (each warp converts and tracks the events of its own lanes); events that do not fit a warp's stack
      // arrive in the next queue and are handled by ordinary rounds.  One 4-byte read-back per generation decides.
      if (ctx->d_wstack && !ctx->cascade_skip && ctx->p.metric_kind == 1 && first_block && round >= 1 && round < last && round + 2 < MAXROUND) {
        int n_next = 0;
        CK(cudaMemcpyAsync(&n_next, out.count, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (n_next > 0 && n_next <= qcap && n_next < ctx->cascade_max) {
          round++;
          Queue out2{(round & 1) ? ctx->d_qB : ctx->d_qA, cnt + 3 + round, qcap};
          Queue wst{ctx->d_wstack, cnt + 66, track_wstack_per_warp()};
          CK(cudaMemsetAsync(esc.count, 0, sizeof(int), st));
          TIMED(GM_T_TRACK, st, launch_track(ctx->P, 3, in, in_count, in_cap, cnt + 1, out2, esc, wst, 0, 0, tally, stats, trace, oflow_in, ctx->n_sm, st));
          TIMED(GM_T_COMPTON, st, launch_compton(ctx->P, out2, stats, trace, ctx->n_sm, st));
          TIMED(GM_T_ESCAPE, st, launch_escape(ctx->P, esc, cnt + 1, out2, tally, stats, trace, oflow, ctx->n_sm, st));
          in = out2.buf; in_count = out2.count; in_cap = qcap;
          round++;
          cascaded = true;
          break;
        }
      }
    }
    CK(cudaMemcpyAsync(h_counts, cnt, NCNT * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    for (int r = 0; r < round; r++) if (h_counts[3 + r] > mq) mq = h_counts[3 + r];
    // the free-flight and hand-over queues hold at most one record per input superphoton and launch, and are sized
    // for a whole tracker input: an overflow there is a logic error, reported, never a silent loss
    // the cascade sends the leavers of ALL remaining generations to the free-flight queue in one launch: if that
    // overflows, the caller restores its snapshot and redoes the batch without the cascade
    if (cascaded && (h_counts[67] & ~2) == 0 && h_counts[64] <= parkA.capacity && h_counts[65] <= parkB.capacity &&
        ((h_counts[67] & 2) || h_counts[2] > esc.capacity)) {
      ctx->cascade_overflowed = true;
      *max_queue = qcap + 1;
      return GM_OK;
    }
    if (h_counts[67] & 4)
      return fail(ctx, GM_ERR_BOUND, "cold-pass bound violated: a superphoton's exact scattering opacity, bias or Theta_e exceeded the "
                  "per-cell upper bound a bounded step was decided with (gm_stats.n_bound_violations); the tally of this run is not "
                  "valid.  Run with gm_set_phase_passes(ctx, 0, ...) (no bounded steps) and report the grid");
    if (h_counts[67] != 0 || h_counts[64] > parkA.capacity || h_counts[65] > parkB.capacity || h_counts[2] > esc.capacity)
      return fail(ctx, GM_ERR_OVERFLOW, "internal queue overflow (flags %d; free-flight %d/%d, hand-over %d, %d/%d records)",
                  h_counts[67], h_counts[2], esc.capacity, h_counts[64], h_counts[65], parkA.capacity);
    if (mq > qcap || h_counts[3 + round - 1] == 0) break;            // overflow (caller redoes) or drained
    if (round >= MAXROUND)
      return fail(ctx, GM_ERR_STATE, "superphotons still re-entering the grid after %d tracker rounds", round);
  }
  *max_queue = mq;
  return GM_OK;
}

// Emit and transport the id range into `tally` / `stats` in batches; an overflowing batch is redone in smaller pieces
// from a snapshot of the accumulators (nothing is dropped silently).
static int run_range(gm_ctx* ctx, int64_t first_id, int64_t n_ids, Tally tally, DevStats* stats, cudaStream_t st) {
  int r = ensure_run_buffers(ctx, n_ids);
  if (r != GM_OK) return r;
  const int nb = ctx->p.n_th * ctx->p.n_nu;
  long long done = 0;
  long long batch = ctx->batch_primaries;
  if (batch < 1) return fail(ctx, GM_ERR_STATE, "run buffers are not allocated");
  TraceBuf notrace{nullptr};
  while (done < n_ids) {
    long long nthis = n_ids - done < batch ? n_ids - done : batch;
    // snapshot so that an overflowing batch can be redone in smaller pieces (nothing is dropped silently)
    CK(cudaMemcpyAsync(ctx->tally_snap.A, tally.A, (size_t)nb * 4 * sizeof(double), cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(ctx->d_stats_snap, stats, sizeof(DevStats), cudaMemcpyDeviceToDevice, st));
    int mq = 0;
    r = run_batch(ctx, first_id + done, (int)nthis, nullptr, notrace, false, tally, stats, st, &mq);
    if (r != GM_OK) { ctx->cascade_skip = false; ctx->cascade_overflowed = false; return r; }
    if (mq > ctx->queue_records) {
      CK(cudaMemcpyAsync(tally.A, ctx->tally_snap.A, (size_t)nb * 4 * sizeof(double), cudaMemcpyDeviceToDevice, st));
      CK(cudaMemcpyAsync(stats, ctx->d_stats_snap, sizeof(DevStats), cudaMemcpyDeviceToDevice, st));
      if (ctx->cascade_overflowed) { ctx->cascade_overflowed = false; ctx->cascade_skip = true; continue; }   // same batch, no cascade
      if (nthis <= 256)
        return fail(ctx, GM_ERR_OVERFLOW, "scattered-superphoton queue (%lld records) overflows with a batch of %lld primaries; "
                    "raise it with gm_set_batch or lower the bias", ctx->queue_records, nthis);
      // shrink in proportion to the overshoot, with a margin
      double shrink = 0.7 * (double)ctx->queue_records / (double)mq;
      long long nb2 = (long long)(nthis * (shrink < 0.5 ? shrink : 0.5));
      batch = nb2 < 256 ? 256 : nb2;
      continue;
    }
    done += nthis;
    ctx->cascade_skip = false;
  }
  return GM_OK;
}

int gm_run(gm_ctx* ctx, int64_t first_id, int64_t n_ids, void* cuda_stream) {
  if (!ctx) return GM_ERR_PARAM;
  if (!ctx->prepared) return fail(ctx, GM_ERR_STATE, "gm_run before gm_prepare");
  if (first_id < 0 || n_ids < 0 || first_id + n_ids > ctx->n_primaries)
    return fail(ctx, GM_ERR_PARAM, "id range [%lld,%lld) outside [0,%lld)", (long long)first_id,
                (long long)(first_id + n_ids), ctx->n_primaries);
  if (n_ids == 0) return GM_OK;
  return run_range(ctx, first_id, n_ids, ctx->tally, ctx->d_stats, (cudaStream_t)cuda_stream);
}

// On-the-fly bias tuning (262-264, 304; G32): one factor per scattering generation, tuned on a
// pilot -- the first min(n, 32768) primaries and their descendants, tracked into a scratch tally -- until every
// generation with >= 200 parents spawns bias_target scattered superphotons per parent within 5 %; the rule is stated
// in DESIGN.md G32 (low counts: x16 until the count stops growing; otherwise x clamp(target/ratio, 1/4, 4) while the
// generation gets closer to the target, else back to its best factor and frozen).  One read-back of the 64
// per-generation counters per pilot pass.  The factors are frozen afterwards.
static int tune_bias(gm_ctx* ctx, cudaStream_t st) {
  const gm_params& p = ctx->p;
  for (int g = 0; g < 64; g++) ctx->P.bias_fac[g] = 1.0;
  ctx->tune_iterations = 0;
  if (!p.bias_tune || !p.scattering_on || p.nsc_max < 1) return GM_OK;
  const long long n_pilot = ctx->n_primaries < 32768 ? ctx->n_primaries : 32768;
  if (n_pilot < 200) return GM_OK;
  const int G = p.nsc_max < 63 ? p.nsc_max : 63;
  const int nb = p.n_th * p.n_nu;
  double* d_tl = nullptr; DevStats* d_st = nullptr;
  CK(cudaMalloc((void**)&d_tl, (size_t)nb * 4 * sizeof(double)));
  if (cudaMalloc((void**)&d_st, sizeof(DevStats)) != cudaSuccess) { cudaFree(d_tl); return fail(ctx, GM_ERR_CUDA, "tune_bias: allocation failed"); }
  Tally scratch{d_tl, d_tl + nb, d_tl + 2 * nb, (unsigned long long*)(d_tl + 3 * nb)};
  double best_fac[64], best_err[64], low_base[64];
  long long last_spawned[64];
  int low_fail[64], in_low[64], frozen[64];
  for (int g = 0; g < 64; g++) { best_fac[g] = 1.0; best_err[g] = 1e300; low_base[g] = 1.0; last_spawned[g] = -1; low_fail[g] = in_low[g] = frozen[g] = 0; }
  int rc = GM_OK;
  DevStats* h = new DevStats;
  double prev_fac[64];                                     // factors of the last pilot pass that ran to its end
  for (int g = 0; g < 64; g++) prev_fac[g] = ctx->P.bias_fac[g];
  for (int iter = 0; iter < 2 * G + 8 && rc == GM_OK; iter++) {
    if (cudaMemsetAsync(d_tl, 0, (size_t)nb * 4 * sizeof(double), st) != cudaSuccess ||
        cudaMemsetAsync(d_st, 0, sizeof(DevStats), st) != cudaSuccess) {
      rc = fail(ctx, GM_ERR_CUDA, "tune_bias: clearing the scratch tally failed"); break;
    }
    rc = run_range(ctx, 0, n_pilot, scratch, d_st, st);
    if (rc == GM_ERR_OVERFLOW && iter > 0) {
      // the last update (a x16 or x4 climb) spawns more than the scattered queue holds even for the smallest batch:
      // the queue capacity caps the climb -- take the step back, freeze those generations, go on with the others
      bool any = false;
      for (int g = 0; g < G; g++)
        if (ctx->P.bias_fac[g] != prev_fac[g]) { ctx->P.bias_fac[g] = prev_fac[g]; frozen[g] = 1; any = true; }
      if (any) { rc = GM_OK; continue; }
    }
    if (rc != GM_OK) break;
    for (int g = 0; g < 64; g++) prev_fac[g] = ctx->P.bias_fac[g];
    if (cudaMemcpyAsync(h, d_st, sizeof(DevStats), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
      rc = fail(ctx, GM_ERR_CUDA, "tune_bias: read-back failed"); break;
    }
    ctx->tune_iterations = iter + 1;
    bool done = true;
    long long parents = n_pilot;
    for (int g = 0; g < G; g++) {
      const long long spawned = (long long)h->gen[g];
      double& fac = ctx->P.bias_fac[g];
      if (parents >= 200) {
        if (!frozen[g]) {
          const double r = (double)spawned / (double)parents;
          const double err = spawned > 0 ? std::fabs(std::log(r / p.bias_target)) : 1e30;
          if (!(err < 0.05)) {
            done = false;
            if (spawned < 50) {
              if (!in_low[g]) { in_low[g] = 1; low_base[g] = fac; low_fail[g] = 0; last_spawned[g] = -1; }
              low_fail[g] = spawned > last_spawned[g] ? 0 : low_fail[g] + 1;
              last_spawned[g] = spawned;
              if (low_fail[g] >= 3) { fac = low_base[g]; frozen[g] = 1; }
              else fac *= 16.0;
            } else if (err < best_err[g]) {
              in_low[g] = 0;
              best_err[g] = err; best_fac[g] = fac;
              double f = p.bias_target / r;
              f = f > 4.0 ? 4.0 : (f < 0.25 ? 0.25 : f);
              fac *= f;
            } else {
              fac = best_fac[g]; frozen[g] = 1;
            }
          }
        }
      } else if (g > 0 && !frozen[g]) {
        fac = ctx->P.bias_fac[g - 1];
      }
      parents = spawned;
    }
    if (done) break;
  }
  delete h;
  cudaFree(d_tl); cudaFree(d_st);
  if (rc != GM_OK) {                                       // no half-tuned table behind a failed gm_prepare
    for (int g = 0; g < 64; g++) ctx->P.bias_fac[g] = 1.0;
    ctx->prepared = false;
  }
  return rc;
}

int gm_get_bias_table(gm_ctx* ctx, double* fac, int64_t* gen_spawn, int* pilot_passes) {
  if (!ctx) return GM_ERR_PARAM;
  if (fac) for (int g = 0; g < 64; g++) fac[g] = ctx->P.bias_fac[g];
  if (gen_spawn) {
    DevStats* h = new DevStats;
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(h, ctx->d_stats, sizeof(DevStats), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) for (int g = 0; g < 64; g++) gen_spawn[g] = (int64_t)h->gen[g];
    delete h;
    if (e != cudaSuccess) return fail(ctx, GM_ERR_CUDA, "gm_get_bias_table: %s", cudaGetErrorString(e));
  }
  if (pilot_passes) *pilot_passes = ctx->tune_iterations;
  return GM_OK;
}

int gm_set_bias_table(gm_ctx* ctx, const double* fac) {
  if (!ctx || !fac) return GM_ERR_PARAM;
  for (int g = 0; g < 64; g++)
    if (!(fac[g] > 0.0) || !std::isfinite(fac[g])) return fail(ctx, GM_ERR_PARAM, "bias factor %d must be positive and finite", g);
  for (int g = 0; g < 64; g++) ctx->P.bias_fac[g] = fac[g];
  return GM_OK;
}

int gm_get_tally(gm_ctx* ctx, double* A, double* Q, double* W, int64_t* n) {
  if (!ctx) return GM_ERR_PARAM;
  const size_t nb = (size_t)ctx->p.n_th * ctx->p.n_nu;
  CK(cudaDeviceSynchronize());
  if (A) CK(cudaMemcpy(A, ctx->tally.A, nb * 8, cudaMemcpyDeviceToHost));
  if (Q) CK(cudaMemcpy(Q, ctx->tally.Q, nb * 8, cudaMemcpyDeviceToHost));
  if (W) CK(cudaMemcpy(W, ctx->tally.W, nb * 8, cudaMemcpyDeviceToHost));
  if (n) CK(cudaMemcpy(n, ctx->tally.n, nb * 8, cudaMemcpyDeviceToHost));
  return GM_OK;
}

int gm_get_spectrum(gm_ctx* ctx, double* nuLnu, double* sigma, int64_t* nphot) {
  if (!ctx) return GM_ERR_PARAM;
  const size_t nb = (size_t)ctx->p.n_th * ctx->p.n_nu;
  TIMED(GM_T_SPECTRUM, 0, launch_spectrum(ctx->P, ctx->tally, ctx->d_spec, ctx->d_spec + nb, 0));
  CK(cudaDeviceSynchronize());
  if (nuLnu) CK(cudaMemcpy(nuLnu, ctx->d_spec, nb * 8, cudaMemcpyDeviceToHost));
  if (sigma) CK(cudaMemcpy(sigma, ctx->d_spec + nb, nb * 8, cudaMemcpyDeviceToHost));
  if (nphot) CK(cudaMemcpy(nphot, ctx->tally.n, nb * 8, cudaMemcpyDeviceToHost));
  return GM_OK;
}

int gm_spectrum_device(gm_ctx* ctx, double* d_nuLnu, double* d_sigma, void* cuda_stream) {
  if (!ctx || !d_nuLnu || !d_sigma) return GM_ERR_PARAM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  TIMED(GM_T_SPECTRUM, st, launch_spectrum(ctx->P, ctx->tally, d_nuLnu, d_sigma, st));
  return GM_OK;
}

int gm_get_stats(gm_ctx* ctx, gm_stats* out) {
  if (!ctx || !out) return GM_ERR_PARAM;
  DevStats h;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(&h, ctx->d_stats, sizeof(h), cudaMemcpyDeviceToHost));
  int64_t* ni = &out->n_primary;
  static_assert(offsetof(gm_stats, n_bound_violations) == 15 * sizeof(int64_t) && offsetof(gm_stats, sum_w_emit) == 16 * sizeof(int64_t), "gm_stats layout");
  for (int i = 0; i < 16; i++) ni[i] = (int64_t)h.n[i];
  double* sd = &out->sum_w_emit;
  for (int i = 0; i < 12; i++) sd[i] = h.s[i];
  return GM_OK;
}

int gm_emit(gm_ctx* ctx, const int64_t* ids, int n, gm_emit_rec* out) {
  if (!ctx || !ids || !out || n < 0) return GM_ERR_PARAM;
  if (!ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  if (n == 0) return GM_OK;
  for (int i = 0; i < n; i++)
    if (ids[i] < 0 || ids[i] >= ctx->n_primaries) return fail(ctx, GM_ERR_PARAM, "id %lld out of range", (long long)ids[i]);
  long long* d_ids = nullptr; gm_emit_rec* d_rec = nullptr;
  CK(cudaMalloc((void**)&d_ids, n * sizeof(long long)));
  CK(cudaMalloc((void**)&d_rec, n * sizeof(gm_emit_rec)));
  CK(cudaMemcpy(d_ids, ids, n * sizeof(long long), cudaMemcpyHostToDevice));
  cudaError_t e = launch_emit(ctx->P, ctx->Z, ctx->nz, 0, n, d_ids, nullptr, nullptr, nullptr, d_rec, false, 0);
  if (e == cudaSuccess) e = cudaMemcpy(out, d_rec, n * sizeof(gm_emit_rec), cudaMemcpyDeviceToHost);
  cudaFree(d_ids); cudaFree(d_rec);
  if (e != cudaSuccess) return fail(ctx, GM_ERR_CUDA, "gm_emit: %s", cudaGetErrorString(e));
  return GM_OK;
}

int gm_trace(gm_ctx* ctx, const int64_t* ids, int n, gm_trace_rec* out) {
  if (!ctx || !ids || !out || n < 0) return GM_ERR_PARAM;
  if (!ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  if (n == 0) return GM_OK;
  for (int i = 0; i < n; i++)
    if (ids[i] < 0 || ids[i] >= ctx->n_primaries) return fail(ctx, GM_ERR_PARAM, "id %lld out of range", (long long)ids[i]);
  int r = ensure_run_buffers(ctx, n);
  if (r != GM_OK) return r;
  const int nb = ctx->p.n_th * ctx->p.n_nu;
  long long* d_ids = nullptr; gm_trace_rec* d_rec = nullptr; DevStats* d_st = nullptr; double* d_tl = nullptr;
  CK(cudaMalloc((void**)&d_ids, n * sizeof(long long)));
  CK(cudaMalloc((void**)&d_rec, n * sizeof(gm_trace_rec)));
  CK(cudaMalloc((void**)&d_st, sizeof(DevStats)));
  CK(cudaMalloc((void**)&d_tl, (size_t)nb * 4 * sizeof(double)));
  Tally scratch{d_tl, d_tl + nb, d_tl + 2 * nb, (unsigned long long*)(d_tl + 3 * nb)};
  int rc = GM_OK;
  long long chunk = ctx->batch_primaries;
  for (long long done = 0; done < n && rc == GM_OK;) {
    long long nthis = n - done < chunk ? n - done : chunk;
    cudaMemset(d_rec + done, 0, nthis * sizeof(gm_trace_rec));
    cudaMemset(d_st, 0, sizeof(DevStats));
    cudaMemset(d_tl, 0, (size_t)nb * 4 * sizeof(double));
    cudaMemcpy(d_ids, ids + done, nthis * sizeof(long long), cudaMemcpyHostToDevice);
    int mq = 0;
    TraceBuf tb{d_rec + done};
    rc = run_batch(ctx, 0, (int)nthis, d_ids, tb, true, scratch, d_st, 0, &mq);
    if (rc == GM_OK && mq > ctx->queue_records && ctx->cascade_overflowed) {
      ctx->cascade_overflowed = false; ctx->cascade_skip = true;
      continue;                                          // the same chunk again, without the cascade
    }
    ctx->cascade_skip = false;
    if (rc == GM_OK && mq > ctx->queue_records) {
      if (nthis <= 16) rc = fail(ctx, GM_ERR_OVERFLOW, "gm_trace: scattered-superphoton queue overflow");
      else { chunk = nthis / 2; continue; }
    }
    done += nthis;
  }
  if (rc == GM_OK && cudaMemcpy(out, d_rec, n * sizeof(gm_trace_rec), cudaMemcpyDeviceToHost) != cudaSuccess)
    rc = fail(ctx, GM_ERR_CUDA, "gm_trace: copy back failed");
  cudaFree(d_ids); cudaFree(d_rec); cudaFree(d_st); cudaFree(d_tl);
  return rc;
}

int gm_eval(gm_ctx* ctx, int what, const double* in, int n, double* out) {
  if (!ctx || !in || !out || n < 0) return GM_ERR_PARAM;
  static const int nin[] = {8, 4, 4, 8, 13, 5, 1, 8}, nout[] = {4, 33, 12, 3, 13, 3, 3, 6};
  if (what < 0 || what > GM_EVAL_BOUND) return fail(ctx, GM_ERR_PARAM, "unknown eval %d", what);
  if ((what == GM_EVAL_PLASMA || what == GM_EVAL_OPAC) && !ctx->have_grid) return fail(ctx, GM_ERR_STATE, "no grid");
  if (what == GM_EVAL_BOUND && !ctx->prepared) return fail(ctx, GM_ERR_STATE, "not prepared");
  if (n == 0) return GM_OK;
  double *d_in = nullptr, *d_out = nullptr;
  CK(cudaMalloc((void**)&d_in, (size_t)n * nin[what] * sizeof(double)));
  CK(cudaMalloc((void**)&d_out, (size_t)n * nout[what] * sizeof(double)));
  cudaError_t e = cudaMemcpy(d_in, in, (size_t)n * nin[what] * sizeof(double), cudaMemcpyHostToDevice);
  DevParams P = ctx->P;
  if (!ctx->p.scattering_on) P.lnSigH = nullptr;
  if (e == cudaSuccess) e = launch_eval(P, what, d_in, n, d_out, 0);
  if (e == cudaSuccess) e = cudaMemcpy(out, d_out, (size_t)n * nout[what] * sizeof(double), cudaMemcpyDeviceToHost);
  cudaFree(d_in); cudaFree(d_out);
  if (e != cudaSuccess) return fail(ctx, GM_ERR_CUDA, "gm_eval: %s", cudaGetErrorString(e));
  return GM_OK;
}

int gm_timing(gm_ctx* ctx, int enable, double* ms_out, int64_t* launches_out) {
  if (!ctx) return GM_ERR_PARAM;
  CK(cudaDeviceSynchronize());
  double ms[GM_T_COUNT] = {0};
  int64_t nl[GM_T_COUNT] = {0};
  for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, ctx->ev_pool[i], ctx->ev_pool[i + 1]) == cudaSuccess) {
      int c = ctx->ev_cat[i / 2];
      ms[c] += t; nl[c] += 1;
    }
  }
  // kernels per launch wrapper: tables 1, prepare 7, others 1
  nl[GM_T_PREPARE] *= 7;
  if (ms_out) for (int c = 0; c < GM_T_COUNT; c++) ms_out[c] = ms[c];
  if (launches_out) for (int c = 0; c < GM_T_COUNT; c++) launches_out[c] = nl[c];
  ctx->ev_used = 0; ctx->ev_cat.clear();
  ctx->timing = enable != 0;
  return GM_OK;
}

void gm_abi_sizes(int out[4]) {
  out[0] = (int)sizeof(gm_params); out[1] = (int)sizeof(gm_stats);
  out[2] = (int)sizeof(gm_trace_rec); out[3] = (int)sizeof(gm_emit_rec);
}

int gm_fp64_peak(double* flops_out, double* sm_clock_mhz_out) {
  if (!flops_out) return GM_ERR_PARAM;
  cudaError_t e = run_fp64_peak(flops_out, sm_clock_mhz_out);
  if (e != cudaSuccess) return fail(nullptr, GM_ERR_CUDA, "gm_fp64_peak: %s", cudaGetErrorString(e));
  return GM_OK;
}

}  // extern "C"
