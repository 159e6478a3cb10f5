// Shared device declarations of the CUDA path: constants, the device parameter block, Philox,
// photon record.  (The CPU oracle under oracle/ shares nothing with this tree.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/gpumonty_b200.h"

namespace gm {

// ---- CGS constants (G0) ---------------------------------------------------------
constexpr double C_EE = 4.80320680e-10;
constexpr double C_CL = 2.99792458e10;
constexpr double C_ME = 9.1093826e-28;
constexpr double C_MP = 1.67262171e-24;
constexpr double C_HPL = 6.6260693e-27;
constexpr double C_SIGT = 6.65245873e-25;
constexpr double C_PI = 3.14159265358979323846;
constexpr double C_MEC2 = C_ME * C_CL * C_CL;
constexpr double C_MEC2_H = C_MEC2 / C_HPL;          // nu = eps * C_MEC2_H
constexpr double C_H_MEC2 = C_HPL / C_MEC2;          // eps = nu * C_H_MEC2
constexpr double C_NUC_B = C_EE / (2.0 * C_PI * C_ME * C_CL);   // nu_c = C_NUC_B * B
// sqrt(2) pi e^2/(3c): prefactor of Eq. 3 in the Leung et al. (2011) form (G1)
constexpr double C_JPREF = 1.4142135623730951 * C_PI * C_EE * C_EE / (3.0 * C_CL);
constexpr double C_2_11_12 = 1.8877486253633870;     // 2^(11/12)

// ---- table geometry (G6, G7, G23) -------------------------------------------------
constexpr int NK2 = 200, NF = 260, NSE = 220, NST = 80, NW = 200;
constexpr double K2_TMIN = 0.3, K2_TMAX = 100.0;
constexpr double F_KMIN = 1e-6, F_KMAX = 1e7;
constexpr double SH_LE0 = -12.0, SH_LE1 = 6.0, SH_LT0 = -4.0, SH_LT1 = 4.0;

// Philox stream tags (O5 / G11)
constexpr uint32_t TAG_ZONE = 0x5a4f4e45u, TAG_EMIT = 0x454d4954u, TAG_STEP = 0x53544550u,
                   TAG_SCAT = 0x53434154u, TAG_SPAWN = 0x5350574eu;

// ---- device parameter block: gm_params + derived constants + table pointers -------------------
struct DevParams {
  // geometry / grid
  double a_spin, hslope;
  double startx1, startx2, startx3, dx1, dx2, dx3, inv_dx1, inv_dx2, inv_dx3;
  double x1lo, x1hi;
  double cell_c1, cell_c2, cell_c3;                   // -startx/dx - 1/2: stencil index of a coordinate as one FMA (cell_index)
  int n1, n2, n3, metric_kind;
  // units
  double L_unit, T_unit, B_unit, Ne_unit, Cfac;       // Cfac = h L_unit/(m_e c^2)
  // electrons
  int thetae_mode, pad0;
  double thetae_fixed, trat, R_low, R_high, gam_ad, thetae_min, thetae_max;
  // emission
  double nu_min, lnnu_min, Lam, inv_Dlw, w_min, Ns_target, dV;   // Lam = ln(nu_max/nu_min), Dlw = Lam/NW
  // transport
  double step_eps, verlet_tol, r_max, r_horizon_stop, lnr_max, lnr_hor;
  long long max_steps;
  int verlet_maxit;
  // scattering
  int scattering_on, nsc_max, bias_p, bias_q, pad1;
  double bias0, roulette, inv_roulette;
  double bias_fac[64];                                // tuned factor per scattering generation (G32); 1 without tuning
  // tally
  int n_th, n_nu, fold_theta, emit_mode;
  double nu_lo, inv_db, db;
  // RNG
  uint32_t seed_lo, seed_hi;
  // device pointers
  const double* __restrict__ prim;
  const double* __restrict__ lnK2;
  const double* __restrict__ lnF;
  const double* __restrict__ lnSigH;
  const double* __restrict__ lnw;
  // per interpolation cell (indexed like its lowest corner zone): {S, Theta_B}, upper bounds of the scattering
  // opacity per unit k^t and of Theta_e anywhere in the cell (cell_bound_kernel; the tracker's cold pass)
  const double2* __restrict__ cellB;
  double bound_debug_scale;                           // 1; GPUMONTY_B200_BOUND_SCALE (read at gm_create) multiplies S: lets a test
                                                      // shrink the bound on purpose and watch the run-time guard fire
};

// ---- superphoton record (160 B, 16-B aligned) -------------------------------------------------
struct __align__(16) Photon {
  double x[4], k[4], a[4];
  double w, nua_a, nua_s, bias;
  uint32_t id0, id1, id2, nstep;
  int32_t nsc; uint32_t jscat; int32_t root; int32_t flags;
};
static_assert(sizeof(Photon) == 160, "Photon record must be 160 bytes");

// per-run device accumulators
struct DevStats {
  unsigned long long n[16];
  double s[12];
  unsigned long long gen[64];                         // scattered superphotons spawned by generation n_sc (G32)
};
enum { SN_PRIMARY = 0, SN_SPAWNED, SN_RECORDED, SN_HORIZON, SN_ROUL_KILLED, SN_ROUL_SURV, SN_MAXSTEP,
       SN_OUTOFRANGE, SN_STEPS, SN_VITERS, SN_VCAPPED, SN_BADSCAT, SN_ANALOG, SN_STEPS_FREE, SN_REENTER,
       SN_BOUND_VIOL /* FLAG_BOUND records whose exact opacities exceeded the bounds they carried (must stay 0) */ };
enum { SS_EMIT = 0, SS_REC, SS_HORIZON, SS_ROUL_KILLED, SS_ROUL_GAIN, SS_OUTOFRANGE, SS_MAXSTEP,
       SS_ABSORBED, SS_WE_EMIT, SS_WE_REC, SS_BAD, SS_SPAWNED };

struct Tally { double* A; double* Q; double* W; unsigned long long* n; };

// ---- Philox4x32-10 ----------------------------------------------------------------------------
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       uint32_t k0, uint32_t k1, uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; r++) {
#ifdef __CUDA_ARCH__
    uint32_t hi0 = __umulhi(M0, c0), hi1 = __umulhi(M1, c2);
#else
    uint32_t hi0 = (uint32_t)(((uint64_t)M0 * c0) >> 32), hi1 = (uint32_t)(((uint64_t)M1 * c2) >> 32);
#endif
    uint32_t lo0 = M0 * c0, lo1 = M1 * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__host__ __device__ __forceinline__ double u53(uint32_t hi, uint32_t lo) {
  unsigned long long v = ((unsigned long long)hi << 32) | lo;
  return (double)(v >> 11) * (1.0 / 9007199254740992.0);
}
__device__ __forceinline__ void uniform_pair(const DevParams& P, uint32_t tag, uint32_t c0, uint32_t c1,
                                             uint32_t c2, uint32_t n, double& u0, double& u1) {
  uint32_t o[4];
  philox4x32_10(c0, c1, c2, n, P.seed_lo ^ tag, P.seed_hi, o);
  u0 = u53(o[0], o[1]); u1 = u53(o[2], o[3]);
}
// sequential stream of uniforms: block n of (id, tag) yields two doubles
struct RngStream {
  uint32_t c0, c1, c2, n, k0, k1; double spare; int have;
  __device__ __forceinline__ RngStream(const DevParams& P, uint32_t tag, uint32_t i0, uint32_t i1, uint32_t i2,
                                       uint32_t key1_xor = 0)
      : c0(i0), c1(i1), c2(i2), n(0), k0(P.seed_lo ^ tag), k1(P.seed_hi ^ key1_xor), spare(0.0), have(0) {}
  __device__ __forceinline__ double next() {
    if (have) { have = 0; return spare; }
    uint32_t o[4];
    philox4x32_10(c0, c1, c2, n, k0, k1, o);
    n++;
    spare = u53(o[2], o[3]); have = 1;
    return u53(o[0], o[1]);
  }
};

}  // namespace gm
