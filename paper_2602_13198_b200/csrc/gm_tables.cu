// Device tables (S0), zone plasma state (S1), weight reduction (S2), zone counts (S3) and the
// exclusive prefix sum (S4) of SURVEY.md section 8(a).
//
//  K2 table      K_2(x) = int_0^inf exp(-x cosh t) cosh 2t dt by the trapezoid rule (geometric
//                convergence); "K2(1/Theta) ~ 2 Theta^2" above Theta = 100 is applied at lookup
//                (PAPER.md:61).
//  F table       angle integral of Eq. 3 by tanh-sinh quadrature.
//  sigma_h table Eq. 23 for Maxwell-Juttner electrons, nested
//                Gauss-Legendre quadrature, "calculated a priori and stored in a lookup table"
//                (PAPER.md:166).
//  weights       Eq. 2, counts Eq. 5-6, Eq. 8 maximum.
#include "gm_host.h"
#include "gm_physics.cuh"
#include <cmath>
#include <cstdio>
#include <mutex>
#include <vector>

namespace gm {

// ------------------------------------------------------------------------------------------------
// one warp per node: the lanes share the terms of the sum (a single thread per node left each of these two
// kernels a 224-term dependent chain on 201 / 261 threads: 0.07 + 0.24 ms of every gm_build_tables)
__global__ void k2_table_kernel(double* __restrict__ lnK2) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (i > NK2) return;
  const double l0 = log(K2_TMIN), dl = log(K2_TMAX / K2_TMIN) / NK2;
  double x = 1.0 / exp(l0 + i * dl);
  // trapezoid in t with step 1/16; the integrand falls below 1e-300 before t = 14 for x >= 0.01
  const double h = 1.0 / 16.0;
  double sum = lane == 0 ? 0.5 * exp(-x) : 0.0;
  for (int n = 1 + lane; n < 16 * 14; n += 32) {
    double t = n * h;
    double ch = cosh(t);
    double arg = x * ch;
    if (arg > 745.0) break;
    sum += exp(-arg) * cosh(2.0 * t);
  }
  sum = warp_sum(sum);
  if (lane == 0) lnK2[i] = log(sum * h);
}

__device__ __forceinline__ double F_integrand(double K, double s) {
  if (!(s > 0.0)) return 0.0;
  double X = K / s;
  double x13 = cbrt(X);
  double t = sqrt(X) + C_2_11_12 * sqrt(x13);
  return s * s * t * t * exp(-x13);
}
__global__ void f_table_kernel(double* __restrict__ lnF) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (i > NF) return;
  const double k0 = log(F_KMIN), dk = log(F_KMAX / F_KMIN) / NF;
  double K = exp(k0 + i * dk);
  // theta = (pi/4)(1 + tanh(pi/2 sinh t)); the distance to the nearer endpoint is formed
  // without cancellation so that sin(theta) stays accurate next to 0 and pi/2
  const double h = 1.0 / 32.0;
  const int N = 112;   // t in [-3.5, 3.5]
  double sum = 0.0;
  for (int n = -N + lane; n <= N; n += 32) {
    double t = n * h;
    double u = 0.5 * C_PI * sinh(t);
    double e2 = exp(-2.0 * fabs(u));
    double delta = 0.5 * C_PI * e2 / (1.0 + e2);          // (pi/4)(1 - tanh|u|)
    double wgt = 0.25 * C_PI * (0.5 * C_PI * cosh(t)) * 4.0 * e2 / ((1.0 + e2) * (1.0 + e2));
    double s = (u < 0.0) ? sin(delta) : cos(delta);        // theta = delta or pi/2 - delta
    sum += wgt * F_integrand(K, s);
  }
  sum = warp_sum(sum);
  if (lane == 0) lnF[i] = log(4.0 * C_PI * sum * h);
}

// Gauss-Legendre nodes/weights on [-1,1]
__constant__ double c_gl32_x[32], c_gl32_w[32], c_gl12_x[12], c_gl12_w[12];
static void gauss_legendre(int n, double* x, double* w) {
  for (int i = 0; i < n; i++) {
    double z = std::cos(3.14159265358979323846 * (i + 0.75) / (n + 0.5));
    double pp = 0.0;
    for (int it = 0; it < 100; it++) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 1; j <= n; j++) { double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      double z1 = z;
      z = z1 - p1 / pp;
      if (std::fabs(z - z1) < 1e-16) break;
    }
    x[i] = -z;
    w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

// mean of (1 - mu beta) sigma_KN(eps gamma (1 - mu beta)) over mu in [-1,1], for gamma = 1 + t,
// gamma beta = gb; substitution d = 1 - mu beta = exp(s), composite 12-point Gauss-Legendre in s
__device__ double mu_average(double eps, double gam, double gb) {
  double beta = gb / gam;
  if (beta < 1e-9) return sigma_kn(eps * gam);
  double slo = -log1p(gb * (gb + gam));      // ln(1 - beta)
  double shi = log1p(beta);                  // ln(1 + beta)
  if (slo < shi - 46.0) slo = shi - 46.0;    // d^2 weighting: below e^-46 of the top nothing is left
  double range = shi - slo;
  int np = (int)ceil(range);
  if (np < 1) np = 1;
  double hp = range / np;
  double eg = eps * gam;
  double sum = 0.0;
  for (int p = 0; p < np; p++) {
    double c = slo + (p + 0.5) * hp;
    double part = 0.0;
#pragma unroll 4
    for (int q = 0; q < 12; q++) {
      double d = exp(c + 0.5 * hp * c_gl12_x[q]);
      part += c_gl12_w[q] * d * d * sigma_kn(eg * d);
    }
    sum += part;
  }
  return sum * 0.5 * hp / (2.0 * beta);
}

// one block (128 threads = 4 panels x 32 Gauss-Legendre nodes in y) per table node
__global__ void __launch_bounds__(128) sigh_table_kernel(double* __restrict__ lnSigH) {
  const int node = blockIdx.x;
  const int i = node / (NST + 1), j = node % (NST + 1);
  const double LN10 = 2.302585092994046;
  const double eps = exp(LN10 * (SH_LE0 + i * ((SH_LE1 - SH_LE0) / NSE)));
  const double th = exp(LN10 * (SH_LT0 + j * ((SH_LT1 - SH_LT0) / NST)));
  const double edges[5] = {0.0, 0.25, 1.5, 4.0, 10.0};
  const int panel = threadIdx.x >> 5, q = threadIdx.x & 31;
  const double ya = edges[panel], yb = edges[panel + 1];
  const double y = 0.5 * (ya + yb) + 0.5 * (yb - ya) * c_gl32_x[q];
  const double wq = 0.5 * (yb - ya) * c_gl32_w[q];
  // gamma = 1 + Theta y^2; f_MJ dgamma ~ y^2 (1 + Theta y^2) sqrt(2 + Theta y^2) exp(-y^2) dy
  const double t = th * y * y;
  const double gy = y * y * (1.0 + t) * sqrt(2.0 + t) * exp(-y * y);
  const double gb = y * sqrt(th) * sqrt(2.0 + t);
  double den = wq * gy;
  double num = den * mu_average(eps, 1.0 + t, gb);
  __shared__ double sn[4], sd[4];
  num = warp_sum(num); den = warp_sum(den);
  if (q == 0) { sn[panel] = num; sd[panel] = den; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double N = (sn[0] + sn[1]) + (sn[2] + sn[3]), Dn = (sd[0] + sd[1]) + (sd[2] + sd[3]);
    lnSigH[node] = log(N / Dn);
  }
}

cudaError_t build_K2_table(double* d, cudaStream_t st) {
  k2_table_kernel<<<(NK2 + 4) / 4, 128, 0, st>>>(d);
  return cudaGetLastError();
}
cudaError_t build_F_table(double* d, cudaStream_t st) {
  f_table_kernel<<<(NF + 4) / 4, 128, 0, st>>>(d);
  return cudaGetLastError();
}
cudaError_t build_sigh_table(double* d, cudaStream_t st) {
  double x32[32], w32[32], x12[12], w12[12];
  gauss_legendre(32, x32, w32);
  gauss_legendre(12, x12, w12);
  cudaError_t e;
  if ((e = cudaMemcpyToSymbolAsync(c_gl32_x, x32, sizeof(x32), 0, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
  if ((e = cudaMemcpyToSymbolAsync(c_gl32_w, w32, sizeof(w32), 0, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
  if ((e = cudaMemcpyToSymbolAsync(c_gl12_x, x12, sizeof(x12), 0, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
  if ((e = cudaMemcpyToSymbolAsync(c_gl12_w, w12, sizeof(w12), 0, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;   // host arrays are on this stack frame
  sigh_table_kernel<<<(NSE + 1) * (NST + 1), 128, 0, st>>>(d);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S1: zone plasma state at the zone centre -> A_i, nu0_i, volume factor
template <bool KERR>
__global__ void zone_state_kernel(const DevParams P, ZoneArrays Z, long nz) {
  long z = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nz) return;
  int k3 = (int)(z % P.n3);
  int j2 = (int)((z / P.n3) % P.n2);
  int i1 = (int)(z / ((long)P.n3 * P.n2));
  double x1 = __dadd_rn(P.startx1, __dmul_rn(i1 + 0.5, P.dx1)), x2 = __dadd_rn(P.startx2, __dmul_rn(j2 + 0.5, P.dx2));
  (void)k3;
  Geom G;
  geom_at<KERR, false>(P, x1, x2, G, nullptr);
  double pr[8];
  load_zone(P.prim, z, pr);
  bool finite = true;
#pragma unroll
  for (int q = 0; q < 8; q++) finite = finite && isfinite(pr[q]);
  if (!finite) atomicExch(Z.bad, 1);
  double A = 0.0, nu0 = 0.0;
  if (finite && pr[0] > 0.0) {
    Plasma S;
    plasma_from_prim(P, G, pr, S);
    if (S.ne > 0.0 && S.B > 0.0 && S.thetae >= P.thetae_min) {
      nu0 = (2.0 / 9.0) * (C_NUC_B * S.B) * S.thetae * S.thetae;
      A = C_JPREF * S.ne * nu0 / K2_eval(P, S.thetae);
    }
  }
  double vol = G.gdet * P.dV;
  if (P.emit_mode == 1) {
    // exact coordinate-volume integral of sqrt(-g) = (r^2 + a^2 cos^2) sin r theta' over the zone (G31)
    const double rlo = exp(__dadd_rn(P.startx1, __dmul_rn((double)i1, P.dx1))), rhi = exp(__dadd_rn(P.startx1, __dmul_rn((double)(i1 + 1), P.dx1)));
    const double x2lo = __dadd_rn(P.startx2, __dmul_rn((double)j2, P.dx2)), x2hi = __dadd_rn(P.startx2, __dmul_rn((double)(j2 + 1), P.dx2));
    const double om = 0.5 * (1.0 - P.hslope);
    const double clo = cos(C_PI * x2lo + om * sin(2.0 * C_PI * x2lo)), chi = cos(C_PI * x2hi + om * sin(2.0 * C_PI * x2hi));
    const double a2 = P.a_spin * P.a_spin;
    vol = P.dx3 * ((rhi * rhi * rhi - rlo * rlo * rlo) / 3.0 * (clo - chi) + a2 * (rhi - rlo) * (clo * clo * clo - chi * chi * chi) / 3.0) *
          (P.L_unit * P.L_unit * P.L_unit);
  }
  Z.A[z] = A; Z.nu0[z] = nu0; Z.vol[z] = vol;
}

// S2: partial sums of sqrt(-g) d3x A_i F(nu_k/nu0_i) over a tile of 256 zones, for every node k
__global__ void __launch_bounds__(256) weight_partial_kernel(const DevParams P, ZoneArrays Z, long nz) {
  __shared__ double sm[8][NW + 1];
  long z = (long)blockIdx.x * 256 + threadIdx.x;
  double A = 0.0, nu0 = 1.0, vA = 0.0;
  if (z < nz) { A = Z.A[z]; if (A > 0.0) { nu0 = Z.nu0[z]; vA = Z.vol[z] * A; } }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int k = 0; k <= NW; k++) {
    double v = 0.0;
    if (A > 0.0) v = vA * F_of_lnK(P, log(Z.nu_nodes[k] / nu0));
    v = warp_sum(v);
    if (lane == 0) sm[warp][k] = v;
  }
  __syncthreads();
  for (int k = threadIdx.x; k <= NW; k += 256) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < 8; w++) s += sm[w][k];
    Z.partial[(long)blockIdx.x * (NW + 1) + k] = s;
  }
}
// fixed-order final reduction: block k sums partial[:, k]
__global__ void __launch_bounds__(256) weight_final_kernel(const DevParams P, ZoneArrays Z, int nblk,
                                                           double* __restrict__ lnw) {
  __shared__ double sm[256];
  const int k = blockIdx.x;
  double s = 0.0;
  for (int b = threadIdx.x; b < nblk; b += 256) s += Z.partial[(long)b * (NW + 1) + k];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    // Eq. 2 with Delta ln nu = ln(nu_max/nu_min) (G8) and the minimum-weight floor
    double w = P.T_unit * P.Lam / (C_HPL * P.Ns_target) * sm[0] + P.w_min;
    Z.wk[k] = w;
    lnw[k] = w > 0.0 ? log(w) : -700.0;
  }
}

// S3: expected count (Eq. 5, trapezoid on the weight nodes, G9), Eq. 8 maximum, integerisation (G10)
__global__ void __launch_bounds__(128) zone_count_kernel(const DevParams P, ZoneArrays Z, long nz) {
  __shared__ double s_nu[NW + 1], s_iw[NW + 1];
  for (int k = threadIdx.x; k <= NW; k += blockDim.x) {
    s_nu[k] = Z.nu_nodes[k];
    double w = Z.wk[k];
    s_iw[k] = w > 0.0 ? w : 0.0;
  }
  __syncthreads();
  long z = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nz) return;
  double A = Z.A[z];
  double Nexp = 0.0, qmax = 0.0;
  int n = 0;
  if (A > 0.0) {
    double nu0 = Z.nu0[z];
    double sum = 0.0;
    for (int k = 0; k <= NW; k++) {
      double q = s_iw[k] > 0.0 ? F_of_lnK(P, log(s_nu[k] / nu0)) / s_iw[k] : 0.0;
      double ck = (k == 0 || k == NW) ? 0.5 : 1.0;
      sum = sum + ck * q;
      if (q > qmax) qmax = q;
    }
    double C = P.T_unit * Z.vol[z] * A / C_HPL;
    Nexp = C * ((P.Lam / NW) * sum);
    double u0, u1;
    uniform_pair(P, TAG_ZONE, (uint32_t)((unsigned long long)z & 0xffffffffu),
                 (uint32_t)((unsigned long long)z >> 32), 0u, 0u, u0, u1);
    double fl = floor(Nexp);
    n = (int)fl + ((u0 < Nexp - fl) ? 1 : 0);
  }
  Z.Nexp[z] = Nexp; Z.qmax[z] = qmax; Z.n[z] = n;
}

// S4: exclusive prefix sum int32 -> int64, three phases over tiles of 1024 zones
constexpr int SCAN_TILE = 1024;
__global__ void __launch_bounds__(256) scan_tile_sum_kernel(const int32_t* __restrict__ n, long nz,
                                                            long long* __restrict__ blocksum) {
  __shared__ long long sm[8];
  long base = (long)blockIdx.x * SCAN_TILE;
  long long s = 0;
  for (int i = threadIdx.x; i < SCAN_TILE; i += 256) { long z = base + i; if (z < nz) s += n[z]; }
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { long long t = 0; for (int w = 0; w < 8; w++) t += sm[w]; blocksum[blockIdx.x] = t; }
}
__global__ void scan_blocksum_kernel(long long* __restrict__ blocksum, int nblk, long long* __restrict__ offset,
                                     long nz) {
  // one warp: serial chunks of 32 with a shuffle scan
  long long carry = 0;
  const int lane = threadIdx.x;
  for (int b0 = 0; b0 < nblk; b0 += 32) {
    int b = b0 + lane;
    long long v = b < nblk ? blocksum[b] : 0, incl = v;
    for (int o = 1; o < 32; o <<= 1) { long long t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    if (b < nblk) blocksum[b] = carry + incl - v;
    carry += __shfl_sync(0xffffffffu, incl, 31);
  }
  if (lane == 0) offset[nz] = carry;
}
__global__ void __launch_bounds__(256) scan_tile_kernel(const int32_t* __restrict__ n, long nz,
                                                        const long long* __restrict__ blocksum,
                                                        long long* __restrict__ offset) {
  __shared__ long long sm[8];
  long base = (long)blockIdx.x * SCAN_TILE + threadIdx.x * 4;
  int v[4];
  long long tsum = 0;
#pragma unroll
  for (int i = 0; i < 4; i++) { long z = base + i; v[i] = z < nz ? n[z] : 0; tsum += v[i]; }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  long long incl = tsum;
  for (int o = 1; o < 32; o <<= 1) { long long t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) sm[warp] = incl;
  __syncthreads();
  long long wbase = 0;
  for (int w = 0; w < warp; w++) wbase += sm[w];
  long long run = blocksum[blockIdx.x] + wbase + incl - tsum;
#pragma unroll
  for (int i = 0; i < 4; i++) { long z = base + i; if (z < nz) offset[z] = run; run += v[i]; }
}

// ------------------------------------------------------------------------------------------------
// Upper bounds per interpolation cell, for the tracker's cold pass (DESIGN.md section 6 "bounded steps").
// The plasma state at a point is derived from the multilinear interpolant of the primitives between the 4 (2-D)
// or 8 (3-D) zone centres around it (G4): a convex combination.  Over such a cell
//   n_e = rho Ne_unit                       <= max_c rho_c Ne_unit;
//   u/rho of the interpolant                <= max_c u_c/rho_c (mediant inequality), hence
//   Theta_e (G3)                            <= its value at that ratio, in mode 2 with the smallest R the cell allows:
//                                            R rises with beta^2 = N^2/D^2 (for R_high >= R_low), N = (gam-1) u >=
//                                            (gam-1) min_c u_c, D = b^2/2 <= g_ij B^i B^j / 2 (b^2 <= alpha^2 g_ij B^i B^j,
//                                            the normal observer's field), convex in B^i; capped by thetae_max;
//   gamma^2 = 1 + g_ij u~^i u~^j (convex in u~) <= 1 + 100 max_c q_c, q_c formed with the metric at corner c: the
//                                            factor covers the variation of g_ij over the cell and the half zones
//                                            beyond the outermost centres (sin^2 theta changes by <= 9 next to the axis);
//   eps = -k.u = gamma E_n (1 - v.n)        <= gamma (1 + v) E_n,  E_n = alpha k^t <= k^t (alpha = (1+f)^-1/2 <= 1),
//                                            gamma (1 + v) = gamma + sqrt(gamma^2 - 1), rising with gamma;
//   sigma_h / sigma_T                       <= 1.
// So nu alpha_s <= k^t S with S = (gamma_B + sqrt(gamma_B^2 - 1)) n_e,B sigma_T m_e c^2/h, and the bias b(Theta_e) <= b(Theta_B) (G21 is
// non-decreasing in Theta_e).  Theta_B carries a margin of 1e-6 against the rounding of the exact evaluation, S one of 1 %.
// A cell whose state cannot be bounded (non-finite input, u > 0 on rho = 0) gets Theta_B = inf: never skipped.
template <bool KERR>
__global__ void cell_bound_kernel(const DevParams P, double2* __restrict__ cellB, long nz) {
  long z = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nz) return;
  const int k3 = (int)(z % P.n3), j2 = (int)((z / P.n3) % P.n2), i1 = (int)(z / ((long)P.n3 * P.n2));
  double rho_max = 0.0, ratio_max = 0.0, q_max = 0.0, bb_max = 0.0, u_min = INFINITY;
  bool ok = true;
  for (int di = 0; di < 2; di++)
    for (int dj = 0; dj < 2; dj++)
      for (int dk = 0; dk < 2; dk++) {
        const int i = min(i1 + di, P.n1 - 1), j = min(j2 + dj, P.n2 - 1);
        const int k = P.n3 > 1 ? (k3 + dk) % P.n3 : 0;
        double pr[8];
        load_zone(P.prim, ((long)i * P.n2 + j) * P.n3 + k, pr);
#pragma unroll
        for (int q = 0; q < 8; q++) ok = ok && isfinite(pr[q]);
        Geom G;
        geom_at<KERR, false>(P, P.startx1 + (i + 0.5) * P.dx1, P.startx2 + (j + 0.5) * P.dx2, G, nullptr);
        const double q = G.g11 * pr[2] * pr[2] + 2.0 * fabs(G.g13 * pr[2] * pr[4]) + G.g22 * pr[3] * pr[3] + G.g33 * pr[4] * pr[4];
        q_max = fmax(q_max, q);
        bb_max = fmax(bb_max, G.g11 * pr[5] * pr[5] + 2.0 * fabs(G.g13 * pr[5] * pr[7]) + G.g22 * pr[6] * pr[6] + G.g33 * pr[7] * pr[7]);
        u_min = fmin(u_min, pr[1]);
        rho_max = fmax(rho_max, pr[0]);
        if (pr[0] > 0.0) ratio_max = fmax(ratio_max, pr[1] / pr[0]);
        else if (pr[1] > 0.0 || pr[0] < 0.0) ok = false;
      }
  double thB;
  if (P.thetae_mode == 0) thB = P.thetae_fixed;
  else if (P.thetae_mode == 1) thB = (C_MP / C_ME) * (P.gam_ad - 1.0) * ratio_max / (1.0 + P.trat);
  else {
    double Rmin = fmin(P.R_low, P.R_high);
    if (P.R_high >= P.R_low && u_min > 0.0) {
      const double N = (P.gam_ad - 1.0) * u_min, D = 0.5 * 100.0 * bb_max;
      const double N2 = N * N, D2 = D * D;
      if (isfinite(N2) && isfinite(D2) && N2 + D2 > 0.0) Rmin = (P.R_high * N2 + P.R_low * D2) / (N2 + D2) * (1.0 - 1e-6);
    }
    thB = (C_MP / C_ME) * (2.0 / 3.0) * ratio_max / (2.0 + Rmin);
  }
  thB = fmin(thB * (1.0 + 1e-6), P.thetae_max);
  const double gamB = sqrt(1.0 + 100.0 * q_max);
  // (x 1.01: the decomposition k = E_n (n + n^) assumes a null k; the integrated k.k drifts from 0 by a small multiple of
  // verlet_tol, which lets the spatial part exceed E_n by that much)
  double S = (gamB + sqrt(100.0 * q_max)) * (rho_max * P.Ne_unit) * C_SIGT * C_MEC2_H * 1.01 * P.bound_debug_scale;
  if (!ok || !isfinite(S) || !isfinite(thB)) { S = INFINITY; thB = INFINITY; }
  cellB[z] = make_double2(S, thB);
}

cudaError_t launch_prepare(const DevParams& P, const ZoneArrays& Z, double* d_lnw, long nz, cudaStream_t st) {
  int nb128 = (int)((nz + 127) / 128);
  if (P.metric_kind == 1) cell_bound_kernel<true><<<nb128, 128, 0, st>>>(P, const_cast<double2*>(P.cellB), nz);
  else cell_bound_kernel<false><<<nb128, 128, 0, st>>>(P, const_cast<double2*>(P.cellB), nz);
  if (P.metric_kind == 1) zone_state_kernel<true><<<nb128, 128, 0, st>>>(P, Z, nz);
  else zone_state_kernel<false><<<nb128, 128, 0, st>>>(P, Z, nz);
  int nblk = (int)((nz + 255) / 256);
  weight_partial_kernel<<<nblk, 256, 0, st>>>(P, Z, nz);
  weight_final_kernel<<<NW + 1, 256, 0, st>>>(P, Z, nblk, d_lnw);
  zone_count_kernel<<<nb128, 128, 0, st>>>(P, Z, nz);
  int ntile = (int)((nz + SCAN_TILE - 1) / SCAN_TILE);
  scan_tile_sum_kernel<<<ntile, 256, 0, st>>>(Z.n, nz, Z.blocksum);
  scan_blocksum_kernel<<<1, 32, 0, st>>>(Z.blocksum, ntile, Z.offset, nz);
  scan_tile_kernel<<<ntile, 256, 0, st>>>(Z.n, nz, Z.blocksum, Z.offset);
  return cudaGetLastError();
}

}  // namespace gm

// ------------------------------------------------------------------------------------------------
// gm_scan_counts_static: the S4 prefix sum for callers that must not allocate (include/gpumonty_b200.h).
//
// The three-phase scan above needs one partial sum per 1024-zone tile between its phases.  gm_prepare keeps those in
// a cudaMalloc'ed buffer of the context.  This entry point is for code that has no context and may not call
// cudaMalloc at all -- a plugin running inside a host application whose memory pool owns the whole device, a step
// replayed inside someone else's captured region, a real-time loop that must not hit the allocator's device-wide
// lock -- so its tile sums live in the file-scope array below, which is part of the library's image: every GPU that
// loads the library holds these 32 KiB from load to exit, whether or not the entry point is ever called.
//
// `g_scan_static_tiles` as written in HOST code is only the host-side handle of that symbol, not an address the GPU
// can use (a kernel handed it would fault, or on a system where the GPU can reach host memory quietly scribble over
// whatever host data sits there).  The device address is looked up with cudaGetSymbolAddress, once per device, with
// that device current, and that pointer is what the kernels get.
constexpr long GM_SCAN_STATIC_TILES = GM_SCAN_STATIC_MAX_ZONES / gm::SCAN_TILE;
static_assert(GM_SCAN_STATIC_TILES * gm::SCAN_TILE == GM_SCAN_STATIC_MAX_ZONES, "maximum must be whole tiles");
static __device__ __align__(256) long long g_scan_static_tiles[GM_SCAN_STATIC_TILES];

namespace {
constexpr int SCAN_STATIC_MAX_DEVICES = 64;
long long* s_scan_static_addr[SCAN_STATIC_MAX_DEVICES];   // device address of the array, per device ordinal (0: not looked up yet)
std::mutex s_scan_static_mutex;
}  // namespace

extern "C" int gm_scan_counts_static(const int32_t* d_counts, int64_t n_zones, int64_t* d_offsets, void* cuda_stream) {
  char msg[256];
  if (!d_counts || !d_offsets) { gm::note_global_error("gm_scan_counts_static: d_counts / d_offsets is NULL"); return GM_ERR_PARAM; }
  if (n_zones < 0 || n_zones > (int64_t)GM_SCAN_STATIC_MAX_ZONES) {
    snprintf(msg, sizeof(msg), "gm_scan_counts_static: n_zones = %lld is outside [0, %lld] (GM_SCAN_STATIC_MAX_ZONES: the built-in "
             "scratch holds one partial sum per 1024 zones and cannot grow)", (long long)n_zones, (long long)GM_SCAN_STATIC_MAX_ZONES);
    gm::note_global_error(msg);
    return GM_ERR_PARAM;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    snprintf(msg, sizeof(msg), "gm_scan_counts_static: no CUDA device (%s): this library has no CPU path", cudaGetErrorString(e));
    gm::note_global_error(msg);
    return GM_ERR_CUDA;
  }
  if (dev < 0 || dev >= SCAN_STATIC_MAX_DEVICES) {
    snprintf(msg, sizeof(msg), "gm_scan_counts_static: device ordinal %d not supported (< %d)", dev, SCAN_STATIC_MAX_DEVICES);
    gm::note_global_error(msg);
    return GM_ERR_PARAM;
  }
  long long* tiles = nullptr;
  {  // set-up, first call on this device only: ask the runtime where this device keeps its copy of the array
    std::lock_guard<std::mutex> lock(s_scan_static_mutex);
    if (!s_scan_static_addr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_scan_static_tiles);
      if (e != cudaSuccess || !p) {
        snprintf(msg, sizeof(msg), "gm_scan_counts_static: cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
        gm::note_global_error(msg);
        return GM_ERR_CUDA;
      }
      s_scan_static_addr[dev] = (long long*)p;
    }
    tiles = s_scan_static_addr[dev];
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const long nz = (long)n_zones;
  const int ntile = (int)((nz + gm::SCAN_TILE - 1) / gm::SCAN_TILE);
  long long* off = reinterpret_cast<long long*>(d_offsets);
  // Nothing in the array has to start at zero: phase 1 writes tiles[0 .. ntile), phases 2 and 3 read only those, so
  // what an earlier call (of another size) left beyond ntile is never looked at.
  if (ntile > 0) gm::scan_tile_sum_kernel<<<ntile, 256, 0, st>>>(d_counts, nz, tiles);
  gm::scan_blocksum_kernel<<<1, 32, 0, st>>>(tiles, ntile, off, nz);      // also writes d_offsets[n_zones] = total
  if (ntile > 0) gm::scan_tile_kernel<<<ntile, 256, 0, st>>>(d_counts, nz, tiles, off);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(msg, sizeof(msg), "gm_scan_counts_static: launch failed: %s", cudaGetErrorString(e));
    gm::note_global_error(msg);
    return GM_ERR_CUDA;
  }
  return GM_OK;
}
