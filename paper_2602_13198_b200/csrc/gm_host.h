// Host-side declarations shared by the translation units of the library (launch wrappers).
#pragma once
#include "gm_common.cuh"

namespace gm {

// ---- gm_api.cu: text for gm_last_error(NULL), for entry points that have no context ------------------------
void note_global_error(const char* msg);

// ---- gm_tables.cu: parameter-free tables, weights, zone counts, prefix sum ----------------------
// device arrays of length NK2+1, NF+1, (NSE+1)*(NST+1)
cudaError_t build_K2_table(double* d_lnK2, cudaStream_t st);
cudaError_t build_F_table(double* d_lnF, cudaStream_t st);
cudaError_t build_sigh_table(double* d_lnSigH, cudaStream_t st);

struct ZoneArrays {
  double* A;        // [nz] emissivity prefactor A_i (0 = zone does not emit)
  double* nu0;      // [nz] (2/9) nu_c Theta_e^2
  double* vol;      // [nz] sqrt(-g) dx1 dx2 dx3 L_unit^3
  double* Nexp;     // [nz] Eq. 5
  double* qmax;     // [nz] Eq. 8 denominator
  int32_t* n;       // [nz] integer counts
  long long* offset;// [nz+1] exclusive scan
  double* partial;  // [nblk][NW+1] scratch of the weight reduction
  double* nu_nodes; // [NW+1]
  double* wk;       // [NW+1]
  long long* blocksum; // scan scratch
  int* bad;         // non-finite grid flag
};
cudaError_t launch_prepare(const DevParams& P, const ZoneArrays& Z, double* d_lnw, long nz, cudaStream_t st);

// ---- gm_transport.cu -----------------------------------------------------------------------------
struct Queue {
  Photon* buf;            // capacity records
  int* count;             // device counter (may exceed capacity: overflow)
  int capacity;
};
struct TraceBuf {          // optional per-root diagnostics (gm_trace)
  gm_trace_rec* rec;       // [n roots] or nullptr
};
cudaError_t launch_emit(const DevParams& P, const ZoneArrays& Z, long nz, long long first, int n,
                        const long long* d_ids /* or nullptr: ids = first + i */, Photon* out, int* out_count,
                        DevStats* stats, gm_emit_rec* emit_out /* or nullptr */, bool with_root,
                        cudaStream_t st);
// track every photon of `in` (count read from device) until it stops or leaves the grid outwards; scattering
// events append proto-children (parent state at the event) to `out`, leavers go to `esc` (the caller resets
// esc.count once per generation).  phase 0: everything in place; 1 (hot pass): a lane that was cold for k_cold
// committed steps is moved to `park`; 2 (cold pass): a lane that meets hot plasma is moved to `park`.
// carry_lanes > 0: a warp whose input is exhausted hands its last <= carry_lanes flying superphotons to `esc`
// marked as stragglers; launch_escape passes them on to `ret` (the next generation's input).
cudaError_t launch_track(const DevParams& P, int phase, const Photon* in, const int* in_count, int in_capacity,
                         int* work_counter, Queue out, Queue esc, Queue park, int k_cold, int carry_lanes, Tally tally,
                         DevStats* stats, TraceBuf trace, int* overflow, int n_sm, cudaStream_t st);
// opt-in for > 48 KB of dynamic shared memory of every track_kernel instance, on the CURRENT device
cudaError_t track_kernel_optin();
// records of the per-warp event stacks a PHASE_CASCADE launch needs (all warps of its grid) and records per warp
long long track_wstack_records(int n_sm);
int track_wstack_per_warp();
// free flight of the leavers to r_max (record) ; a superphoton that re-enters the grid is appended to `ret`
// `overflow`: sticky device flag word; a consumer kernel ORs 1 (tracker input) / 2 (free-flight queue) into it when
// the queue it reads was filled past its capacity
cudaError_t launch_escape(const DevParams& P, Queue esc, int* work_counter, Queue ret, Tally tally, DevStats* stats,
                          TraceBuf trace, int* overflow, int n_sm, cudaStream_t st);
// turn the proto-children of `q` into scattered superphotons in place (one Compton event each)
cudaError_t launch_compton(const DevParams& P, Queue q, DevStats* stats, TraceBuf trace, int n_sm,
                           cudaStream_t st);
cudaError_t launch_spectrum(const DevParams& P, Tally tally, double* nuLnu, double* sigma, cudaStream_t st);
cudaError_t launch_eval(const DevParams& P, int what, const double* d_in, int n, double* d_out, cudaStream_t st);
cudaError_t run_fp64_peak(double* flops_out, double* clock_mhz_out);

}  // namespace gm
