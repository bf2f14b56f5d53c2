// Internal plan structures shared by the C-ABI implementation and the kernels.
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <ctime>

#include <string>
#include <vector>

#include "../../include/psf.h"
#include "host_tables.hpp"

namespace psf {

// Everything a kernel needs, passed by value.  Notation: n = ceil(N/2), m = ceil(M/2);
// the pupil is folded about both axes into four parity classes ab (a: y parity, b: x parity; e = even, o = odd)
// and each class is pushed through the two DFT stages as two real "chains" (re, im):
//   chain index j = 2 * class + part, class order ee, eo, oe, oo.
struct DevPlan {
  int N, M, n, m, C, Z;
  int per_plane;                 // 1: per-plane Zernike rows and/or shifts -> the producer folds on the fly
  int K;                         // per-plane Zernike terms (0 if none)
  int has_shift;
  float weight[5];
  const float4 *bfold;           // [C][n][n][2]  (ee.re, ee.im, eo.re, eo.im), (oe.re, oe.im, oo.re, oo.im)
  const float2 *kt;              // [n][n]        kappa / 2 pi in turns per um, (hi, lo)
  const float2 *bunf;            // [C][N][N]     unfolded base pupil (per-plane mode)
  const float *zb;               // [K][N][N]     Zernike basis / 2 pi (turns per radian of coefficient)
  const float *coef;             // [Z][K]        per-plane coefficients
  const float *zbq;              // [K][n][n]     the same basis on the folded quadrant, terms sorted by parity class
  const float *coefq;            // [Z][K]        coefficient rows in that order
  int zcnt[4];                   // terms per parity class: even/even, odd in x, odd in y, odd/odd
  const float4 *planes;          // [Z]           (z_hi, z_lo, t_x, t_y): t = k s_max x_b / 2 pi
  const float *cosT, *sinT;      // [m][n]        cos / sin of k s_max u_q x_mi
};

struct TcState;      // tcgen05 path (kernels_tc.cu)
struct BesselState;  // spherical parametrisation (kernels_bessel.cu)
struct GradState;    // adjoint / gradients (kernels_grad.cu)
struct CztState;     // chirp-Z by FFT (kernels_czt.cu)
struct SmlmState;    // emitter-batch kernel (kernels_smlm.cu)

}  // namespace psf

struct psf_plan {
  psf_plan_desc desc;
  std::vector<double> z;
  std::string err;
  std::string kernel_names;      // psf_kernel_names
  int device = 0;
  int sm_count = 0;
  // problem
  psf::DevPlan dp{};
  int zchunk = 1;                // planes per launch pair (bounds the T scratch)
  // Zernike / shift state (host copies)
  std::vector<float> zern_shared;
  int noll_first = 4;
  std::vector<float> zern_rows;  // [Z][K]
  std::vector<int> zorder;       // parity-sorted order of the K per-plane terms (the coefq / zbq tables)
  int K_rows = 0;
  std::vector<float> shifts;     // [Z][2]
  std::vector<float> phase_mask; // [N][N] radians (psf_set_phase_mask), empty = none
  // host caches: static pupil without any Zernike term, and the Zernike basis of the last (noll_first, K)
  psf::HostPupil hp0;
  std::vector<double> zbasis;    // [K][N][N]
  std::vector<psf::cplx> h_base; // static pupil times the shared Zernike phase (kept across refreshes)
  std::vector<float4> h_bfold;
  std::vector<float2> h_kt;
  int zb_first = 0, zb_K = 0;
  long long upload_bytes = 0;
  // profiling (psf_profile_enable)
  bool prof = false, prof_valid = false;
  std::vector<cudaEvent_t> prof_ev;
  std::vector<int> prof_stage;   // stage of the launch that ends at event i+1
  int prof_n = 0;
  // device buffers (owned)
  void *d_bfold = nullptr, *d_kt = nullptr, *d_bunf = nullptr, *d_zb = nullptr, *d_coef = nullptr;
  void *d_planes = nullptr, *d_cos = nullptr, *d_sin = nullptr, *d_T = nullptr, *d_zbq = nullptr, *d_coefq = nullptr;
  size_t cap_zbq = 0, cap_coefq = 0;
  size_t T_bytes = 0;
  size_t cap_bfold = 0, cap_kt = 0, cap_bunf = 0, cap_zb = 0, cap_coef = 0, cap_planes = 0, cap_cos = 0, cap_sin = 0;
  int path = 0;                  // 0 = ffma, 1 = tc3xtf32, 2 = tc3xf16, 3 = ffma_fused (small grids), 4 = czt_fft
  psf::TcState *tc = nullptr;
  psf::BesselState *bessel = nullptr;
  psf::GradState *grad = nullptr;
  psf::CztState *czt = nullptr;
  psf::SmlmState *smlm = nullptr;
  int mat_mode = 0;              // 1: the tensor path's operand scales come from mat_qmax / mat_rmax (materialised pupils)
  double mat_qmax = 0, mat_rmax = 0;
  int tune_grad_tensor = 1;      // 1: psf_gradients on the tensor cores where the plan qualifies; 0: the FFMA route
  int tune_smlm = 1;             // 1: the emitter-batch kernel k_smlm where it qualifies; 0: always k_small
  // psf_plan_tune knobs (tests and A/B runs; defaults = the library's own choice)
  int tune_pair_mask = 3;        // ANDed with the plan's choice: bit 0 = stage 1 on CTA pairs, bit 1 = stage 2
  int tune_scratch_mb = 0;       // > 0: budget of the tensor path's T^T scratch in MB (several launch pairs per stack)
  int tune_fused_window = 0;     // 1: the fused launch carries a persisting L2 access-policy window over its ring (measured: no gain, more DRAM writes)
  int tune_fused = 1;            // 1: both stages in one launch (k12_fused) where eligible; 0: always two launches
  int tune_k1p_handoff = 0;      // k1_pair: 0 plain remote arrive, 1 .release.cluster arrive per producer warp of the non-leader CTA
  int tune_k1p_asplit = 1;       // k1_pair: 1 = the TMA-written table half of a stage buffer is released right behind its own stage
  int tune_k1p_defer = 2;        // k1_pair: K = 16 steps of the next stage issued before a stage buffer is released (profiles/r5_soak.md)
  cudaEvent_t done_ev = nullptr; // recorded on the caller's stream after the last launch of every compute call: table
                                 // refreshes wait for it before they overwrite tables a launch in flight may still read
  long long table_version = 0;   // bumped by every table refresh (psf_set_*): derived copies check it
  long long static_version = 0;  // bumped by every full (host) refresh: a device-side refresh of the shared phase leaves it alone
  long long phase_mask_version = 0;   // bumped by psf_set_phase_mask (device copies of the mask check it)
  bool host_base_stale = false;  // the last refresh ran on the device (tc_refresh_device): h_base / h_bfold are behind; see host_base()
  int tune_k1p_waitfirst = 1;    // k1_pair producers await the operand slot before computing its rows (0: after, round 2's earlier order)
  int tune_pdl = 1;              // 1: stage-2 kernels of the two-kernel tensor path are launched as programmatic dependents of stage 1
  int tune_dev_refresh = 1;      // 1: shared-phase changes of a 3xFP16 pair plan are refreshed on the device; 0: always the host path
  std::vector<double> phi;       // zoomed-DFT phase table [m][n] (fp64)
};

namespace psf {
// PSF_TIMING=1: wall-clock phases of the host table refresh on stderr (development aid)
struct PhaseTimer {
  bool on; double t0;
  static double now() { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); return ts.tv_sec * 1e3 + ts.tv_nsec * 1e-6; }
  PhaseTimer() : on(getenv("PSF_TIMING") != nullptr), t0(on ? now() : 0.0) {}
  void mark(const char *what) { if (!on) return; const double t = now(); fprintf(stderr, "[psf timing] %-28s %8.3f ms\n", what, t - t0); t0 = t; }
};
// Marks the end of one kernel launch of `stage` for the profiler (no-op unless psf_profile_enable is on).
inline void prof_mark(const psf_plan *p, cudaStream_t st, int stage) {
  psf_plan *q = const_cast<psf_plan *>(p);
  if (!q->prof || q->prof_n + 1 >= (int)q->prof_ev.size()) return;
  q->prof_stage[q->prof_n] = stage;
  cudaEventRecord(q->prof_ev[++q->prof_n], st);
}
// kernels_ffma.cu
cudaError_t launch_ffma(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field);
int ffma_launches(const psf_plan *p);
// kernels_small.cu
bool small_eligible(const psf_plan *p);
cudaError_t small_setup();       // per-device function attributes (call with the plan's device current)
cudaError_t launch_small(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field);
// kernels_tc.cu
bool tc_eligible(const psf_plan *p);
psf_status tc_setup(psf_plan *p, const std::vector<float4> &bfold, const std::vector<float2> &kt, const std::vector<double> &phi,
                    bool f16);
void tc_free(psf_plan *p);
int tc_launches(const psf_plan *p);
bool tc_fused_aborted(const psf_plan *p);
const char *tc_kernel_names(const psf_plan *p);
cudaError_t launch_tc(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field);
cudaError_t launch_tc_mat(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field, const float4 *pupils);
float tc_pupil_scale(const psf_plan *p);
int tc_n_pad(const psf_plan *p);
bool tc_pair_stage1(const psf_plan *p);
bool tc_refresh_device_ok(const psf_plan *p);
psf_status tc_refresh_device(psf_plan *p);
const float2 *tc_device_pupil(const psf_plan *p);
const std::vector<cplx> &host_base(psf_plan *p);   // h_base, recomputed first if a device-side refresh left it behind
// api.cu: turns a plan into the carrier of a materialised-pupil transform (used by the adjoint for its back-projection plan)
psf_status plan_set_materialised(psf_plan *p, double qmax, double rmax);
// kernels_bessel.cu
psf_status bessel_setup(psf_plan *p, int n_nodes);
void bessel_free(psf_plan *p);
cudaError_t launch_bessel(const psf_plan *p, cudaStream_t st, float *intensity);
// kernels_smlm.cu
psf_status smlm_setup(psf_plan *p, const std::vector<float> &zbq_sorted);
void smlm_free(psf_plan *p);
cudaError_t launch_smlm(const psf_plan *p, cudaStream_t st, float *intensity);
bool smlm_on_tensor_cores(const psf_plan *p);
// kernels_czt.cu
bool czt_supported(const psf_plan *p, std::string &why);
psf_status czt_setup(psf_plan *p);
void czt_free(psf_plan *p);
int czt_launches(const psf_plan *p);
cudaError_t launch_czt(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field);
// kernels_grad.cu
psf_status grad_setup(psf_plan *p);
bool grad_needs_setup(const psf_plan *p);
void grad_free(psf_plan *p);
int grad_terms(const psf_plan *p);
const char *grad_route(const psf_plan *p);
cudaError_t launch_grad(const psf_plan *p, cudaStream_t st, const float *dL_dI, double *dL_dz, double *dL_dc);
}  // namespace psf
