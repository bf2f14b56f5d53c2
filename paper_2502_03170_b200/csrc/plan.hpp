// Internal plan structures shared by the C-ABI implementation and the kernels.
#pragma once
#include <cuda_runtime.h>

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
  const float4 *planes;          // [Z]           (z_hi, z_lo, t_x, t_y): t = k s_max x_b / 2 pi
  const float *cosT, *sinT;      // [m][n]        cos / sin of k s_max u_q x_mi
};

struct TcState;   // tcgen05 path (kernels_tc.cu)

}  // namespace psf

struct psf_plan {
  psf_plan_desc desc;
  std::vector<double> z;
  std::string err;
  int device = 0;
  int sm_count = 0;
  // problem
  psf::DevPlan dp{};
  int zchunk = 1;                // planes per launch pair (bounds the T scratch)
  // Zernike / shift state (host copies)
  std::vector<float> zern_shared;
  int noll_first = 4;
  std::vector<float> zern_rows;  // [Z][K]
  int K_rows = 0;
  std::vector<float> shifts;     // [Z][2]
  // device buffers (owned)
  void *d_bfold = nullptr, *d_kt = nullptr, *d_bunf = nullptr, *d_zb = nullptr, *d_coef = nullptr;
  void *d_planes = nullptr, *d_cos = nullptr, *d_sin = nullptr, *d_T = nullptr;
  size_t T_bytes = 0;
  int path = 0;                  // 0 = ffma, 1 = tc3xtf32
  psf::TcState *tc = nullptr;
};

namespace psf {
// kernels_ffma.cu
cudaError_t launch_ffma(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field);
int ffma_launches(const psf_plan *p);
}  // namespace psf
