// Emitter-batch kernel (k_smlm): the per-plane mode of the fused small-grid path, restructured for the SMLM regime of
// BASELINE.json config 4 (thousands of independent single-plane PSFs, n = ceil(N/2) <= 32, m = ceil(M/2) <= 32, each emitter
// with its own defocus, tilt and Zernike row).  Same arithmetic route as k_small (kernels_small.cu: phasors -> folded pupil Q ->
// row DFT -> column DFT -> mirror butterfly -> |E|^2, all fp32 out of shared memory); what changes is where the time went
// there (profiles/r2_ncu_cfg4.md: issue-bound at 4 warps per scheduler, every emitter re-reading 130 KB of tables from L2):
//
//   * persistent CTAs, one per SM, of LANES independent 128-thread "lanes", each working through its own emitters with its
//     own named barrier: the FFMA-heavy and the latency-heavy phases of different emitters overlap on the same SM;
//   * the static tables are staged in shared memory ONCE per CTA: folded Zernike basis, kappa, the cos / sin table and the
//     base pupil - the latter not unfolded (98 KB) but split into its parity classes on the folded quadrant,
//         P_c(s_x q_x, s_y q_y) = sum_ab sigma_ab(s_x, s_y) B_c,ab(q),   sigma_ee = 1, sigma_eo = s_x, sigma_oe = s_y, sigma_oo = s_x s_y,
//     of which a pure polarisation component has ONE non-zero class (8 KB); with the parity transform of the phasor field,
//         Phi_g(q) = sum_mirrors sigma_g exp(i phi(mirror)),   the folded pupil is   Q_c,g(q) = sum_ab B_c,ab(q) Phi_(g xor ab)(q):
//     four complex multiplies per sample and class instead of four loads, four multiplies and the fold;
//   * the two FFMA loops run on the packed fp32 FMA of sm_100 (fma.rn.f32x2: the re / im chains of a class are one register
//     pair; the broadcast pairs (c, c), (s, s) of the table are built in registers - a table stored as broadcast pairs
//     doubled the shared-memory wavefronts and made the kernel slower than k_small): 16 FFMA2 + 4..5 LDS.128 + 4..8 MOV per
//     contraction index where k_small issues 32 FFMA + 4..6 loads.
// Measured (profiles/r2_ncu_cfg4.md): config 4 0.374 -> 0.285 ms; 117 M warp instructions instead of 175 M, 49 M shared-memory
// wavefronts; still issue-latency bound at three warps per scheduler (40 % issue activity).
#include <algorithm>
#include <cmath>
#include <complex>

#include <cuda_fp16.h>

#include "plan.hpp"
#include "pupil_gen.cuh"
#include "tc_common.cuh"

namespace psf {

struct SmlmState {
  int ncls = 0, lanes = 0, K = 0;
  int comp_start[6] = {0, 0, 0, 0, 0, 0};
  int cls_ab[12] = {0};
  void *d_bcls = nullptr;      // [ncls][32][32] float2, zero padded
  void *d_xd = nullptr;        // [32][MQ] float2 = (cos, sin) of k s_max u_q x_m, zero padded
  void *d_ktp = nullptr;       // [32][32] float2 kappa / 2 pi (hi, lo), zero padded
  void *d_zbp = nullptr;       // [K][32][32] float folded basis / 2 pi, terms sorted by parity class, zero padded
  int smem = 0, mq = 16;
  long long version = -1;
  // tensor-core variant (k_smlm_tc): m <= 16, precision AUTO / 3xFP16
  bool tc = false;
  void *d_bcls_tc = nullptr;   // the class tables times the operand scale s_Q
  void *d_xy = nullptr;        // 4096 bytes: the cos | sin table as the UMMA B operand (fp16 hi | lo rows, swizzled)
  int smem_tc = 0, lanes_tc = 0;
  float sQ = 1.f, fs2 = 1.f;
};

namespace {

constexpr int SL_THREADS = 128;
constexpr int SL_NQ = 32;
constexpr int SL_QROW = SL_NQ * 8 + 4;
constexpr int SL_KMAX = 12;
constexpr int SL_MAXCLS = 6;

struct SmlmArgs {
  const float2 *bcls;
  const float2 *xd;
  const float2 *ktp;
  const float *zbp;
  int ncls, K;
  int comp_start[6];
  int cls_ab[12];
};

__device__ __forceinline__ void sl_sincos_turns(float t, float &sn, float &cs) {
  t -= rintf(t);
  const float x = 6.283185307179586f * t;
  sn = __sinf(x);
  cs = __cosf(x);
}
__device__ __forceinline__ void sl_bar(int lane_id) { asm volatile("bar.sync %0, %1;" ::"r"(1 + lane_id), "r"(SL_THREADS) : "memory"); }
__device__ __forceinline__ float2 cfma(float2 a, float2 b, float2 c) {   // c + a b
  return make_float2(fmaf(a.x, b.x, fmaf(-a.y, b.y, c.x)), fmaf(a.x, b.y, fmaf(a.y, b.x, c.y)));
}

// Stages `count16` 16-byte words of a table into shared memory with the whole CTA, eight loads in flight per thread (a plain loop
// is one DRAM round trip per iteration when the tables are cold).
__device__ __forceinline__ void sl_stage16(void *dst, const void *src, int count16) {
  uint4 *d = reinterpret_cast<uint4 *>(dst);
  const uint4 *g = reinterpret_cast<const uint4 *>(src);
  for (int i0 = threadIdx.x; i0 < count16; i0 += 8 * blockDim.x) {
    uint4 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int i = i0 + u * blockDim.x;
      if (i < count16) v[u] = __ldg(g + i);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int i = i0 + u * blockDim.x;
      if (i < count16) d[i] = v[u];
    }
  }
}

template <int MQ, int LANES>
__global__ void __launch_bounds__(SL_THREADS *LANES, 1) k_smlm(const DevPlan P, const SmlmArgs A, float *__restrict__ I) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  // layout: Xd [32][MQ] float2 | kt [32][32] float2 | bcls [ncls][32][32] float2 | zb [K][32][32] float | per lane: Qs, Ts
  float2 *Xd = reinterpret_cast<float2 *>(smem_raw);
  float2 *kts = reinterpret_cast<float2 *>(Xd + SL_NQ * MQ);
  float2 *bcl = kts + SL_NQ * SL_NQ;
  float *zbs = reinterpret_cast<float *>(bcl + (size_t)A.ncls * SL_NQ * SL_NQ);
  constexpr int TS_ROW = 2 * MQ * 4 + 4;
  float *lane_base = zbs + (size_t)A.K * SL_NQ * SL_NQ;
  const int lane_id = threadIdx.x / SL_THREADS, lt = threadIdx.x % SL_THREADS;
  float *Qs = lane_base + (size_t)lane_id * (SL_NQ * SL_QROW + SL_NQ * TS_ROW + 16);
  float *Ts = Qs + SL_NQ * SL_QROW;
  float *cfs = Ts + SL_NQ * TS_ROW;             // the emitter's coefficient row (16 floats)

  // ---- stage the static tables (whole CTA) ----
  sl_stage16(Xd, A.xd, SL_NQ * MQ / 2);
  sl_stage16(kts, A.ktp, SL_NQ * SL_NQ / 2);
  sl_stage16(bcl, A.bcls, A.ncls * SL_NQ * SL_NQ / 2);
  sl_stage16(zbs, A.zbp, A.K * SL_NQ * SL_NQ / 4);
  __syncthreads();

  const int m = P.m, M = P.M, N = P.N, K = A.K;
  constexpr int PASS1 = MQ / 16, PASS2 = (MQ / 2) * (MQ / 2) / 64;

  for (int b = lane_id * gridDim.x + blockIdx.x; b < P.Z; b += gridDim.x * LANES) {   // lane-major rounds: the emitters of a partial last round go to one lane each of as many CTAs
    const float4 pl = __ldg(P.planes + b);
    if (lt < K) cfs[lt] = __ldg(P.coefq + (size_t)b * K + lt);
    {
      // the lane's next emitter: its plane entry and coefficient row into L1 now, so that the two loads above are hits then
      const int bn = b + gridDim.x * LANES;
      if (bn < P.Z) {
        if (lt == 32) asm volatile("prefetch.global.L1 [%0];" ::"l"(P.planes + bn));
        if (lt == 64) {
          asm volatile("prefetch.global.L1 [%0];" ::"l"(P.coefq + (size_t)bn * K));
          asm volatile("prefetch.global.L1 [%0];" ::"l"(P.coefq + (size_t)bn * K + (K > 0 ? K - 1 : 0)));
        }
      }
    }
    sl_bar(lane_id);

    // ---- phase 0: the parity transform Phi_g of the emitter's phasor field, 8 folded samples per thread, in registers ----
    // (term loops outermost, the thread's 8 samples inside: 8 independent FMA chains per shared-memory round trip)
    float2 phi[8][4];
    {
      float pcl[8][4];
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        pcl[r][0] = kz_turns(kts[lt + SL_THREADS * r], pl.x, pl.y);     // phase parts: even/even, x-odd, y-odd, odd/odd (turns)
        pcl[r][1] = pcl[r][2] = pcl[r][3] = 0.f;
      }
      int j = 0;
      float cnext = cfs[0];
#pragma unroll
      for (int cls = 0; cls < 4; ++cls)
        for (int e = j + P.zcnt[cls]; j < e; ++j) {
          const float cj = cnext;
          cnext = cfs[j + 1];                              // (one past the row at the end: the buffer has 16 floats)
          const float *zb = zbs + j * (SL_NQ * SL_NQ) + lt;
#pragma unroll
          for (int r = 0; r < 8; ++r) pcl[r][cls] = fmaf(cj, zb[SL_THREADS * r], pcl[r][cls]);
        }
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int f = lt + SL_THREADS * r;
        const int qy = f >> 5, qx = f & 31;
        if (P.has_shift) {
          const float ux = (float)(2 * qx + 1 - N) / (float)N, uy = (float)(2 * qy + 1 - N) / (float)N;
          pcl[r][1] = fmaf(-ux, pl.z, pcl[r][1]);
          pcl[r][2] = fmaf(-uy, pl.w, pcl[r][2]);
        }
        float2 e[4];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
          for (int bb = 0; bb < 2; ++bb) {
            const float sx = bb ? -1.f : 1.f, sy = a ? -1.f : 1.f;
            sl_sincos_turns(pcl[r][0] + sx * pcl[r][1] + sy * pcl[r][2] + sx * sy * pcl[r][3], e[a * 2 + bb].y, e[a * 2 + bb].x);
          }
        const float2 s01 = make_float2(e[0].x + e[1].x, e[0].y + e[1].y), d01 = make_float2(e[0].x - e[1].x, e[0].y - e[1].y);
        const float2 s23 = make_float2(e[2].x + e[3].x, e[2].y + e[3].y), d23 = make_float2(e[2].x - e[3].x, e[2].y - e[3].y);
        phi[r][0] = make_float2(s01.x + s23.x, s01.y + s23.y);      // sigma = 1
        phi[r][1] = make_float2(d01.x + d23.x, d01.y + d23.y);      // sigma = s_x
        phi[r][2] = make_float2(s01.x - s23.x, s01.y - s23.y);      // sigma = s_y
        phi[r][3] = make_float2(d01.x - d23.x, d01.y - d23.y);      // sigma = s_x s_y
      }
    }

    float inten[PASS2][2][4];
#pragma unroll
    for (int p = 0; p < PASS2; ++p)
#pragma unroll
      for (int ix = 0; ix < 2; ++ix)
#pragma unroll
        for (int q = 0; q < 4; ++q) inten[p][ix][q] = 0.f;

    for (int c = 0; c < P.C; ++c) {
      sl_bar(lane_id);                                   // Qs / Ts of the previous component (or emitter) are free
      // ---- Q_g = sum_ab B_ab Phi_(g xor ab) ----
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int f = lt + SL_THREADS * r;
        float2 o[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        for (int ci = A.comp_start[c]; ci < A.comp_start[c + 1]; ++ci) {
          const float2 bv = bcl[ci * (SL_NQ * SL_NQ) + f];
          switch (A.cls_ab[ci]) {                        // static register indices in every branch
            case 0: o[0] = cfma(bv, phi[r][0], o[0]); o[1] = cfma(bv, phi[r][1], o[1]); o[2] = cfma(bv, phi[r][2], o[2]); o[3] = cfma(bv, phi[r][3], o[3]); break;
            case 1: o[0] = cfma(bv, phi[r][1], o[0]); o[1] = cfma(bv, phi[r][0], o[1]); o[2] = cfma(bv, phi[r][3], o[2]); o[3] = cfma(bv, phi[r][2], o[3]); break;
            case 2: o[0] = cfma(bv, phi[r][2], o[0]); o[1] = cfma(bv, phi[r][3], o[1]); o[2] = cfma(bv, phi[r][0], o[2]); o[3] = cfma(bv, phi[r][1], o[3]); break;
            default: o[0] = cfma(bv, phi[r][3], o[0]); o[1] = cfma(bv, phi[r][2], o[1]); o[2] = cfma(bv, phi[r][1], o[2]); o[3] = cfma(bv, phi[r][0], o[3]); break;
          }
        }
        float4 *dst = reinterpret_cast<float4 *>(&Qs[(f >> 5) * SL_QROW + (f & 31) * 8]);
        const float4 v0 = make_float4(o[0].x, o[0].y, o[1].x, o[1].y);     // ee, eo
        const float4 v1 = make_float4(o[2].x, o[2].y, o[3].x, o[3].y);     // oe, oo
        const int hsw = lt & 1;                          // odd lanes store their second half first: no two-way bank conflict
        dst[hsw] = hsw ? v1 : v0;
        dst[hsw ^ 1] = hsw ? v0 : v1;
      }
      sl_bar(lane_id);

      // ---- stage 1: rows.  thread = (qy, group of 4 mx); a register pair = (re, im) of one class ----
      {
        const int qy = lt >> 2;
#pragma unroll
        for (int p = 0; p < PASS1; ++p) {
          const int mx0 = ((lt & 3) + 4 * p) * 4;
          float2 acc[4][4];                              // [class][mx]
#pragma unroll
          for (int g = 0; g < 4; ++g)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[g][i] = make_float2(0.f, 0.f);
#pragma unroll 8
          for (int k = 0; k < SL_NQ; ++k) {
            const float4 q0 = *reinterpret_cast<const float4 *>(&Qs[qy * SL_QROW + k * 8]);
            const float4 q1 = *reinterpret_cast<const float4 *>(&Qs[qy * SL_QROW + k * 8 + 4]);
            const float4 x01 = *reinterpret_cast<const float4 *>(&Xd[k * MQ + mx0]);       // (c, s) of mx0, mx0 + 1
            const float4 x23 = *reinterpret_cast<const float4 *>(&Xd[k * MQ + mx0 + 2]);
            const float cc[4] = {x01.x, x01.z, x23.x, x23.z}, ss[4] = {x01.y, x01.w, x23.y, x23.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float2 xc = make_float2(cc[i], cc[i]), xs = make_float2(ss[i], ss[i]);   // broadcast pairs built in registers
              acc[0][i] = __ffma2_rn(make_float2(q0.x, q0.y), xc, acc[0][i]);   // ee: even in x -> cos
              acc[1][i] = __ffma2_rn(make_float2(q0.z, q0.w), xs, acc[1][i]);   // eo: odd in x -> sin
              acc[2][i] = __ffma2_rn(make_float2(q1.x, q1.y), xc, acc[2][i]);   // oe
              acc[3][i] = __ffma2_rn(make_float2(q1.z, q1.w), xs, acc[3][i]);   // oo
            }
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            *reinterpret_cast<float4 *>(&Ts[qy * TS_ROW + (mx0 + i) * 4]) = make_float4(acc[0][i].x, acc[0][i].y, acc[1][i].x, acc[1][i].y);
            *reinterpret_cast<float4 *>(&Ts[qy * TS_ROW + MQ * 4 + (mx0 + i) * 4]) = make_float4(acc[2][i].x, acc[2][i].y, acc[3][i].x, acc[3][i].y);
          }
        }
      }
      sl_bar(lane_id);

      // ---- stage 2: columns.  lane pair = one 2 x 2 pixel tile, each lane sums every other q_y ----
      const float w = P.weight[c];
      const int kh = lt & 1;
#pragma unroll
      for (int p = 0; p < PASS2; ++p) {
        const int tile = (lt >> 1) + 64 * p;
        const int my0 = (tile / (MQ / 2)) * 2, mx0 = (tile % (MQ / 2)) * 2;
        float2 acc[4][2][2];                             // [class][iy][ix]
#pragma unroll
        for (int g = 0; g < 4; ++g) acc[g][0][0] = acc[g][0][1] = acc[g][1][0] = acc[g][1][1] = make_float2(0.f, 0.f);
#pragma unroll 4
        for (int kk = 0; kk < SL_NQ / 2; ++kk) {
          const int qy = 2 * kk + kh;
          const float4 y01 = *reinterpret_cast<const float4 *>(&Xd[qy * MQ + my0]);              // (c, s) of my0, my0 + 1
          const float4 t00 = *reinterpret_cast<const float4 *>(&Ts[qy * TS_ROW + mx0 * 4]);            // ee, eo at mx0
          const float4 t01 = *reinterpret_cast<const float4 *>(&Ts[qy * TS_ROW + mx0 * 4 + 4]);        // ee, eo at mx0 + 1
          const float4 t10 = *reinterpret_cast<const float4 *>(&Ts[qy * TS_ROW + MQ * 4 + mx0 * 4]);   // oe, oo
          const float4 t11 = *reinterpret_cast<const float4 *>(&Ts[qy * TS_ROW + MQ * 4 + mx0 * 4 + 4]);
          const float2 yc[2] = {make_float2(y01.x, y01.x), make_float2(y01.z, y01.z)};
          const float2 ys[2] = {make_float2(y01.y, y01.y), make_float2(y01.w, y01.w)};
#pragma unroll
          for (int iy = 0; iy < 2; ++iy) {
            acc[0][iy][0] = __ffma2_rn(make_float2(t00.x, t00.y), yc[iy], acc[0][iy][0]);   // ee, eo: even in y -> cos
            acc[0][iy][1] = __ffma2_rn(make_float2(t01.x, t01.y), yc[iy], acc[0][iy][1]);
            acc[1][iy][0] = __ffma2_rn(make_float2(t00.z, t00.w), yc[iy], acc[1][iy][0]);
            acc[1][iy][1] = __ffma2_rn(make_float2(t01.z, t01.w), yc[iy], acc[1][iy][1]);
            acc[2][iy][0] = __ffma2_rn(make_float2(t10.x, t10.y), ys[iy], acc[2][iy][0]);   // oe, oo: odd in y -> sin
            acc[2][iy][1] = __ffma2_rn(make_float2(t11.x, t11.y), ys[iy], acc[2][iy][1]);
            acc[3][iy][0] = __ffma2_rn(make_float2(t10.z, t10.w), ys[iy], acc[3][iy][0]);
            acc[3][iy][1] = __ffma2_rn(make_float2(t11.z, t11.w), ys[iy], acc[3][iy][1]);
          }
        }
        // combine the two halves of the contraction; lane kh then finishes pixel row my0 + kh
        float2 a[4][2];
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
          for (int ix = 0; ix < 2; ++ix) {
            float2 r0, r1;
            r0.x = acc[g][0][ix].x + __shfl_xor_sync(0xffffffffu, acc[g][0][ix].x, 1);
            r0.y = acc[g][0][ix].y + __shfl_xor_sync(0xffffffffu, acc[g][0][ix].y, 1);
            r1.x = acc[g][1][ix].x + __shfl_xor_sync(0xffffffffu, acc[g][1][ix].x, 1);
            r1.y = acc[g][1][ix].y + __shfl_xor_sync(0xffffffffu, acc[g][1][ix].y, 1);
            a[g][ix] = kh ? r1 : r0;
          }
#pragma unroll
        for (int ix = 0; ix < 2; ++ix) {
          const float a0 = a[0][ix].x, a1 = a[0][ix].y, a2 = a[1][ix].x, a3 = a[1][ix].y;
          const float a4 = a[2][ix].x, a5 = a[2][ix].y, a6 = a[3][ix].x, a7 = a[3][ix].y;
          // E(sy, sx) = F_ee + i sx F_eo + i sy F_oe - sx sy F_oo
          const float re0 = a0 - a3 - a5 - a6, im0 = a1 + a2 + a4 - a7;   // (+y, +x)
          const float re1 = a0 + a3 - a5 + a6, im1 = a1 - a2 + a4 + a7;   // (+y, -x)
          const float re2 = a0 - a3 + a5 + a6, im2 = a1 + a2 - a4 + a7;   // (-y, +x)
          const float re3 = a0 + a3 + a5 - a6, im3 = a1 - a2 - a4 - a7;   // (-y, -x)
          inten[p][ix][0] = fmaf(w, re0 * re0 + im0 * im0, inten[p][ix][0]);
          inten[p][ix][1] = fmaf(w, re1 * re1 + im1 * im1, inten[p][ix][1]);
          inten[p][ix][2] = fmaf(w, re2 * re2 + im2 * im2, inten[p][ix][2]);
          inten[p][ix][3] = fmaf(w, re3 * re3 + im3 * im3, inten[p][ix][3]);
        }
      }
    }

    float *Ib = I + (size_t)b * M * M;
#pragma unroll
    for (int p = 0; p < PASS2; ++p) {
      const int tile = (lt >> 1) + 64 * p;
      const int my = (tile / (MQ / 2)) * 2 + (lt & 1), mx0 = (tile % (MQ / 2)) * 2;
      if (my < m) {
        const int myr = M - 1 - my;
        // the two pixels of the thread are adjacent: 8-byte stores (M even: every pair is aligned in all four quadrants)
        if (mx0 + 1 < m) {
          *reinterpret_cast<float2 *>(Ib + (size_t)my * M + mx0) = make_float2(inten[p][0][0], inten[p][1][0]);
          *reinterpret_cast<float2 *>(Ib + (size_t)my * M + (M - 2 - mx0)) = make_float2(inten[p][1][1], inten[p][0][1]);
          *reinterpret_cast<float2 *>(Ib + (size_t)myr * M + mx0) = make_float2(inten[p][0][2], inten[p][1][2]);
          *reinterpret_cast<float2 *>(Ib + (size_t)myr * M + (M - 2 - mx0)) = make_float2(inten[p][1][3], inten[p][0][3]);
        } else if (mx0 < m) {
          Ib[(size_t)my * M + mx0] = inten[p][0][0];
          Ib[(size_t)my * M + (M - 1 - mx0)] = inten[p][0][1];
          Ib[(size_t)myr * M + mx0] = inten[p][0][2];
          Ib[(size_t)myr * M + (M - 1 - mx0)] = inten[p][0][3];
        }
      }
    }
  }
}

// ---- k_smlm_tc: the same emitter batch with both DFT stages on tcgen05 (3xFP16 split), SURVEY 8 / round-1 review item 5 option B ----
// Per emitter and component the folded pupil is the A operand of stage 1: two tiles (x-parity b) of 128 rows = (a, re/im) x 32 q_y,
// K = 32 q_x, against the shared cos (b = e) or sin (b = o) table as B (N = 16 m_x); the accumulator D1[(a, ri, q_y)][m_x] comes
// back through registers as the A operand of stage 2, rows = (class, re/im, m_x) = 128, K = 32 q_y - each warp reads its TMEM
// quarter (one chain, lane = q_y) and the 32 lanes write 32 consecutive K positions of a row, so the transposition costs
// nothing - against the same table (cos rows | sin rows, N = 32: a chain uses the half that matches its y-parity).  A row
// of every operand is 128 bytes = [hi(32 k) | lo(32 k)] fp16, SWIZZLE_128B, so x = hi + lo on both sides is three K = 32
// products picked by the K offsets of the descriptors.  A lane (128 threads = the four TMEM quarters) does everything for
// its emitter - generate, issue, drain, issue, combine - and LANES lanes interleave on the SM.
constexpr int ST_TILE = 16384;                 // [128 rows][128 B]
constexpr int ST_LANE_BYTES = 3 * ST_TILE;     // A1 (two parity tiles) + A2 (later the F exchange buffer)
constexpr int ST_XY = 4096;                    // [32 rows][128 B]: rows 0..15 cos, 16..31 sin
constexpr int ST_FCH = 16 * 16 + 16;           // floats per chain in the F buffer (padded: the re / im halves of a warp hit different banks)
constexpr float ST_XSCALE = 256.f;

struct SmlmTcArgs {
  const float2 *bcls;         // class tables, pre-scaled by s_Q
  const uint4 *xy;            // the table, fp16 hi | lo, already swizzled: 4096 bytes in stage 1's K order, 4096 in stage 2's
  const float2 *ktp;
  const float *zbp;
  int ncls, K;
  int comp_start[6];
  int cls_ab[12];
  float fs2;                  // (1 / (s_T s_X))^2: |D2|^2 -> |F|^2
};

template <int LANES>
__global__ void __launch_bounds__(SL_THREADS *LANES, 1) k_smlm_tc(const DevPlan P, const SmlmTcArgs A, float *__restrict__ I) {
  using namespace tc;
  constexpr uint32_t IDESC1 = umma_idesc_f16(128, 16), IDESC2 = umma_idesc_f16(128, 32);
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // (pointer arithmetic: the compiler keeps the shared address space)
  uint8_t *xy = smem, *xy2 = smem + ST_XY;             // the table in natural K order (stage 1) and in the drain's K order (stage 2)
  float2 *kts = reinterpret_cast<float2 *>(smem + 2 * ST_XY + LANES * ST_LANE_BYTES);
  float2 *bcl = kts + SL_NQ * SL_NQ;
  float *zbs = reinterpret_cast<float *>(bcl + (size_t)A.ncls * SL_NQ * SL_NQ);
  float *cf_all = zbs + (size_t)A.K * SL_NQ * SL_NQ;
  __shared__ uint64_t mbar1[LANES], mbar2[LANES];
  __shared__ uint32_t tmem_slot;
  // warp-uniform by construction (the broadcast tells the compiler so: addresses and descriptors derived from them stay in uniform registers)
  const int wu = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane_id = wu >> 2, warp = wu & 3, lt = threadIdx.x % SL_THREADS, l = threadIdx.x & 31;
  uint8_t *A1 = smem + 2 * ST_XY + lane_id * ST_LANE_BYTES, *A2 = A1 + 2 * ST_TILE;
  float *Fb = reinterpret_cast<float *>(A2);
  float *cfs = cf_all + lane_id * 16;

  if (threadIdx.x == 0) {
    for (int i = 0; i < LANES; ++i) { mbar_init(&mbar1[i], 2); mbar_init(&mbar2[i], 1); }
    fence_barrier_init();
  }
  if (threadIdx.x < 32) tmem_alloc(&tmem_slot, 512);
  sl_stage16(xy, A.xy, 2 * ST_XY / 16);
  sl_stage16(kts, A.ktp, SL_NQ * SL_NQ / 2);
  sl_stage16(bcl, A.bcls, A.ncls * SL_NQ * SL_NQ / 2);
  sl_stage16(zbs, A.zbp, A.K * SL_NQ * SL_NQ / 4);
  fence_proxy_async_smem();                    // the table is read by the async proxy
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem = tmem_slot + lane_id * 128;      // this lane's columns: D1(c, b) at c * 32 + b * 16, D2(c) over them
  const uint32_t tq = tmem + ((uint32_t)(warp * 32) << 16);

  const int m = P.m, M = P.M, N = P.N, K = A.K;
  // generation: a thread owns four adjacent q_x (8 bytes of a row's hi half, 8 of its lo half) at two q_y, 16 rows apart; the
  // quarter-warps of a warp sit four rows apart, so a half-warp's 8-byte stores cover all 32 banks once (rows r and r + 4 swizzle
  // into different halves of the 128-byte row)
  const int qxq = l & 7, qx0 = 4 * qxq, qyb = warp + 4 * (l >> 3);
  uint32_t ph1 = 0, ph2 = 0;
  // operand addresses of the thread's stores: the swizzle phase (q_y & 7) and the word inside the row do not change over the 4 q_y
  const uint32_t sw = (uint32_t)(qyb & 7);
  const uint32_t off_hi = ((((uint32_t)qxq >> 1) ^ sw) << 4) + (((uint32_t)qxq & 1u) << 3);     // the lo half sits at off_hi ^ 0x40
  // drain stores (fragment layout of tmem_ld_16x256b_x2): the thread holds q_y = rr, rr + 8, rr + 16, rr + 24 (rr = lane / 4) at
  // m_x = 2 (lane % 4) + {0, 1, 8, 9}; the stage-2 contraction order puts q_y = rr, rr + 8 side by side (k = 2 rr, 2 rr + 1, and
  // 16 + 2 rr, 17 + 2 rr for the upper pair), so a thread packs its own values into whole fp16 pairs: no exchange between lanes.
  // row = chain8 * 16 + m_x; word rr (+ 8) of the row's hi half; the row's swizzle phase is m_x & 7 = 2 (lane % 4) + (column & 1)
  uint32_t a2_off[2][2];
  {
    const uint32_t rrw = (uint32_t)(l >> 2);
#pragma unroll
    for (int jb = 0; jb < 2; ++jb)
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        const uint32_t mx = 2u * (uint32_t)(l & 3) + (uint32_t)jb;
        a2_off[jb][half] = smem_u32(A2) + (uint32_t)(((warp >> 1) * 4 + (warp & 1)) * 16) * 128u + mx * 128u +
                           ((((uint32_t)half * 2u + (rrw >> 2)) ^ (mx & 7u)) << 4) + ((rrw & 3u) << 2);
      }
  }
  const uint32_t a1_hi = smem_u32(A1) + (uint32_t)qyb * 128u + off_hi;

  for (int b = lane_id * gridDim.x + blockIdx.x; b < P.Z; b += gridDim.x * LANES) {   // lane-major rounds: the emitters of a partial last round go to one lane each of as many CTAs
    const float4 pl = __ldg(P.planes + b);
    sl_bar(lane_id);                                     // the previous emitter's reads of cfs are done
    if (lt < K) cfs[lt] = __ldg(P.coefq + (size_t)b * K + lt);
    {
      // the lane's next emitter: its plane entry and coefficient row into L1 now, so that the two loads above are hits then
      const int bn = b + gridDim.x * LANES;
      if (bn < P.Z) {
        if (lt == 32) asm volatile("prefetch.global.L1 [%0];" ::"l"(P.planes + bn));
        if (lt == 64) {
          asm volatile("prefetch.global.L1 [%0];" ::"l"(P.coefq + (size_t)bn * K));
          asm volatile("prefetch.global.L1 [%0];" ::"l"(P.coefq + (size_t)bn * K + (K > 0 ? K - 1 : 0)));     // (a row can straddle two sectors)
        }
      }
    }
    sl_bar(lane_id);

    // ---- phase 0: parity transform Phi_g of the emitter's phasor field at the thread's 8 folded samples ----
    // (term loops outermost, the thread's 8 samples inside: 8 independent FMA chains per shared-memory round trip)
    float2 phi[8][4];
    {
      float pcl[8][4];
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int f = (qyb + 16 * (r >> 2)) * SL_NQ + qx0 + (r & 3);
        pcl[r][0] = kz_turns(kts[f], pl.x, pl.y);
        pcl[r][1] = pcl[r][2] = pcl[r][3] = 0.f;
      }
      // software pipeline: the coefficient and the basis values of term j + 1 are loaded while term j is accumulated (the last
      // iteration re-reads its own basis row; the coefficient buffer has 16 floats for the read one past the row)
      int j = 0;
      float cnext = cfs[0];
      const float *zb0 = zbs + qyb * SL_NQ + qx0;
      float4 zn0 = make_float4(0.f, 0.f, 0.f, 0.f), zn1 = zn0;
      if (K > 0) { zn0 = *reinterpret_cast<const float4 *>(zb0); zn1 = *reinterpret_cast<const float4 *>(zb0 + 16 * SL_NQ); }   // (no basis staged without terms)
#pragma unroll
      for (int cls = 0; cls < 4; ++cls)
        for (int e = j + P.zcnt[cls]; j < e; ++j) {
          const float cj = cnext;
          const float4 z0 = zn0, z1 = zn1;
          cnext = cfs[j + 1];
          const float *zb = zb0 + (j + 1 < K ? j + 1 : j) * (SL_NQ * SL_NQ);
          zn0 = *reinterpret_cast<const float4 *>(zb);
          zn1 = *reinterpret_cast<const float4 *>(zb + 16 * SL_NQ);
          pcl[0][cls] = fmaf(cj, z0.x, pcl[0][cls]); pcl[1][cls] = fmaf(cj, z0.y, pcl[1][cls]);
          pcl[2][cls] = fmaf(cj, z0.z, pcl[2][cls]); pcl[3][cls] = fmaf(cj, z0.w, pcl[3][cls]);
          pcl[4][cls] = fmaf(cj, z1.x, pcl[4][cls]); pcl[5][cls] = fmaf(cj, z1.y, pcl[5][cls]);
          pcl[6][cls] = fmaf(cj, z1.z, pcl[6][cls]); pcl[7][cls] = fmaf(cj, z1.w, pcl[7][cls]);
        }
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const int qy = qyb + 16 * (r >> 2), qx = qx0 + (r & 3);
        if (P.has_shift) {
          const float ux = (float)(2 * qx + 1 - N) / (float)N, uy = (float)(2 * qy + 1 - N) / (float)N;
          pcl[r][1] = fmaf(-ux, pl.z, pcl[r][1]);
          pcl[r][2] = fmaf(-uy, pl.w, pcl[r][2]);
        }
        float2 e[4];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
          for (int bb = 0; bb < 2; ++bb) {
            const float sx = bb ? -1.f : 1.f, sy = a ? -1.f : 1.f;
            sl_sincos_turns(pcl[r][0] + sx * pcl[r][1] + sy * pcl[r][2] + sx * sy * pcl[r][3], e[a * 2 + bb].y, e[a * 2 + bb].x);
          }
        const float2 s01 = make_float2(e[0].x + e[1].x, e[0].y + e[1].y), d01 = make_float2(e[0].x - e[1].x, e[0].y - e[1].y);
        const float2 s23 = make_float2(e[2].x + e[3].x, e[2].y + e[3].y), d23 = make_float2(e[2].x - e[3].x, e[2].y - e[3].y);
        phi[r][0] = make_float2(s01.x + s23.x, s01.y + s23.y);
        phi[r][1] = make_float2(d01.x + d23.x, d01.y + d23.y);
        phi[r][2] = make_float2(s01.x - s23.x, s01.y - s23.y);
        phi[r][3] = make_float2(d01.x - d23.x, d01.y - d23.y);
      }
    }

    float inten[2][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int q = 0; q < 4; ++q) inten[i][q] = 0.f;

    // second half of a component: D2 -> F buffer -> butterfly + |E|^2.  Runs one component behind the first half, so that the
    // stage-2 product of component c is in flight while the operands of c + 1 are generated, and the stage-1 product of c + 1
    // while this runs.
    auto finish = [&](int cc) {
      mbar_wait(&mbar2[lane_id], ph2);
      ph2 ^= 1;
      tcgen05_fence_after();

      // ---- D2: warp = class (re rows 0..15, im rows 16..31 of the quarter), lane = (ri, m_x); its y-parity picks the column half ----
      {
        uint32_t v[16];
        tmem_ld_32x32b_x16(tq + cc * 32 + (warp >> 1) * 16, v);
        tmem_ld_wait();
        float *dst = Fb + (warp * 2 + (l >> 4)) * ST_FCH + (l & 15);
#pragma unroll
        for (int my = 0; my < 16; ++my) dst[my * 16] = __uint_as_float(v[my]);
      }
      tcgen05_fence_before();
      sl_bar(lane_id);
      // ---- butterfly + |E|^2 at the thread's two pixels of the quadrant ----
      const float w = P.weight[cc] * A.fs2;
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int px = lt + SL_THREADS * i;                // = my * 16 + mx
        const float a0 = Fb[0 * ST_FCH + px], a1 = Fb[1 * ST_FCH + px], a2 = Fb[2 * ST_FCH + px], a3 = Fb[3 * ST_FCH + px];
        const float a4 = Fb[4 * ST_FCH + px], a5 = Fb[5 * ST_FCH + px], a6 = Fb[6 * ST_FCH + px], a7 = Fb[7 * ST_FCH + px];
        const float re0 = a0 - a3 - a5 - a6, im0 = a1 + a2 + a4 - a7;
        const float re1 = a0 + a3 - a5 + a6, im1 = a1 - a2 + a4 + a7;
        const float re2 = a0 - a3 + a5 + a6, im2 = a1 + a2 - a4 + a7;
        const float re3 = a0 + a3 + a5 - a6, im3 = a1 - a2 - a4 - a7;
        inten[i][0] = fmaf(w, re0 * re0 + im0 * im0, inten[i][0]);
        inten[i][1] = fmaf(w, re1 * re1 + im1 * im1, inten[i][1]);
        inten[i][2] = fmaf(w, re2 * re2 + im2 * im2, inten[i][2]);
        inten[i][3] = fmaf(w, re3 * re3 + im3 * im3, inten[i][3]);
      }
    };

    for (int c = 0; c < P.C; ++c) {
      // ---- Q_g = sum_ab B_ab Phi_(g xor ab), scaled, split, into the two stage-1 operand tiles ----
      const int c0 = A.comp_start[c], c1 = A.comp_start[c + 1];
      if (c1 - c0 == 1) {
        // one parity class in this component (a pure polarisation component): Q_g = B Phi_(g xor x), no sum.  The product with
        // Phi_h goes to class g = h xor x: only the store address depends on x (uniform integer arithmetic, no branch)
        const int x = A.cls_ab[c0];
        uint32_t at_h[4];
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          const int g = h ^ x;
          at_h[h] = a1_hi + (uint32_t)(g & 1) * ST_TILE + (uint32_t)((g >> 1) * 2 * 32) * 128u;
        }
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
          const float4 *bp = reinterpret_cast<const float4 *>(&bcl[c0 * (SL_NQ * SL_NQ) + (qyb + 16 * rr) * SL_NQ + qx0]);
          const float4 b01 = bp[0], b23 = bp[1];
          const float2 bv[4] = {make_float2(b01.x, b01.y), make_float2(b01.z, b01.w), make_float2(b23.x, b23.y), make_float2(b23.z, b23.w)};
#pragma unroll
          for (int h = 0; h < 4; ++h) {
            float2 q[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float2 f = phi[4 * rr + e][h];
              q[e] = make_float2(fmaf(bv[e].x, f.x, -bv[e].y * f.y), fmaf(bv[e].x, f.y, bv[e].y * f.x));
            }
            const uint32_t at = at_h[h] + (uint32_t)(16 * rr) * 128u;
            uint32_t h0, l0, h1, l1;
            split_f16x2(q[0].x, q[1].x, h0, l0);
            split_f16x2(q[2].x, q[3].x, h1, l1);
            st_shared_v2_u32(at, h0, h1);
            st_shared_v2_u32(at ^ 0x40u, l0, l1);
            split_f16x2(q[0].y, q[1].y, h0, l0);
            split_f16x2(q[2].y, q[3].y, h1, l1);
            st_shared_v2_u32(at + 32 * 128, h0, h1);
            st_shared_v2_u32((at + 32 * 128) ^ 0x40u, l0, l1);
          }
        }
      } else {
#pragma unroll
      for (int rr = 0; rr < 2; ++rr) {
        float2 o[4][4];
#pragma unroll
        for (int e = 0; e < 4; ++e) o[e][0] = o[e][1] = o[e][2] = o[e][3] = make_float2(0.f, 0.f);
        for (int ci = c0; ci < c1; ++ci) {
          const float4 *bp = reinterpret_cast<const float4 *>(&bcl[ci * (SL_NQ * SL_NQ) + (qyb + 16 * rr) * SL_NQ + qx0]);
          const float4 b01 = bp[0], b23 = bp[1];
          const float2 bv[4] = {make_float2(b01.x, b01.y), make_float2(b01.z, b01.w), make_float2(b23.x, b23.y), make_float2(b23.z, b23.w)};
          // Phi index = g xor x; x is uniform: one branch per (q_y row, class), static register indices in every arm
#define SL_ACC(i0, i1, i2, i3)                                                                                     \
  _Pragma("unroll") for (int e = 0; e < 4; ++e) {                                                                  \
    const int r = 4 * rr + e;                                                                                      \
    o[e][0] = cfma(bv[e], phi[r][i0], o[e][0]); o[e][1] = cfma(bv[e], phi[r][i1], o[e][1]);                        \
    o[e][2] = cfma(bv[e], phi[r][i2], o[e][2]); o[e][3] = cfma(bv[e], phi[r][i3], o[e][3]);                        \
  }
          switch (A.cls_ab[ci]) {
            case 0: SL_ACC(0, 1, 2, 3) break;
            case 1: SL_ACC(1, 0, 3, 2) break;
            case 2: SL_ACC(2, 3, 0, 1) break;
            default: SL_ACC(3, 2, 1, 0) break;
          }
#undef SL_ACC
        }
        // class g = 2 a + xb -> tile xb, rows (2 a + ri) * 32 + qy; the four q_x are two 32-bit words of the row's hi half, two of its lo half
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          const uint32_t at = a1_hi + (uint32_t)(g & 1) * ST_TILE + (uint32_t)(((g >> 1) * 2) * 32 + 16 * rr) * 128u;
          uint32_t h0, l0, h1, l1;
          split_f16x2(o[0][g].x, o[1][g].x, h0, l0);
          split_f16x2(o[2][g].x, o[3][g].x, h1, l1);
          st_shared_v2_u32(at, h0, h1);
          st_shared_v2_u32(at ^ 0x40u, l0, l1);
          split_f16x2(o[0][g].y, o[1][g].y, h0, l0);
          split_f16x2(o[2][g].y, o[3][g].y, h1, l1);
          st_shared_v2_u32(at + 32 * 128, h0, h1);
          st_shared_v2_u32((at + 32 * 128) ^ 0x40u, l0, l1);
        }
      }
      }
      fence_proxy_async_smem();
      tcgen05_fence_before();                            // (the previous component's TMEM reads of this lane are behind us)
      sl_bar(lane_id);
      if (warp < 2 && elect_one()) {                     // one issuing thread per accumulator tile: warp 0 -> x-even, warp 1 -> x-odd
        tcgen05_fence_after();
        const int xb = warp;
        const uint32_t d = tmem + c * 32 + xb * 16;
        const uint32_t a = smem_u32(A1) + xb * ST_TILE, t = smem_u32(xy) + xb * 2048;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const uint32_t o = k * 32;
          umma_f16(d, umma_desc_sw128(a + 64 + o), umma_desc_sw128(t + o), IDESC1, k == 0 ? 0u : 1u);   // lo x hi
          umma_f16(d, umma_desc_sw128(a + o), umma_desc_sw128(t + 64 + o), IDESC1, 1u);                 // hi x lo
          umma_f16(d, umma_desc_sw128(a + o), umma_desc_sw128(t + o), IDESC1, 1u);                      // hi x hi
        }
        umma_commit(&mbar1[lane_id]);
      }
      if (c > 0) finish(c - 1);
      mbar_wait(&mbar1[lane_id], ph1);
      ph1 ^= 1;
      tcgen05_fence_after();
      if (c > 0) sl_bar(lane_id);                        // every warp is done reading the F buffer, which the drain overwrites

      // ---- drain D1: warp = chain (a, ri) of tile xb, lane = q_y; write T^T rows (class, ri, m_x), K = q_y ----
#pragma unroll
      for (int xb = 0; xb < 2; ++xb) {
        uint32_t r[8], s[8];
        tmem_ld_16x256b_x2(tq + c * 32 + xb * 16, r);
        tmem_ld_16x256b_x2(tq + (16u << 16) + c * 32 + xb * 16, s);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 4; ++j) {                                          // columns m_x = 2 (lane % 4) + {0, 1, 8, 9}
          const int i0 = (j & 1) + 4 * (j >> 1);
          const uint32_t rel = (uint32_t)xb * (2 * 16 * 128) + (uint32_t)(j >> 1) * (8 * 128);      // chain8 = ((a 2 + xb) 2 + ri)
          uint32_t hi, lo;
          split_f16x2(__uint_as_float(r[i0]), __uint_as_float(r[i0 + 2]), hi, lo);      // q_y = rr, rr + 8
          st_shared_u32(a2_off[j & 1][0] + rel, hi);
          st_shared_u32((a2_off[j & 1][0] + rel) ^ 0x40u, lo);                 // the lo half sits four 16-byte chunks on: bit 6 after the swizzle
          split_f16x2(__uint_as_float(s[i0]), __uint_as_float(s[i0 + 2]), hi, lo);      // q_y = rr + 16, rr + 24
          st_shared_u32(a2_off[j & 1][1] + rel, hi);
          st_shared_u32((a2_off[j & 1][1] + rel) ^ 0x40u, lo);
        }
      }
      fence_proxy_async_smem();
      tcgen05_fence_before();
      sl_bar(lane_id);
      if (warp == 0 && elect_one()) {
        tcgen05_fence_after();
        const uint32_t d = tmem + c * 32;
        const uint32_t a = smem_u32(A2), t = smem_u32(xy2);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const uint32_t o = k * 32;
          umma_f16(d, umma_desc_sw128(a + 64 + o), umma_desc_sw128(t + o), IDESC2, k == 0 ? 0u : 1u);
          umma_f16(d, umma_desc_sw128(a + o), umma_desc_sw128(t + 64 + o), IDESC2, 1u);
          umma_f16(d, umma_desc_sw128(a + o), umma_desc_sw128(t + o), IDESC2, 1u);
        }
        umma_commit(&mbar2[lane_id]);
      }
    }
    finish(P.C - 1);

    float *Ib = I + (size_t)b * M * M;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int px = lt + SL_THREADS * i, my = px >> 4, mx = px & 15;
      if (my < m && mx < m) {
        const int myr = M - 1 - my;
        Ib[(size_t)my * M + mx] = inten[i][0];
        Ib[(size_t)my * M + (M - 1 - mx)] = inten[i][1];
        Ib[(size_t)myr * M + mx] = inten[i][2];
        Ib[(size_t)myr * M + (M - 1 - mx)] = inten[i][3];
      }
    }
  }
  tcgen05_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) tmem_dealloc(tmem_slot, 512);
}

template <int MQ, int LANES>
cudaError_t sl_launch(const psf_plan *p, const SmlmState *t, const SmlmArgs &A, cudaStream_t st, float *intensity) {
  const int per = (p->dp.Z + LANES - 1) / LANES;
  const int grid = per < p->sm_count ? per : p->sm_count;
  k_smlm<MQ, LANES><<<grid, SL_THREADS * LANES, t->smem, st>>>(p->dp, A, intensity);
  return cudaGetLastError();
}

template <typename T>
bool sl_up(void **d, const std::vector<T> &h, long long *acc) {
  if (*d) { cudaFree(*d); *d = nullptr; }
  if (h.empty()) return true;
  if (cudaMalloc(d, h.size() * sizeof(T)) != cudaSuccess) return false;
  if (cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
  if (acc) *acc += (long long)(h.size() * sizeof(T));
  return true;
}

}  // namespace

void smlm_free(psf_plan *p) {
  SmlmState *t = p->smlm;
  if (!t) return;
  void *bufs[] = {t->d_bcls, t->d_xd, t->d_ktp, t->d_zbp, t->d_xy, t->d_bcls_tc};
  for (void *b : bufs)
    if (b) cudaFree(b);
  delete t;
  p->smlm = nullptr;
}

// Builds the emitter-batch tables if the plan qualifies: per-plane mode, even N (no self-mirror row / column), n <= 32,
// m <= 32 (M even), at most SL_KMAX per-plane Zernike terms, and few enough non-zero parity classes of the base pupil for at
// least two lanes to fit in shared memory.  Returns PSF_OK with p->smlm == nullptr when it does not (k_small runs then).
psf_status smlm_setup(psf_plan *p, const std::vector<float> &zbq_sorted) {
  smlm_free(p);
  const DevPlan &D = p->dp;
  const int N = D.N, n = D.n, m = D.m, C = D.C, K = p->K_rows;
  if (!D.per_plane || (N & 1) || (D.M & 1) || n > SL_NQ || m > 32 || K > SL_KMAX) return PSF_OK;
  const size_t NN = (size_t)N * N;
  // parity classes of the base pupil on the folded quadrant
  std::vector<float2> bcls;
  SmlmState *t = new SmlmState();
  double bmax = 0.0;
  for (size_t i = 0; i < (size_t)C * NN; ++i) bmax = std::max(bmax, std::abs(p->h_base[i]));
  int ncls = 0;
  for (int c = 0; c < C; ++c) {
    t->comp_start[c] = ncls;
    const cplx *B = p->h_base.data() + (size_t)c * NN;
    for (int ab = 0; ab < 4; ++ab) {
      std::vector<float2> cls((size_t)SL_NQ * SL_NQ, make_float2(0.f, 0.f));
      double cmax = 0.0;
      for (int qy = 0; qy < n; ++qy)
        for (int qx = 0; qx < n; ++qx) {
          const int ry = N - 1 - qy, rx = N - 1 - qx;
          const cplx p00 = B[(size_t)qy * N + qx], p01 = B[(size_t)qy * N + rx], p10 = B[(size_t)ry * N + qx], p11 = B[(size_t)ry * N + rx];
          const double sx = (ab & 1) ? -1.0 : 1.0, sy = (ab & 2) ? -1.0 : 1.0;     // sigma_ab at the mirrored index
          const cplx v = 0.25 * (p00 + sx * p01 + sy * p10 + sx * sy * p11);
          cmax = std::max(cmax, std::abs(v));
          cls[(size_t)qy * SL_NQ + qx] = make_float2((float)v.real(), (float)v.imag());
        }
      if (cmax > 1e-9 * bmax) {
        if (ncls >= 12) { delete t; return PSF_OK; }
        t->cls_ab[ncls++] = ab;
        bcls.insert(bcls.end(), cls.begin(), cls.end());
      }
    }
  }
  for (int c = C; c < 6; ++c) t->comp_start[c] = ncls;
  t->ncls = ncls;
  t->K = K;
  t->mq = m <= 16 ? 16 : 32;
  const size_t fixed = (size_t)SL_NQ * t->mq * 8 + (size_t)SL_NQ * SL_NQ * 8 + (size_t)ncls * SL_NQ * SL_NQ * 8 + (size_t)K * SL_NQ * SL_NQ * 4;
  const size_t lane = ((size_t)SL_NQ * SL_QROW + (size_t)SL_NQ * (2 * t->mq * 4 + 4) + 16) * 4;
  const size_t limit = 227 * 1024 - 256;
  t->lanes = (fixed + 3 * lane <= limit) ? 3 : (fixed + 2 * lane <= limit) ? 2 : 0;
  if (t->lanes == 0 || ncls > SL_MAXCLS * 2) { delete t; return PSF_OK; }
  t->smem = (int)(fixed + t->lanes * lane);
  // tables, zero padded to 32 (x MQ)
  const int mq = t->mq;
  std::vector<float2> xd((size_t)SL_NQ * mq, make_float2(0.f, 0.f));
  for (int mi = 0; mi < m; ++mi)
    for (int q = 0; q < n; ++q) {
      const double ph = p->phi[(size_t)mi * n + q];
      const float cs = (float)std::cos(ph), sn = (float)std::sin(ph);
      xd[(size_t)q * mq + mi] = make_float2(cs, sn);
    }
  std::vector<float2> ktp((size_t)SL_NQ * SL_NQ, make_float2(0.f, 0.f));
  for (int qy = 0; qy < n; ++qy)
    for (int qx = 0; qx < n; ++qx) ktp[(size_t)qy * SL_NQ + qx] = p->h_kt[(size_t)qy * n + qx];
  std::vector<float> zbp((size_t)K * SL_NQ * SL_NQ, 0.f);
  for (int k = 0; k < K; ++k)
    for (int qy = 0; qy < n; ++qy)
      for (int qx = 0; qx < n; ++qx) zbp[((size_t)k * SL_NQ + qy) * SL_NQ + qx] = zbq_sorted[(size_t)k * n * n + (size_t)qy * n + qx];
  auto fail = [&](const char *msg) { p->err = msg; delete t; return PSF_ERR_ALLOC; };
  p->smlm = t;
  if (!sl_up(&t->d_bcls, bcls, &p->upload_bytes) || !sl_up(&t->d_xd, xd, &p->upload_bytes) || !sl_up(&t->d_ktp, ktp, &p->upload_bytes) ||
      !sl_up(&t->d_zbp, zbp, &p->upload_bytes)) {
    p->smlm = nullptr;
    void *bufs[] = {t->d_bcls, t->d_xd, t->d_ktp, t->d_zbp};
    for (void *b : bufs)
      if (b) cudaFree(b);
    return fail("smlm: table upload failed");
  }
  cudaError_t e = cudaSuccess;
  if (mq == 16) {
    e = t->lanes == 3 ? cudaFuncSetAttribute(k_smlm<16, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem)
                      : cudaFuncSetAttribute(k_smlm<16, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem);
  } else {
    e = t->lanes == 3 ? cudaFuncSetAttribute(k_smlm<32, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem)
                      : cudaFuncSetAttribute(k_smlm<32, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem);
  }
  if (e != cudaSuccess) { p->err = std::string("smlm: cudaFuncSetAttribute: ") + cudaGetErrorString(e); smlm_free(p); return PSF_ERR_CUDA; }
  t->version = p->table_version;
  // ---- tensor-core variant: both DFT stages on tcgen05 (3xFP16), where the quadrant fits one 16-column tile ----
  const psf_precision prec = p->desc.precision;
  if (p->tune_smlm == 1 && m <= 16 && (prec == PSF_PREC_AUTO || prec == PSF_PREC_3XF16)) {
    // operand scales from phase-independent bounds: |Phi_g| <= 4, |Q_g| <= 4 sum_ab |B_ab|, |T| <= sum_qx |Q|
    double qmax = 0.0, rmax = 0.0;
    for (int c = 0; c < C; ++c)
      for (int qy = 0; qy < n; ++qy) {
        double rs = 0.0;
        for (int qx = 0; qx < n; ++qx) {
          double a = 0.0;
          for (int ci = t->comp_start[c]; ci < t->comp_start[c + 1]; ++ci) {
            const float2 v = bcls[(size_t)ci * SL_NQ * SL_NQ + (size_t)qy * SL_NQ + qx];
            a += std::sqrt((double)v.x * v.x + (double)v.y * v.y);
          }
          a *= 4.0;
          qmax = std::max(qmax, a);
          rs += a;
        }
        rmax = std::max(rmax, rs);
      }
    auto pow2 = [](double v, double limit) { return v > 0 ? std::exp2(std::floor(std::log2(limit / v))) : 1.0; };
    // s_Q so that the stage-1 accumulator s_Q s_X T is the stage-2 operand as it stands (|s_Q s_X T| <= 2^15): no rescaling in the drain
    const double sX = (double)ST_XSCALE, sQ = std::min(pow2(qmax, 16384.0), pow2(rmax, 32768.0 / sX)), sT = sQ * sX;
    t->sQ = (float)sQ;
    t->fs2 = (float)((1.0 / (sT * sX)) * (1.0 / (sT * sX)));
    // two copies: K in natural order (stage 1: K = q_x) and in the order the drain writes T^T in (stage 2: K = q_y at position
    // 16 (q / 16) + 2 (q % 8) + (q / 8) % 2, see the drain's comment in k_smlm_tc)
    std::vector<__half> xy((size_t)ST_XY, __float2half_rn(0.f));
    for (int copy = 0; copy < 2; ++copy)
      for (int row = 0; row < 32; ++row) {
        const int mi = row & 15;
        if (mi >= m) continue;
        for (int q = 0; q < n; ++q) {
          const double ph = p->phi[(size_t)mi * n + q];
          const double v = sX * ((row >> 4) ? std::sin(ph) : std::cos(ph));
          const __half hi = __float2half_rn((float)v);
          const __half lo = __float2half_rn((float)(v - (double)__half2float(hi)));
          const int k = copy ? 16 * (q / 16) + 2 * (q % 8) + (q / 8) % 2 : q;
          const int bh = 2 * k, bl = 64 + 2 * k;          // byte offsets in the 128-byte row, before the swizzle
          const int ph_hi = row * 128 + ((((bh >> 4) ^ (row & 7)) << 4) | (bh & 15));
          const int ph_lo = row * 128 + ((((bl >> 4) ^ (row & 7)) << 4) | (bl & 15));
          xy[(size_t)copy * (ST_XY / 2) + ph_hi / 2] = hi;
          xy[(size_t)copy * (ST_XY / 2) + ph_lo / 2] = lo;
        }
      }
    const size_t fixed_tc = 2 * (size_t)ST_XY + (size_t)SL_NQ * SL_NQ * 8 + (size_t)ncls * SL_NQ * SL_NQ * 8 + (size_t)K * SL_NQ * SL_NQ * 4 + 1024 + 256;
    const int lanes_tc = (fixed_tc + 3 * (size_t)ST_LANE_BYTES <= limit) ? 3 : (fixed_tc + 2 * (size_t)ST_LANE_BYTES <= limit) ? 2 : 0;
    std::vector<float2> bcls_s(bcls.size());
    for (size_t i = 0; i < bcls.size(); ++i) bcls_s[i] = make_float2((float)(sQ * bcls[i].x), (float)(sQ * bcls[i].y));   // power of two: exact
    if (lanes_tc && sl_up(&t->d_xy, xy, &p->upload_bytes) && sl_up(&t->d_bcls_tc, bcls_s, &p->upload_bytes)) {
      t->lanes_tc = lanes_tc;
      t->smem_tc = (int)(fixed_tc + lanes_tc * (size_t)ST_LANE_BYTES);
      e = lanes_tc == 3 ? cudaFuncSetAttribute(k_smlm_tc<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem_tc)
                        : cudaFuncSetAttribute(k_smlm_tc<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, t->smem_tc);
      if (e != cudaSuccess) { p->err = std::string("smlm: cudaFuncSetAttribute (tensor variant): ") + cudaGetErrorString(e); smlm_free(p); return PSF_ERR_CUDA; }
      t->tc = true;
    }
  }
  return PSF_OK;
}

bool smlm_on_tensor_cores(const psf_plan *p) { return p->smlm && p->smlm->tc; }

cudaError_t launch_smlm(const psf_plan *p, cudaStream_t st, float *intensity) {
  const SmlmState *t = p->smlm;
  if (t->tc) {
    SmlmTcArgs T;
    T.bcls = (const float2 *)t->d_bcls_tc; T.xy = (const uint4 *)t->d_xy; T.ktp = (const float2 *)t->d_ktp; T.zbp = (const float *)t->d_zbp;
    T.ncls = t->ncls; T.K = t->K;
    for (int i = 0; i < 6; ++i) T.comp_start[i] = t->comp_start[i];
    for (int i = 0; i < 12; ++i) T.cls_ab[i] = t->cls_ab[i];
    T.fs2 = t->fs2;
    const int L = t->lanes_tc, per = (p->dp.Z + L - 1) / L;
    const int grid = per < p->sm_count ? per : p->sm_count;
    if (L == 3) k_smlm_tc<3><<<grid, SL_THREADS * 3, t->smem_tc, st>>>(p->dp, T, intensity);
    else k_smlm_tc<2><<<grid, SL_THREADS * 2, t->smem_tc, st>>>(p->dp, T, intensity);
    prof_mark(p, st, 0);
    return cudaGetLastError();
  }
  SmlmArgs A;
  A.bcls = (const float2 *)t->d_bcls; A.xd = (const float2 *)t->d_xd; A.ktp = (const float2 *)t->d_ktp; A.zbp = (const float *)t->d_zbp;
  A.ncls = t->ncls; A.K = t->K;
  for (int i = 0; i < 6; ++i) A.comp_start[i] = t->comp_start[i];
  for (int i = 0; i < 12; ++i) A.cls_ab[i] = t->cls_ab[i];
  cudaError_t e;
  if (t->mq == 16) e = t->lanes == 3 ? sl_launch<16, 3>(p, t, A, st, intensity) : sl_launch<16, 2>(p, t, A, st, intensity);
  else e = t->lanes == 3 ? sl_launch<32, 3>(p, t, A, st, intensity) : sl_launch<32, 2>(p, t, A, st, intensity);
  prof_mark(p, st, 0);
  return e;
}

}  // namespace psf
