// Plain fp32 FFMA path (PSF_PREC_FP32, and the small-N choice of PSF_PREC_AUTO).
//
//   k1_stage1 : pupil producer fused with the row DFT.   T_j[qy, mx] = sum_qx Q_j[qy, qx] X_j[mx, qx]
//   k2_stage2 : column DFT + mirror butterfly + |E|^2.     F_j[my, mx] = sum_qy Y_j[my, qy] T_j[qy, mx]
//
// j runs over the 8 real chains (4 parity classes x re/im) of one scalar pupil; X_j / Y_j is the cos table for an even
// class in that axis and the sin table for an odd one.  The per-plane pupil only ever exists in shared
// memory; T is an L2-sized scratch ring owned by the plan.
#include "plan.hpp"
#include "pupil_gen.cuh"

namespace psf {

namespace {

constexpr int K1_ROWS = 16;   // qy per CTA
constexpr int K1_COLS = 64;   // mx per CTA
constexpr int K1_KC = 16;     // qx per k-chunk
constexpr int K1_THREADS = 128;

template <bool PER_PLANE>
__global__ void __launch_bounds__(K1_THREADS) k1_stage1(const DevPlan P, int z0, float *__restrict__ T) {
  __shared__ __align__(16) float Qs[K1_ROWS][K1_KC][8];
  __shared__ __align__(16) float Xc[K1_KC][K1_COLS];
  __shared__ __align__(16) float Xs[K1_KC][K1_COLS];
  const int tid = threadIdx.x;
  const int tx = tid & 7, ty = tid >> 3;            // 8 x 16 threads; thread tile = 8 chains x 8 columns
  const int mx0 = blockIdx.x * K1_COLS;
  const int qy0 = blockIdx.y * K1_ROWS;
  const int zl = blockIdx.z / P.C, c = blockIdx.z % P.C;
  const int b = z0 + zl;
  const float4 pl = __ldg(P.planes + b);
  const int n = P.n, m = P.m;

  float acc[8][8];
#pragma unroll
  for (int j = 0; j < 8; ++j)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[j][i] = 0.f;

  for (int k0 = 0; k0 < n; k0 += K1_KC) {
    // producer: 16 x 16 samples, two per thread
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int s = tid + r * K1_THREADS;
      const int ql = s >> 4, kl = s & 15;
      const int qy = qy0 + ql, qx = k0 + kl;
      float v[8];
      if (qy < n && qx < n) {
        if (PER_PLANE) gen_per_plane(P, c, b, qy, qx, pl, v);
        else gen_static(P, c, qy, qx, pl.x, pl.y, v);
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = 0.f;
      }
      *reinterpret_cast<float4 *>(&Qs[ql][kl][0]) = make_float4(v[0], v[1], v[2], v[3]);
      *reinterpret_cast<float4 *>(&Qs[ql][kl][4]) = make_float4(v[4], v[5], v[6], v[7]);
    }
    // DFT tile, transposed to [k][mx]
#pragma unroll
    for (int r = 0; r < (K1_KC * K1_COLS) / K1_THREADS; ++r) {
      const int s = tid + r * K1_THREADS;
      const int kl = s & 15, ml = s >> 4;
      const int mx = mx0 + ml, qx = k0 + kl;
      float vc = 0.f, vs = 0.f;
      if (mx < m && qx < n) { vc = __ldg(P.cosT + (size_t)mx * n + qx); vs = __ldg(P.sinT + (size_t)mx * n + qx); }
      Xc[kl][ml] = vc;
      Xs[kl][ml] = vs;
    }
    __syncthreads();
#pragma unroll
    for (int kl = 0; kl < K1_KC; ++kl) {
      const float4 q0 = *reinterpret_cast<const float4 *>(&Qs[ty][kl][0]);
      const float4 q1 = *reinterpret_cast<const float4 *>(&Qs[ty][kl][4]);
      const float4 c0 = *reinterpret_cast<const float4 *>(&Xc[kl][tx * 8]);
      const float4 c1 = *reinterpret_cast<const float4 *>(&Xc[kl][tx * 8 + 4]);
      const float4 s0 = *reinterpret_cast<const float4 *>(&Xs[kl][tx * 8]);
      const float4 s1 = *reinterpret_cast<const float4 *>(&Xs[kl][tx * 8 + 4]);
      const float xc[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
      const float xs[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
      const float q[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        acc[0][i] = fmaf(q[0], xc[i], acc[0][i]);   // ee: even in x -> cos
        acc[1][i] = fmaf(q[1], xc[i], acc[1][i]);
        acc[2][i] = fmaf(q[2], xs[i], acc[2][i]);   // eo: odd in x -> sin
        acc[3][i] = fmaf(q[3], xs[i], acc[3][i]);
        acc[4][i] = fmaf(q[4], xc[i], acc[4][i]);   // oe
        acc[5][i] = fmaf(q[5], xc[i], acc[5][i]);
        acc[6][i] = fmaf(q[6], xs[i], acc[6][i]);   // oo
        acc[7][i] = fmaf(q[7], xs[i], acc[7][i]);
      }
    }
    __syncthreads();
  }
  const int qy = qy0 + ty;
  if (qy < n) {
    float *base = T + (((size_t)zl * P.C + c) * 8) * (size_t)n * m + (size_t)qy * m + mx0 + tx * 8;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float *row = base + (size_t)j * n * m;
#pragma unroll
      for (int i = 0; i < 8; ++i)
        if (mx0 + tx * 8 + i < m) row[i] = acc[j][i];
    }
  }
}

constexpr int K2_MY = 32;     // my per CTA
constexpr int K2_MX = 64;     // mx per CTA
constexpr int K2_KC = 16;     // qy per k-chunk
constexpr int K2_THREADS = 256;

template <bool FIELD>
__global__ void __launch_bounds__(K2_THREADS) k2_stage2(const DevPlan P, int z0, const float *__restrict__ T,
                                                         float *__restrict__ I, float2 *__restrict__ field) {
  __shared__ __align__(16) float Yc[K2_KC][K2_MY];
  __shared__ __align__(16) float Ys[K2_KC][K2_MY];
  __shared__ __align__(16) float Ts[8][K2_KC][K2_MX];
  const int tid = threadIdx.x;
  const int tx = tid & 31, ty = tid >> 5;           // thread tile: my = ty*4 .. +3, mx = tx, tx + 32
  const int mx0 = blockIdx.x * K2_MX, my0 = blockIdx.y * K2_MY;
  const int zl = blockIdx.z, b = z0 + zl;
  const int n = P.n, m = P.m, M = P.M;

  float inten[4][4][2];                             // [quadrant][my][mx]
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int i = 0; i < 4; ++i) inten[q][i][0] = inten[q][i][1] = 0.f;

  for (int c = 0; c < P.C; ++c) {
    float acc[8][4][2];
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < 4; ++i) acc[j][i][0] = acc[j][i][1] = 0.f;
    const float *Tc = T + (((size_t)zl * P.C + c) * 8) * (size_t)n * m;

    for (int k0 = 0; k0 < n; k0 += K2_KC) {
      // Y tiles: [k][my]
#pragma unroll
      for (int r = 0; r < (K2_KC * K2_MY) / K2_THREADS; ++r) {
        const int s = tid + r * K2_THREADS;
        const int kl = s & 15, ml = s >> 4;
        const int my = my0 + ml, qy = k0 + kl;
        float vc = 0.f, vs = 0.f;
        if (my < m && qy < n) { vc = __ldg(P.cosT + (size_t)my * n + qy); vs = __ldg(P.sinT + (size_t)my * n + qy); }
        Yc[kl][ml] = vc;
        Ys[kl][ml] = vs;
      }
      // T tiles: 8 chains x 16 x 64
#pragma unroll
      for (int r = 0; r < (8 * K2_KC * K2_MX) / K2_THREADS; ++r) {
        const int s = tid + r * K2_THREADS;
        const int ml = s & 63, kl = (s >> 6) & 15, j = s >> 10;
        const int mx = mx0 + ml, qy = k0 + kl;
        Ts[j][kl][ml] = (mx < m && qy < n) ? __ldg(Tc + ((size_t)j * n + qy) * m + mx) : 0.f;
      }
      __syncthreads();
#pragma unroll
      for (int kl = 0; kl < K2_KC; ++kl) {
        const float4 yc4 = *reinterpret_cast<const float4 *>(&Yc[kl][ty * 4]);
        const float4 ys4 = *reinterpret_cast<const float4 *>(&Ys[kl][ty * 4]);
        const float yc[4] = {yc4.x, yc4.y, yc4.z, yc4.w};
        const float ys[4] = {ys4.x, ys4.y, ys4.z, ys4.w};
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float t0 = Ts[j][kl][tx], t1 = Ts[j][kl][tx + 32];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float y = (j < 4) ? yc[i] : ys[i];   // classes ee, eo are even in y -> cos; oe, oo odd -> sin
            acc[j][i][0] = fmaf(y, t0, acc[j][i][0]);
            acc[j][i][1] = fmaf(y, t1, acc[j][i][1]);
          }
        }
      }
      __syncthreads();
    }
    // butterfly: E(sy, sx) = F_ee + i sx F_eo + i sy F_oe - sx sy F_oo  (sx, sy = +1 at (my, mx), -1 at the mirror index)
    const float w = P.weight[c];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const float a0 = acc[0][i][u], a1 = acc[1][i][u], a2 = acc[2][i][u], a3 = acc[3][i][u];
        const float a4 = acc[4][i][u], a5 = acc[5][i][u], a6 = acc[6][i][u], a7 = acc[7][i][u];
        float re[4], im[4];
        re[0] = a0 - a3 - a5 - a6;  im[0] = a1 + a2 + a4 - a7;   // (+y, +x)
        re[1] = a0 + a3 - a5 + a6;  im[1] = a1 - a2 + a4 + a7;   // (+y, -x)  mirrored column
        re[2] = a0 - a3 + a5 + a6;  im[2] = a1 + a2 - a4 + a7;   // (-y, +x)  mirrored row
        re[3] = a0 + a3 + a5 - a6;  im[3] = a1 - a2 - a4 - a7;   // (-y, -x)
#pragma unroll
        for (int q = 0; q < 4; ++q) inten[q][i][u] = fmaf(w, re[q] * re[q] + im[q] * im[q], inten[q][i][u]);
        if (FIELD) {
          const int my = my0 + ty * 4 + i, mx = mx0 + tx + 32 * u;
          if (my < m && mx < m) {
            float2 *f = field + ((size_t)c * P.Z + b) * (size_t)M * M;
            const int myr = M - 1 - my, mxr = M - 1 - mx;
            f[(size_t)my * M + mx] = make_float2(re[0], im[0]);
            f[(size_t)my * M + mxr] = make_float2(re[1], im[1]);
            f[(size_t)myr * M + mx] = make_float2(re[2], im[2]);
            f[(size_t)myr * M + mxr] = make_float2(re[3], im[3]);
          }
        }
      }
    }
  }
  float *Ib = I + (size_t)b * M * M;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int my = my0 + ty * 4 + i, mx = mx0 + tx + 32 * u;
      if (my < m && mx < m) {
        const int myr = M - 1 - my, mxr = M - 1 - mx;
        Ib[(size_t)my * M + mx] = inten[0][i][u];
        Ib[(size_t)my * M + mxr] = inten[1][i][u];
        Ib[(size_t)myr * M + mx] = inten[2][i][u];
        Ib[(size_t)myr * M + mxr] = inten[3][i][u];
      }
    }
  }
}

}  // namespace

int ffma_launches(const psf_plan *p) { return 2 * ((p->dp.Z + p->zchunk - 1) / p->zchunk); }

cudaError_t launch_ffma(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field) {
  const DevPlan &P = p->dp;
  float *T = static_cast<float *>(p->d_T);
  for (int z0 = 0; z0 < P.Z; z0 += p->zchunk) {
    const int zc = (P.Z - z0 < p->zchunk) ? (P.Z - z0) : p->zchunk;
    dim3 g1((P.m + K1_COLS - 1) / K1_COLS, (P.n + K1_ROWS - 1) / K1_ROWS, zc * P.C);
    if (P.per_plane) k1_stage1<true><<<g1, K1_THREADS, 0, st>>>(P, z0, T);
    else k1_stage1<false><<<g1, K1_THREADS, 0, st>>>(P, z0, T);
    prof_mark(p, st, 0);
    dim3 g2((P.m + K2_MX - 1) / K2_MX, (P.m + K2_MY - 1) / K2_MY, zc);
    if (field) k2_stage2<true><<<g2, K2_THREADS, 0, st>>>(P, z0, T, intensity, field);
    else k2_stage2<false><<<g2, K2_THREADS, 0, st>>>(P, z0, T, intensity, nullptr);
    prof_mark(p, st, 1);
  }
  return cudaGetLastError();
}

}  // namespace psf
