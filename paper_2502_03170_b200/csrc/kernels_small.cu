// Fused small-grid path (n = ceil(N/2) <= 32 and m = ceil(M/2) <= 32): one CTA per plane / emitter does the whole
// hot path -- pupil producer, row DFT, column DFT, mirror butterfly, |E|^2 -- out of shared memory, in fp32 FFMA.
// This is the SMLM-batch regime of BASELINE.json config 4 (4096 emitters, N = 64, M = 32): the matrices are far too
// small for a 128 x 256 tensor tile, there is no T scratch, and HBM sees only the table reads and the intensity write.
//
//   phase 0 : per folded pupil sample, the plane's phasors exp(2 pi i t) at its four mirror images
//             (defocus kappa z, per-plane Zernike row, tilt); the Zernike basis is stored folded and sorted by
//             parity, so the four mirror phases cost K loads + K FMAs, not 4K; in per-plane mode the phasors stay in
//             the registers of the thread that made them (it is the only reader), which leaves 54 KB of shared memory
//             per CTA and four CTAs per SM.
//   per scalar pupil c:
//     Q       : base pupil x phasor at the four mirrors, folded into the 8 real chains   -> Qs[qy][qx][8]
//     stage 1 : T_j[qy, mx] = sum_qx Q_j[qy, qx] X_j[mx, qx]   (thread tile 8 chains x 4 mx)   -> Ts[qy][half][mx][4]
//     stage 2 : F_j[my, mx] = sum_qy Y_j[my, qy] T_j[qy, mx]   (thread tile 8 chains x 2 x 2 pixels; the contraction is
//               split over the two lanes of a pair and combined with one shuffle per accumulator), butterfly, |E|^2.
#include "plan.hpp"
#include "pupil_gen.cuh"

namespace psf {

namespace {

constexpr int SM_THREADS = 128;
constexpr int NQ = 32;                 // folded pupil samples per axis held by a CTA
constexpr int QS_ROW = NQ * 8 + 4;     // floats per q_y row of Qs (+4 shifts consecutive rows by one 16-byte bank group)

template <int MQ, bool PER_PLANE>
struct SmallSmem {
  float Qs[NQ][QS_ROW];                // [qy][qx][8 chains]
  float Ts[NQ][2 * MQ * 4 + 4];        // [qy][chains 0-3 | 4-7][mx][4]
  float2 Ph0[PER_PLANE ? 2 : NQ * NQ]; // static mode: one phasor per sample, kept here (small code: tiny stacks start cold)
  float Xc[NQ][MQ], Xs[NQ][MQ];        // cos / sin of k s_max u_q x_m, [q][m]; serves both stages (square grids)
};

__device__ __forceinline__ void sincos_turns(float t, float &sn, float &cs) {
  t -= rintf(t);
  const float x = 6.283185307179586f * t;
  sn = __sinf(x);                      // SFU, |error| ~ 2^-21 on the reduced argument
  cs = __cosf(x);
}

// STRIPS > 1 (static mode, short stacks): a plane is split over STRIPS CTAs by m_x strip; each regenerates the folded pupil
// (cheap) and does its share of both products, so that a 16-plane stack occupies 64 SMs instead of 16.
template <int MQ, bool PER_PLANE, bool FIELD, int STRIPS>
__global__ void __launch_bounds__(SM_THREADS, PER_PLANE ? 4 : 1) k_small(const DevPlan P, float *__restrict__ I, float2 *__restrict__ field) {
  constexpr int MXS = MQ / STRIPS;               // m_x columns of this CTA
  const int mx_base = blockIdx.y * MXS;
  extern __shared__ __align__(16) uint8_t smem_raw[];
  SmallSmem<MQ, PER_PLANE> &S = *reinterpret_cast<SmallSmem<MQ, PER_PLANE> *>(smem_raw);
  const int tid = threadIdx.x;
  const int b = blockIdx.x;
  const int n = P.n, m = P.m, N = P.N, M = P.M;

  // A short stack is nothing but the latencies of its first touches: after other work has gone through the L2 (bench.py flushes
  // it between steps) every table is a DRAM access, and the tables are read in phases that depend on one another (tables ->
  // phasors -> per component the base pupil).  In static mode the thread therefore issues, now, every global load of its
  // prologue - plane, kappa, the base pupil of component 0 - ahead of the table staging (whose loop is fully unrolled as
  // well), and the base pupil of component c + 1 is loaded into registers before the two DFT stages of component c: one
  // overlapped round trip at the start instead of one per phase and per component.
  constexpr int NSAMP = (NQ * NQ) / SM_THREADS;
  float4 bq[PER_PLANE ? 1 : 2 * NSAMP];
  float2 ktv[PER_PLANE ? 1 : NSAMP];
  auto load_bq = [&](int c) {
#pragma unroll
    for (int r = 0; r < NSAMP; ++r) {
      const int f = tid + SM_THREADS * r;
      const int qy = f >> 5, qx = f & 31;
      const bool ok = qy < n && qx < n;
      const size_t s = ok ? ((size_t)c * n * n + (size_t)qy * n + qx) * 2 : 0;
      bq[PER_PLANE ? 0 : 2 * r] = ok ? __ldg(P.bfold + s) : make_float4(0.f, 0.f, 0.f, 0.f);
      bq[PER_PLANE ? 0 : 2 * r + 1] = ok ? __ldg(P.bfold + s + 1) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
  };
  const float4 pl = __ldg(P.planes + b);
  if (!PER_PLANE) {
#pragma unroll
    for (int r = 0; r < NSAMP; ++r) {
      const int f = tid + SM_THREADS * r;
      const int qy = f >> 5, qx = f & 31;
      ktv[PER_PLANE ? 0 : r] = (qy < n && qx < n) ? __ldg(P.kt + (size_t)qy * n + qx) : make_float2(0.f, 0.f);
    }
    load_bq(0);
  }
#pragma unroll
  for (int i = tid; i < NQ * MQ; i += SM_THREADS) {
    const int q = i / MQ, mi = i % MQ;
    const bool ok = q < n && mi < m;
    S.Xc[q][mi] = ok ? __ldg(P.cosT + (size_t)mi * n + q) : 0.f;
    S.Xs[q][mi] = ok ? __ldg(P.sinT + (size_t)mi * n + q) : 0.f;
  }

  // ---- phase 0: phasors -------------------------------------------------------------------------------------------
  // phasors (cos, sin) of this thread's 8 samples at their (up to) four mirror images, kept in registers: a thread reads
  // back only the phasors it wrote, and without the 32 KB they took in shared memory more CTAs fit an SM
  float2 phr[PER_PLANE ? (NQ * NQ) / SM_THREADS : 1][PER_PLANE ? 4 : 1];
#pragma unroll 8
  for (int r = 0; r < (NQ * NQ) / SM_THREADS; ++r) {
    const int f = tid + SM_THREADS * r;
    const int qy = f >> 5, qx = f & 31;
    float2 ph[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
    if (qy < n && qx < n) {
      const size_t s = (size_t)qy * n + qx;
      const float t0 = kz_turns(PER_PLANE ? __ldg(P.kt + s) : ktv[PER_PLANE ? 0 : r], pl.x, pl.y);
      if (PER_PLANE) {
        // parity classes of the phase: even/even, x-odd, y-odd, odd/odd
        float pee = t0, pxo = 0.f, pyo = 0.f, poo = 0.f;
        const float *cf = P.coefq + (size_t)b * P.K;
        const float *zq = P.zbq + s;
        const size_t nn = (size_t)n * n;
        int j = 0;
        for (int e = P.zcnt[0]; j < e; ++j) pee = fmaf(__ldg(cf + j), __ldg(zq + j * nn), pee);
        for (int e = j + P.zcnt[1]; j < e; ++j) pxo = fmaf(__ldg(cf + j), __ldg(zq + j * nn), pxo);
        for (int e = j + P.zcnt[2]; j < e; ++j) pyo = fmaf(__ldg(cf + j), __ldg(zq + j * nn), pyo);
        for (int e = j + P.zcnt[3]; j < e; ++j) poo = fmaf(__ldg(cf + j), __ldg(zq + j * nn), poo);
        if (P.has_shift) {
          const float ux = (float)(2 * qx + 1 - N) / (float)N, uy = (float)(2 * qy + 1 - N) / (float)N;
          pxo = fmaf(-ux, pl.z, pxo);      // tilt -(u_x t_x + u_y t_y): odd in x, odd in y respectively
          pyo = fmaf(-uy, pl.w, pyo);
        }
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
          for (int bb = 0; bb < 2; ++bb) {
            const float sx = bb ? -1.f : 1.f, sy = a ? -1.f : 1.f;
            const float t = pee + sx * pxo + sy * pyo + sx * sy * poo;
            sincos_turns(t, ph[a * 2 + bb].y, ph[a * 2 + bb].x);
          }
      } else {
        sincos_turns(t0, ph[0].y, ph[0].x);
      }
    }
    if (PER_PLANE) {
      phr[PER_PLANE ? r : 0][0] = ph[0];
      phr[PER_PLANE ? r : 0][1 % (PER_PLANE ? 4 : 1)] = ph[1]; phr[PER_PLANE ? r : 0][2 % (PER_PLANE ? 4 : 1)] = ph[2]; phr[PER_PLANE ? r : 0][3 % (PER_PLANE ? 4 : 1)] = ph[3];
    } else {
      S.Ph0[PER_PLANE ? 0 : f] = ph[0];
    }
  }

  constexpr int PASS1 = MXS >= 16 ? MXS / 16 : 1;  // stage-1 passes over m_x groups of 4 (4 groups per pass)
  constexpr int G1 = MXS >= 16 ? 4 : MXS / 4;      // m_x groups per pass (a strip of 8 columns keeps half of the threads busy here)
  constexpr int PASS2 = (MQ / 2) * (MXS / 2) / 64; // stage-2 passes over 2 x 2 pixel tiles (64 tiles per pass)
  float inten[PASS2][2][4];
#pragma unroll
  for (int p = 0; p < PASS2; ++p)
#pragma unroll
    for (int ix = 0; ix < 2; ++ix)
#pragma unroll
      for (int q = 0; q < 4; ++q) inten[p][ix][q] = 0.f;

  for (int c = 0; c < P.C; ++c) {
    __syncthreads();                             // Qs / Ts of the previous component are free (and the tables are in)
    // ---- Q: base pupil x phasor, folded (a thread reads back only the phasors it wrote) ----
#pragma unroll 8
    for (int r = 0; r < (NQ * NQ) / SM_THREADS; ++r) {
      const int f = tid + SM_THREADS * r;
      const int qy = f >> 5, qx = f & 31;
      float o[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (qy < n && qx < n) {
        if (PER_PLANE) {
          const int ry = N - 1 - qy, rx = N - 1 - qx;
          const float2 *B = P.bunf + (size_t)c * N * N;
          float2 v[2][2];
#pragma unroll
          for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int bb = 0; bb < 2; ++bb) {
              const float2 bu = __ldg(B + (size_t)(a ? ry : qy) * N + (bb ? rx : qx));
              const float2 e = phr[PER_PLANE ? r : 0][(a * 2 + bb) % (PER_PLANE ? 4 : 1)];
              v[a][bb] = make_float2(bu.x * e.x - bu.y * e.y, bu.x * e.y + bu.y * e.x);
            }
          if (rx == qx) { v[0][1] = make_float2(0.f, 0.f); v[1][1] = make_float2(0.f, 0.f); }   // odd N: self-mirror column
          if (ry == qy) { v[1][0] = make_float2(0.f, 0.f); v[1][1] = make_float2(0.f, 0.f); }   // self-mirror row
          const float2 e0 = make_float2(v[0][0].x + v[0][1].x, v[0][0].y + v[0][1].y);   // even in x, row qy
          const float2 o0 = make_float2(v[0][0].x - v[0][1].x, v[0][0].y - v[0][1].y);   // odd in x
          const float2 e1 = make_float2(v[1][0].x + v[1][1].x, v[1][0].y + v[1][1].y);   // mirror row
          const float2 o1 = make_float2(v[1][0].x - v[1][1].x, v[1][0].y - v[1][1].y);
          const bool selfx = rx == qx, selfy = ry == qy;
          o[0] = e0.x + e1.x;  o[1] = e0.y + e1.y;                                       // ee
          o[2] = selfx ? 0.f : o0.x + o1.x;  o[3] = selfx ? 0.f : o0.y + o1.y;           // eo
          o[4] = selfy ? 0.f : e0.x - e1.x;  o[5] = selfy ? 0.f : e0.y - e1.y;           // oe
          o[6] = (selfx || selfy) ? 0.f : o0.x - o1.x;  o[7] = (selfx || selfy) ? 0.f : o0.y - o1.y;   // oo
        } else {
          const float4 b0 = bq[PER_PLANE ? 0 : 2 * r], b1 = bq[PER_PLANE ? 0 : 2 * r + 1];
          const float2 e = S.Ph0[PER_PLANE ? 0 : f];
          o[0] = b0.x * e.x - b0.y * e.y;  o[1] = b0.x * e.y + b0.y * e.x;
          o[2] = b0.z * e.x - b0.w * e.y;  o[3] = b0.z * e.y + b0.w * e.x;
          o[4] = b1.x * e.x - b1.y * e.y;  o[5] = b1.x * e.y + b1.y * e.x;
          o[6] = b1.z * e.x - b1.w * e.y;  o[7] = b1.z * e.y + b1.w * e.x;
        }
      }
      float4 *dst = reinterpret_cast<float4 *>(&S.Qs[qy][qx * 8]);
      dst[0] = make_float4(o[0], o[1], o[2], o[3]);
      dst[1] = make_float4(o[4], o[5], o[6], o[7]);
    }
    if (!PER_PLANE && c + 1 < P.C) load_bq(c + 1);     // in flight under the two DFT stages of this component
    __syncthreads();

    // ---- stage 1: rows.  thread = (qy, group of 4 mx) ----
    {
      const int qy = tid >> 2;
#pragma unroll
      for (int p = 0; p < PASS1; ++p) {
        if ((tid & 3) >= G1) break;
        const int lx0 = ((tid & 3) + 4 * p) * 4;     // column inside the strip
        const int mx0 = mx_base + lx0;
        float acc[8][4];
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
          for (int i = 0; i < 4; ++i) acc[j][i] = 0.f;
#pragma unroll 8
        for (int k = 0; k < NQ; ++k) {
          const float4 q0 = *reinterpret_cast<const float4 *>(&S.Qs[qy][k * 8]);
          const float4 q1 = *reinterpret_cast<const float4 *>(&S.Qs[qy][k * 8 + 4]);
          const float4 c4 = *reinterpret_cast<const float4 *>(&S.Xc[k][mx0]);
          const float4 s4 = *reinterpret_cast<const float4 *>(&S.Xs[k][mx0]);
          const float xc[4] = {c4.x, c4.y, c4.z, c4.w}, xs[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            acc[0][i] = fmaf(q0.x, xc[i], acc[0][i]);   // ee: even in x -> cos
            acc[1][i] = fmaf(q0.y, xc[i], acc[1][i]);
            acc[2][i] = fmaf(q0.z, xs[i], acc[2][i]);   // eo: odd in x -> sin
            acc[3][i] = fmaf(q0.w, xs[i], acc[3][i]);
            acc[4][i] = fmaf(q1.x, xc[i], acc[4][i]);   // oe
            acc[5][i] = fmaf(q1.y, xc[i], acc[5][i]);
            acc[6][i] = fmaf(q1.z, xs[i], acc[6][i]);   // oo
            acc[7][i] = fmaf(q1.w, xs[i], acc[7][i]);
          }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          *reinterpret_cast<float4 *>(&S.Ts[qy][(lx0 + i) * 4]) = make_float4(acc[0][i], acc[1][i], acc[2][i], acc[3][i]);
          *reinterpret_cast<float4 *>(&S.Ts[qy][MXS * 4 + (lx0 + i) * 4]) = make_float4(acc[4][i], acc[5][i], acc[6][i], acc[7][i]);
        }
      }
    }
    __syncthreads();

    // ---- stage 2: columns.  lane pair = one 2 x 2 pixel tile, each lane sums every other q_y ----
    const float w = P.weight[c];
    const int kh = tid & 1;
#pragma unroll
    for (int p = 0; p < PASS2; ++p) {
      const int tile = (tid >> 1) + 64 * p;
      const int my0 = (tile / (MXS / 2)) * 2, lx0 = (tile % (MXS / 2)) * 2, mx0 = mx_base + lx0;
      float acc[8][2][2];
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[j][0][0] = acc[j][0][1] = acc[j][1][0] = acc[j][1][1] = 0.f;
#pragma unroll 4
      for (int kk = 0; kk < NQ / 2; ++kk) {
        const int qy = 2 * kk + kh;
        const float2 yc = *reinterpret_cast<const float2 *>(&S.Xc[qy][my0]);
        const float2 ys = *reinterpret_cast<const float2 *>(&S.Xs[qy][my0]);
        const float4 t00 = *reinterpret_cast<const float4 *>(&S.Ts[qy][lx0 * 4]);            // chains 0-3, mx0
        const float4 t01 = *reinterpret_cast<const float4 *>(&S.Ts[qy][lx0 * 4 + 4]);        // chains 0-3, mx0 + 1
        const float4 t10 = *reinterpret_cast<const float4 *>(&S.Ts[qy][MXS * 4 + lx0 * 4]);   // chains 4-7
        const float4 t11 = *reinterpret_cast<const float4 *>(&S.Ts[qy][MXS * 4 + lx0 * 4 + 4]);
        const float lo0[4] = {t00.x, t00.y, t00.z, t00.w}, lo1[4] = {t01.x, t01.y, t01.z, t01.w};
        const float hi0[4] = {t10.x, t10.y, t10.z, t10.w}, hi1[4] = {t11.x, t11.y, t11.z, t11.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc[j][0][0] = fmaf(yc.x, lo0[j], acc[j][0][0]);   // classes ee, eo: even in y -> cos
          acc[j][0][1] = fmaf(yc.x, lo1[j], acc[j][0][1]);
          acc[j][1][0] = fmaf(yc.y, lo0[j], acc[j][1][0]);
          acc[j][1][1] = fmaf(yc.y, lo1[j], acc[j][1][1]);
          acc[4 + j][0][0] = fmaf(ys.x, hi0[j], acc[4 + j][0][0]);   // oe, oo: odd in y -> sin
          acc[4 + j][0][1] = fmaf(ys.x, hi1[j], acc[4 + j][0][1]);
          acc[4 + j][1][0] = fmaf(ys.y, hi0[j], acc[4 + j][1][0]);
          acc[4 + j][1][1] = fmaf(ys.y, hi1[j], acc[4 + j][1][1]);
        }
      }
      // combine the two halves of the contraction; lane kh then finishes pixel row my0 + kh
      float a[8][2];
#pragma unroll
      for (int j = 0; j < 8; ++j)
#pragma unroll
        for (int ix = 0; ix < 2; ++ix) {
          const float r0 = acc[j][0][ix] + __shfl_xor_sync(0xffffffffu, acc[j][0][ix], 1);
          const float r1 = acc[j][1][ix] + __shfl_xor_sync(0xffffffffu, acc[j][1][ix], 1);
          a[j][ix] = kh ? r1 : r0;
        }
      const int my = my0 + kh;
#pragma unroll
      for (int ix = 0; ix < 2; ++ix) {
        const float a0 = a[0][ix], a1 = a[1][ix], a2 = a[2][ix], a3 = a[3][ix];
        const float a4 = a[4][ix], a5 = a[5][ix], a6 = a[6][ix], a7 = a[7][ix];
        // E(sy, sx) = F_ee + i sx F_eo + i sy F_oe - sx sy F_oo
        float re[4], im[4];
        re[0] = a0 - a3 - a5 - a6;  im[0] = a1 + a2 + a4 - a7;   // (+y, +x)
        re[1] = a0 + a3 - a5 + a6;  im[1] = a1 - a2 + a4 + a7;   // (+y, -x)  mirrored column
        re[2] = a0 - a3 + a5 + a6;  im[2] = a1 + a2 - a4 + a7;   // (-y, +x)  mirrored row
        re[3] = a0 + a3 + a5 - a6;  im[3] = a1 - a2 - a4 - a7;   // (-y, -x)
#pragma unroll
        for (int q = 0; q < 4; ++q) inten[p][ix][q] = fmaf(w, re[q] * re[q] + im[q] * im[q], inten[p][ix][q]);
        if (FIELD) {
          const int mx = mx0 + ix;
          if (my < m && mx < m) {
            float2 *fo = field + ((size_t)c * P.Z + b) * (size_t)M * M;
            const int myr = M - 1 - my, mxr = M - 1 - mx;
            fo[(size_t)my * M + mx] = make_float2(re[0], im[0]);
            fo[(size_t)my * M + mxr] = make_float2(re[1], im[1]);
            fo[(size_t)myr * M + mx] = make_float2(re[2], im[2]);
            fo[(size_t)myr * M + mxr] = make_float2(re[3], im[3]);
          }
        }
      }
    }
  }

  float *Ib = I + (size_t)b * M * M;
#pragma unroll
  for (int p = 0; p < PASS2; ++p) {
    const int tile = (tid >> 1) + 64 * p;
    const int my = (tile / (MXS / 2)) * 2 + (tid & 1), mx0 = mx_base + (tile % (MXS / 2)) * 2;
#pragma unroll
    for (int ix = 0; ix < 2; ++ix) {
      const int mx = mx0 + ix;
      if (my < m && mx < m) {
        const int myr = M - 1 - my, mxr = M - 1 - mx;
        Ib[(size_t)my * M + mx] = inten[p][ix][0];
        Ib[(size_t)my * M + mxr] = inten[p][ix][1];
        Ib[(size_t)myr * M + mx] = inten[p][ix][2];
        Ib[(size_t)myr * M + mxr] = inten[p][ix][3];
      }
    }
  }
}

template <int MQ, bool PP, bool FIELD, int STRIPS = 1>
cudaError_t launch_one(const DevPlan &P, cudaStream_t st, float *intensity, float2 *field) {
  k_small<MQ, PP, FIELD, STRIPS><<<dim3(P.Z, STRIPS), SM_THREADS, (int)sizeof(SmallSmem<MQ, PP>), st>>>(P, intensity, field);
  return cudaGetLastError();
}

template <int MQ, bool PP, bool FIELD, int STRIPS = 1>
cudaError_t set_attr() {
  return cudaFuncSetAttribute(k_small<MQ, PP, FIELD, STRIPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SmallSmem<MQ, PP>));
}

template <int MQ>
cudaError_t launch_mq(const DevPlan &P, cudaStream_t st, float *intensity, float2 *field) {
  if (P.per_plane) return field ? launch_one<MQ, true, true>(P, st, intensity, field) : launch_one<MQ, true, false>(P, st, intensity, field);
  if (MQ == 32 && !field && P.Z * 4 <= 148) return launch_one<32, false, false, 4>(P, st, intensity, field);   // short static stacks: m_x strips
  if (MQ == 32 && !field && P.Z * 2 <= 148) return launch_one<32, false, false, 2>(P, st, intensity, field);
  return field ? launch_one<MQ, false, true>(P, st, intensity, field) : launch_one<MQ, false, false>(P, st, intensity, field);
}

}  // namespace

bool small_eligible(const psf_plan *p) { return p->dp.n <= NQ && p->dp.m <= 32; }

// The dynamic shared memory of every instantiation exceeds the 48 KB default.  Function attributes are per device, so
// every plan sets them at creation with its own device current (idempotent, no per-process flag).
cudaError_t small_setup() {
  cudaError_t e;
  if ((e = set_attr<16, false, false>()) != cudaSuccess || (e = set_attr<16, false, true>()) != cudaSuccess ||
      (e = set_attr<16, true, false>()) != cudaSuccess || (e = set_attr<16, true, true>()) != cudaSuccess ||
      (e = set_attr<32, false, false>()) != cudaSuccess || (e = set_attr<32, false, true>()) != cudaSuccess ||
      (e = set_attr<32, true, false>()) != cudaSuccess || (e = set_attr<32, true, true>()) != cudaSuccess ||
      (e = set_attr<32, false, false, 2>()) != cudaSuccess || (e = set_attr<32, false, false, 4>()) != cudaSuccess)
    return e;
  return cudaSuccess;
}

cudaError_t launch_small(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field) {
  const DevPlan &P = p->dp;
  cudaError_t e = (P.m <= 16) ? launch_mq<16>(P, st, intensity, field) : launch_mq<32>(P, st, intensity, field);
  prof_mark(p, st, 0);
  return e;
}

}  // namespace psf
