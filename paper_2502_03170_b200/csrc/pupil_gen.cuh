// Device-side pupil-field producer (step a1 of SURVEY.md §8(a)): P_c[b][p] = B_c[p] exp(i(kappa[p] z_b + ...)),
// delivered already folded into the four parity classes.  Shared by the FFMA and the tcgen05 kernels.
#pragma once
#include "plan.hpp"

namespace psf {

// exp(2 pi i * kt * z) with kt = (hi, lo) turns/um and z = (hi, lo) um, evaluated with a compensated product so that
// the reduced argument is accurate to ~1e-8 turns for |kt z| up to hundreds of turns.
__device__ __forceinline__ float kz_turns(float2 kt, float zh, float zl) {
  const float p = kt.x * zh;
  const float e = fmaf(kt.x, zh, -p);                       // exact error of the leading product
  const float r = p - rintf(p);                             // exact
  return r + (e + fmaf(kt.x, zl, kt.y * zh));
}

// Static mode: the four folded class values of component c at folded sample (qy, qx), times exp(i kappa z).
// out[0..7] = (ee.re, ee.im, eo.re, eo.im, oe.re, oe.im, oo.re, oo.im)
__device__ __forceinline__ void gen_static(const DevPlan &P, int c, int qy, int qx, float zh, float zl, float out[8]) {
  const size_t s = (size_t)qy * P.n + qx;
  const float2 kt = __ldg(P.kt + s);
  float sn, cs;
  sincospif(2.0f * kz_turns(kt, zh, zl), &sn, &cs);
  const float4 b0 = __ldg(P.bfold + ((size_t)c * P.n * P.n + s) * 2);
  const float4 b1 = __ldg(P.bfold + ((size_t)c * P.n * P.n + s) * 2 + 1);
  out[0] = b0.x * cs - b0.y * sn;  out[1] = b0.x * sn + b0.y * cs;
  out[2] = b0.z * cs - b0.w * sn;  out[3] = b0.z * sn + b0.w * cs;
  out[4] = b1.x * cs - b1.y * sn;  out[5] = b1.x * sn + b1.y * cs;
  out[6] = b1.z * cs - b1.w * sn;  out[7] = b1.z * sn + b1.w * cs;
}

// Per-plane mode: evaluates the unfolded pupil at the four mirror images of (qy, qx) with the plane's own Zernike
// row and tilt, then folds.
__device__ __forceinline__ void gen_per_plane(const DevPlan &P, int c, int b, int qy, int qx, float4 pl, float out[8]) {
  const int N = P.N;
  const float2 kt = __ldg(P.kt + (size_t)qy * P.n + qx);
  const float t0 = kz_turns(kt, pl.x, pl.y);
  const int iy[2] = {qy, N - 1 - qy}, ix[2] = {qx, N - 1 - qx};
  float2 v[2][2];
#pragma unroll
  for (int a = 0; a < 2; ++a) {
#pragma unroll
    for (int bb = 0; bb < 2; ++bb) {
      const size_t s = (size_t)iy[a] * N + ix[bb];
      float t = 0.f;
      for (int j = 0; j < P.K; ++j) t = fmaf(__ldg(P.coef + (size_t)b * P.K + j), __ldg(P.zb + (size_t)j * N * N + s), t);
      if (P.has_shift) {
        const float ux = (float)(2 * ix[bb] + 1 - N) / (float)N, uy = (float)(2 * iy[a] + 1 - N) / (float)N;
        t -= fmaf(ux, pl.z, uy * pl.w);
      }
      t += t0;
      float sn, cs;
      sincospif(2.0f * (t - rintf(t)), &sn, &cs);
      const float2 bu = __ldg(P.bunf + (size_t)c * N * N + s);
      v[a][bb] = make_float2(bu.x * cs - bu.y * sn, bu.x * sn + bu.y * cs);
    }
  }
  if (ix[1] == ix[0]) { v[0][1] = make_float2(0.f, 0.f); v[1][1] = make_float2(0.f, 0.f); }   // odd N: self-mirror column
  if (iy[1] == iy[0]) { v[1][0] = make_float2(0.f, 0.f); v[1][1] = make_float2(0.f, 0.f); }   // self-mirror row
  // fold x then y
  const float2 e0 = make_float2(v[0][0].x + v[0][1].x, v[0][0].y + v[0][1].y);   // even-x, row qy
  const float2 o0 = make_float2(v[0][0].x - v[0][1].x, v[0][0].y - v[0][1].y);
  const float2 e1 = make_float2(v[1][0].x + v[1][1].x, v[1][0].y + v[1][1].y);   // even-x, mirror row
  const float2 o1 = make_float2(v[1][0].x - v[1][1].x, v[1][0].y - v[1][1].y);
  const bool selfx = ix[1] == ix[0];
  out[0] = e0.x + e1.x;  out[1] = e0.y + e1.y;                                     // ee
  out[2] = selfx ? 0.f : o0.x + o1.x;  out[3] = selfx ? 0.f : o0.y + o1.y;         // eo (even y, odd x)
  out[4] = e0.x - e1.x;  out[5] = e0.y - e1.y;                                     // oe (odd y, even x)
  out[6] = selfx ? 0.f : o0.x - o1.x;  out[7] = selfx ? 0.f : o0.y - o1.y;         // oo
  if (iy[1] == iy[0]) { out[4] = out[5] = out[6] = out[7] = 0.f; }
}

}  // namespace psf
