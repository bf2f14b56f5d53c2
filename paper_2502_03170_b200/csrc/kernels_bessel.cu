// Spherical (Bessel) parametrisation of the same propagation integral, Eq. 10-14 (Eq. 5 for the scalar
// model): for axisymmetric pupils the phi integral is done in closed form and the field needs three 1-D integrals over
// theta per (radius, plane),
//     I_n(rho, z) = sum_j A_j f_n(theta_j) J_n(k rho sin theta_j) exp(i k z cos theta_j),     n = 0, 1, 2,
//     f_0 = q_s + q_p cos theta,  f_1 = q_p sin theta,  f_2 = q_p cos theta - q_s  (q_s = q_p = 1 without PSF_FLAG_FRESNEL),
//     A_j = Simpson weight x a(theta_j) x sin theta_j x exp(i W_j)
// (SURVEY.md §8(f) NEXT-2).  The Bessel values do not depend on the plane and the plane phasors do not depend on the
// radius, so a thread owns one radius, evaluates J_0, J_1 (and J_2 by recurrence) once per node and feeds them to the
// accumulators of ZC planes whose phasors sit in shared memory.  ALU / SFU bound; no tensor cores (the contraction
// [radii x nodes] x [nodes x planes] is 0.2 TFLOP at config-5 size, the cost is the 1e9 Bessel evaluations).
//   k_bessel_integrals : (radius tile, plane chunk) -> I_n[z][r][3] complex fp32
//   k_bessel_combine   : per output pixel, Eq. 11 with the Jones vector, |E|^2 (unpolarised: 1/2 (I_x + I_y))
#include <cmath>
#include <vector>

#include "plan.hpp"
#include "pupil_gen.cuh"

namespace psf {

struct BesselState {
  int n_nodes = 0, R = 0;
  void *d_nodes = nullptr;   // float  [n]: sin theta
  void *d_af = nullptr;      // float2 [3][n]: A_j f_n(theta_j), f_n = (q_s + q_p cos), q_p sin, (q_p cos - q_s)  (scalar: A_j)
  void *d_kt = nullptr;      // float2 [n]: k cos theta / 2 pi in turns per um (hi, lo)
  void *d_kr = nullptr;      // float  [R]: k rho of the distinct radii of the folded output grid
  void *d_int = nullptr;     // float2 [Z][R][3]
  float pref2 = 0.f;         // |prefactor|^2: k^2 / 4 (Eq. 11) or k^2 (Eq. 5)
  float jones[4] = {1, 0, 0, 0};
  int unpol = 0, scalar = 0;
};

namespace {

constexpr int BZ = 16;        // planes per CTA
constexpr int BN = 32;        // nodes per shared-memory chunk
constexpr int BT = 128;       // threads = radii per CTA

template <bool SCALAR>
__global__ void __launch_bounds__(BT)
k_bessel_integrals(const float *__restrict__ sinth, const float2 *__restrict__ af, const float2 *__restrict__ kt,
                   const float *__restrict__ kr, const float4 *__restrict__ planes, float2 *__restrict__ out, int n_nodes, int R, int Z,
                   int chunks_per_split) {
  constexpr int NI = SCALAR ? 1 : 3;
  __shared__ float2 Bs[NI][BN][BZ];   // A_j f_n(theta_j) exp(i k z cos theta_j) of the chunk
  __shared__ float Ss[BN];            // sin theta_j
  const int r = blockIdx.x * BT + threadIdx.x;
  const int z0 = blockIdx.y * BZ;
  const float x_r = r < R ? __ldg(kr + r) : 0.f;
  float2 acc[NI][BZ];
#pragma unroll
  for (int n = 0; n < NI; ++n)
#pragma unroll
    for (int z = 0; z < BZ; ++z) acc[n][z] = make_float2(0.f, 0.f);

  // small grids: the node range is split over gridDim.z CTAs whose partial sums meet in `out` by atomic adds
  const int j_begin = blockIdx.z * chunks_per_split * BN;
  const int j_end = min(n_nodes, j_begin + chunks_per_split * BN);
  for (int j0 = j_begin; j0 < j_end; j0 += BN) {
    __syncthreads();
    for (int i = threadIdx.x; i < BN * BZ; i += BT) {
      const int jl = i / BZ, zl = i % BZ;
      const int j = j0 + jl, z = z0 + zl;
      float sn = 0.f, cs = 0.f;
      const bool ok = j < n_nodes && z < Z;
      if (ok) {
        const float4 pl = __ldg(planes + z);
        sincospif(2.0f * kz_turns(__ldg(kt + j), pl.x, pl.y), &sn, &cs);
      }
#pragma unroll
      for (int n = 0; n < NI; ++n) {
        const float2 a = ok ? __ldg(af + (size_t)n * n_nodes + j) : make_float2(0.f, 0.f);
        Bs[n][jl][zl] = make_float2(a.x * cs - a.y * sn, a.x * sn + a.y * cs);
      }
    }
    if (threadIdx.x < BN) Ss[threadIdx.x] = (j0 + threadIdx.x < n_nodes) ? __ldg(sinth + j0 + threadIdx.x) : 0.f;
    __syncthreads();
    // two-level accumulation: the chunk's partial sums are added to the running totals once per chunk
    float2 part[NI][BZ];
#pragma unroll
    for (int n = 0; n < NI; ++n)
#pragma unroll
      for (int z = 0; z < BZ; ++z) part[n][z] = make_float2(0.f, 0.f);
#pragma unroll 2
    for (int jl = 0; jl < BN; ++jl) {
      const float x = x_r * Ss[jl];
      float w[NI];
      w[0] = j0f(x);
      if (!SCALAR) {
        const float J1 = j1f(x);
        w[1 % NI] = J1;
        w[2 % NI] = x > 1e-3f ? fmaf(2.0f / x, J1, -w[0]) : 0.125f * x * x;   // recurrence; series below 1e-3
      }
#pragma unroll
      for (int n = 0; n < NI; ++n)
#pragma unroll
        for (int z = 0; z < BZ; ++z) {
          const float2 b = Bs[n][jl][z];
          part[n][z].x = fmaf(w[n], b.x, part[n][z].x);
          part[n][z].y = fmaf(w[n], b.y, part[n][z].y);
        }
    }
#pragma unroll
    for (int n = 0; n < NI; ++n)
#pragma unroll
      for (int z = 0; z < BZ; ++z) { acc[n][z].x += part[n][z].x; acc[n][z].y += part[n][z].y; }
  }
  if (r < R) {
#pragma unroll
    for (int z = 0; z < BZ; ++z)
      if (z0 + z < Z) {
        float2 *o = out + ((size_t)(z0 + z) * R + r) * 3;
        if (gridDim.z == 1) {
#pragma unroll
          for (int n = 0; n < NI; ++n) o[n] = acc[n][z];
        } else {
#pragma unroll
          for (int n = 0; n < NI; ++n) { atomicAdd(&o[n].x, acc[n][z].x); atomicAdd(&o[n].y, acc[n][z].y); }
        }
      }
  }
}

struct CombineArgs {
  const float2 *ints;   // [Z][R][3]
  float *intensity;     // [Z][M][M]
  int M, m, R, Z;
  float pixel, pref2;
  float jones[4];
  int unpol, scalar;
};

__device__ __forceinline__ float cabs2(float2 a) { return a.x * a.x + a.y * a.y; }

__global__ void k_bessel_combine(const CombineArgs P) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t MM = (size_t)P.M * P.M;
  if (idx >= MM * P.Z) return;
  const int z = (int)(idx / MM);
  const int iy = (int)((idx % MM) / P.M), ix = (int)(idx % P.M);
  const int my = min(iy, P.M - 1 - iy), mx = min(ix, P.M - 1 - ix);
  const int a = min(my, mx), b = max(my, mx);
  const float2 *I = P.ints + ((size_t)z * P.R + (size_t)b * (b + 1) / 2 + a) * 3;
  const float2 I0 = I[0];
  float val;
  if (P.scalar) {
    val = cabs2(I0);
  } else {
    const float2 I1 = I[1], I2 = I[2];
    const float x = ((float)ix - 0.5f * (float)(P.M - 1)) * P.pixel, y = ((float)iy - 0.5f * (float)(P.M - 1)) * P.pixel;
    const float rr = sqrtf(x * x + y * y);
    const float cp = rr > 0.f ? x / rr : 1.f, sp = rr > 0.f ? y / rr : 0.f;
    const float c2 = cp * cp - sp * sp, s2 = 2.f * sp * cp;
    // Eq. 11 for a Jones vector (px, py): columns of the matrix acting on (px, py)
    const float2 axx = make_float2(I0.x - I2.x * c2, I0.y - I2.y * c2);     // E_x from p_x
    const float2 axy = make_float2(-I2.x * s2, -I2.y * s2);                 // E_x from p_y = E_y from p_x
    const float2 ayy = make_float2(I0.x + I2.x * c2, I0.y + I2.y * c2);     // E_y from p_y
    const float2 azx = make_float2(2.f * I1.y * cp, -2.f * I1.x * cp);      // -2i I_1 cos(phi)
    const float2 azy = make_float2(2.f * I1.y * sp, -2.f * I1.x * sp);
    if (P.unpol) {
      val = 0.5f * (cabs2(axx) + 2.f * cabs2(axy) + cabs2(ayy) + cabs2(azx) + cabs2(azy));
    } else {
      const float2 px = make_float2(P.jones[0], P.jones[1]), py = make_float2(P.jones[2], P.jones[3]);
      auto cm = [](float2 u, float2 v) { return make_float2(u.x * v.x - u.y * v.y, u.x * v.y + u.y * v.x); };
      const float2 ex1 = cm(axx, px), ex2 = cm(axy, py), ey1 = cm(axy, px), ey2 = cm(ayy, py), ez1 = cm(azx, px), ez2 = cm(azy, py);
      val = cabs2(make_float2(ex1.x + ex2.x, ex1.y + ex2.y)) + cabs2(make_float2(ey1.x + ey2.x, ey1.y + ey2.y)) +
            cabs2(make_float2(ez1.x + ez2.x, ez1.y + ez2.y));
    }
  }
  P.intensity[idx] = P.pref2 * val;
}

}  // namespace

void bessel_free(psf_plan *p) {
  BesselState *b = p->bessel;
  if (!b) return;
  void *bufs[] = {b->d_nodes, b->d_af, b->d_kt, b->d_kr, b->d_int};
  for (void *q : bufs)
    if (q) cudaFree(q);
  delete b;
  p->bessel = nullptr;
}

// Host tables of the spherical path for `n_nodes` Simpson nodes; allocates the I_n scratch.
psf_status bessel_setup(psf_plan *p, int n_nodes) {
  const psf_plan_desc &d = p->desc;
  bessel_free(p);
  BesselState *b = new BesselState();
  p->bessel = b;
  BesselNodes B;
  build_bessel_nodes(d, n_nodes, B);
  b->n_nodes = n_nodes;
  const int M = d.out_m, m = (M + 1) / 2;
  b->R = m * (m + 1) / 2;
  b->scalar = d.model == PSF_MODEL_SCALAR;
  b->unpol = !b->scalar && d.pol == PSF_POL_UNPOLARIZED;
  const double pref = b->scalar ? B.k : 0.5 * B.k;
  b->pref2 = (float)(pref * pref);
  const double r2 = std::sqrt(0.5);
  double j[4] = {1, 0, 0, 0};
  switch (d.pol) {
    case PSF_POL_Y: j[0] = 0; j[2] = 1; break;
    case PSF_POL_CIRC_L: j[0] = r2; j[3] = r2; break;
    case PSF_POL_CIRC_R: j[0] = r2; j[3] = -r2; break;
    case PSF_POL_JONES: for (int i = 0; i < 4; ++i) j[i] = d.jones[i]; break;
    default: break;
  }
  for (int i = 0; i < 4; ++i) b->jones[i] = (float)j[i];
  std::vector<float> nodes(n_nodes);
  std::vector<float2> kt(n_nodes), af((size_t)3 * n_nodes);
  const double twopi = 6.283185307179586476925287;
  for (int i = 0; i < n_nodes; ++i) {
    nodes[i] = (float)B.sinth[i];
    for (int n = 0; n < 3; ++n) {
      const cplx v = b->scalar ? B.A[i] : B.A[i] * B.F[n][i];
      af[(size_t)n * n_nodes + i] = make_float2((float)v.real(), (float)v.imag());
    }
    const double t = B.k * B.costh[i] / twopi;
    const float hi = (float)t;
    kt[i] = make_float2(hi, (float)(t - (double)hi));
  }
  std::vector<float> kr(b->R);
  for (int bb = 0; bb < m; ++bb)
    for (int a = 0; a <= bb; ++a) {
      const double x = (a - 0.5 * (M - 1)) * d.pixel_um, y = (bb - 0.5 * (M - 1)) * d.pixel_um;
      kr[(size_t)bb * (bb + 1) / 2 + a] = (float)(B.k * std::sqrt(x * x + y * y));
    }
  auto up = [&](void **dst, const void *src, size_t bytes) {
    return cudaMalloc(dst, bytes) == cudaSuccess && cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!up(&b->d_nodes, nodes.data(), nodes.size() * sizeof(float)) || !up(&b->d_af, af.data(), af.size() * sizeof(float2)) || !up(&b->d_kt, kt.data(), kt.size() * sizeof(float2)) ||
      !up(&b->d_kr, kr.data(), kr.size() * sizeof(float)) ||
      cudaMalloc(&b->d_int, (size_t)d.n_planes * b->R * 3 * sizeof(float2)) != cudaSuccess) {
    p->err = "spherical path: device allocation / upload failed";
    bessel_free(p);
    return PSF_ERR_ALLOC;
  }
  return PSF_OK;
}

cudaError_t launch_bessel(const psf_plan *p, cudaStream_t st, float *intensity) {
  const BesselState *b = p->bessel;
  const DevPlan &D = p->dp;
  dim3 g1((b->R + BT - 1) / BT, (D.Z + BZ - 1) / BZ);
  // fewer CTAs than two per SM: split the Simpson nodes across gridDim.z (partial sums by atomic adds into a zeroed scratch)
  const int chunks = (b->n_nodes + BN - 1) / BN;
  int split = (2 * p->sm_count + (int)(g1.x * g1.y) - 1) / (int)(g1.x * g1.y);
  if (split > chunks) split = chunks;
  if (split < 1) split = 1;
  const int per = (chunks + split - 1) / split;
  g1.z = (chunks + per - 1) / per;
  if (g1.z > 1) cudaMemsetAsync(b->d_int, 0, (size_t)D.Z * b->R * 3 * sizeof(float2), st);
  if (b->scalar)
    k_bessel_integrals<true><<<g1, BT, 0, st>>>((const float *)b->d_nodes, (const float2 *)b->d_af, (const float2 *)b->d_kt,
                                                (const float *)b->d_kr, D.planes, (float2 *)b->d_int, b->n_nodes, b->R, D.Z, per);
  else
    k_bessel_integrals<false><<<g1, BT, 0, st>>>((const float *)b->d_nodes, (const float2 *)b->d_af, (const float2 *)b->d_kt,
                                                 (const float *)b->d_kr, D.planes, (float2 *)b->d_int, b->n_nodes, b->R, D.Z, per);
  prof_mark(p, st, 2);
  CombineArgs a;
  a.ints = (const float2 *)b->d_int; a.intensity = intensity; a.M = D.M; a.m = D.m; a.R = b->R; a.Z = D.Z;
  a.pixel = (float)p->desc.pixel_um; a.pref2 = b->pref2;
  for (int i = 0; i < 4; ++i) a.jones[i] = b->jones[i];
  a.unpol = b->unpol; a.scalar = b->scalar;
  const size_t total = (size_t)D.Z * D.M * D.M;
  k_bessel_combine<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(a);
  prof_mark(p, st, 3);
  return cudaGetLastError();
}

}  // namespace psf
