// Adjoint of the hot path (the paper's motivation for a differentiable PSF):
// gradients of L = sum_{b,y,x} G[b,y,x] I[b,y,x] with respect to the defocus z_b of every plane and to the Zernike
// coefficients, given G = dL/dI.  With Q_c[p] the pupil field of plane b (base pupil x phasor) and A(x, p) the zoomed-DFT
// kernel exp(i k s_max (u_px x + u_py y)),
//     E_c(x)      = sum_p Q_c[p] A(x, p)                         forward, two products (rows, columns)
//     B_c[p]      = sum_x w_c G(x) conj(E_c(x)) A(x, p)          back-projection: the same two products, transposed
//     dL/dphi[p]  = -2 sum_c Im(Q_c[p] B_c[p])                   pupil-side sensitivity
//     dL/dz_b     = sum_p k cos(theta_p) dL/dphi[p],    dL/dc_bj = sum_p Z_j[p] dL/dphi[p].
// Two routes:
//   * FFMA (round 1, the correctness vehicle; every mode): unfolded complex fp32 products (one generic batched kernel
//     C = A B^T used four times) with an own forward pass;
//   * tensor cores (static mode on the 3xFP16 path): the back-projection B_c = A_y^T H_c A_x, H_c = w_c G conj(E_c), is the
//     forward zoomed transform with the roles of the two grids swapped (pupil grid := the M x M image grid, output grid := the
//     N x N pupil grid, pixel' = pixel M / N: k s_max u_p x_m is symmetric in the two).  So: E_c from the plan's own tensor
//     kernels (field epilogue), one kernel that weights with G / max|G| and folds H_c into the four parity classes in the
//     stage-1 producers' table order, the SAME tensor kernels on a second plan ("plan B") whose stage 1 reads that
//     per-plane folded pupil instead of generating one (materialised-pupil mode, launch_tc_mat), and a reduction of
//     Im(Q B) against kappa and the Zernike basis with Q regenerated on the fly.  Neither Q nor T is written to HBM; E, the
//     folded H and B are (8 B per sample each).
#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

#include "plan.hpp"
#include "pupil_gen.cuh"

namespace psf {

struct GradState {
  int Cg = 0;                 // pupils pushed through: 1 scalar, 3 coherent, 6 unpolarised (x input, y input)
  int K = 0;                  // Zernike terms the gradient is taken for (shared or per plane)
  int zc = 1;                 // planes per pass
  float w[6] = {0, 0, 0, 0, 0, 0};
  void *d_base = nullptr;     // float2 [Cg][N][N]  unfolded static pupil (shared Zernike and mask folded in)
  void *d_kt = nullptr;       // float2 [N][N]      k cos(theta) / 2 pi (hi, lo)
  void *d_zb = nullptr;       // float  [K][N][N]   Zernike basis (radians per unit coefficient)
  void *d_ax = nullptr;       // float2 [M][N]      exp(i k s_max u_p x_m)
  void *d_axt = nullptr;      // float2 [N][M]      its transpose
  void *d_Q = nullptr, *d_T = nullptr, *d_E = nullptr, *d_B = nullptr;   // per-pass scratch
  long long version = -1;     // table version these copies were made from
  long long static_version = -1;   // the plan's static version at the last full setup
  int zb_first = 0;           // first Noll index of d_zb
  const float2 *base5 = nullptr;   // what g_dphi reads: d_base5, or the tensor path's own device copy after a device-side refresh
  // tensor-core route
  bool tensor = false;
  psf_plan *planB = nullptr;  // the back-projection plan (sizes swapped), owned
  int C5 = 0;                 // scalar pupils of the forward tensor path (1, 3, or 5 for unpolarised light)
  float w5[5] = {0, 0, 0, 0, 0};
  void *d_base5 = nullptr;    // float2 [C5][N][N]
  void *d_fieldE = nullptr;   // float2 [C5][Z][M][M]
  void *d_fieldB = nullptr;   // float2 [C5][Z][N][N]
  void *d_hfold = nullptr;    // float4 [Z][2][C5][npB][npB], the pair producers' order, times plan B's operand scale
  void *d_dummyI = nullptr;   // float  [Z][max(M, N)^2]
  void *d_gmax = nullptr;     // one float (bit pattern of max |G|)
};

namespace {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// Q[c][zl][p] = base_c[p] exp(2 pi i t),  t = kappa z / 2 pi (+ per-plane Zernike row and tilt)
__global__ void g_pupil(const DevPlan P, const float2 *__restrict__ base, const float2 *__restrict__ kt,
                        float2 *__restrict__ Q, int Cg, int z0, int zc) {
  const size_t NN = (size_t)P.N * P.N;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int zl = blockIdx.y;
  if (i >= NN) return;
  const int b = z0 + zl;
  const float4 pl = __ldg(P.planes + b);
  float t = kz_turns(__ldg(kt + i), pl.x, pl.y);
  if (P.per_plane) {
    for (int j = 0; j < P.K; ++j) t = fmaf(__ldg(P.coef + (size_t)b * P.K + j), __ldg(P.zb + (size_t)j * NN + i), t);
    if (P.has_shift) {
      const int py = (int)(i / P.N), px = (int)(i % P.N);
      const float ux = (float)(2 * px + 1 - P.N) / (float)P.N, uy = (float)(2 * py + 1 - P.N) / (float)P.N;
      t -= fmaf(ux, pl.z, uy * pl.w);
    }
  }
  float sn, cs;
  sincospif(2.0f * (t - rintf(t)), &sn, &cs);
  for (int c = 0; c < Cg; ++c)
    Q[((size_t)c * zc + zl) * NN + i] = cmul(__ldg(base + (size_t)c * NN + i), make_float2(cs, sn));
}

// Batched complex product C[b][i][j] = sum_k A[b][i][k] B[b][j][k]  (both operands K-contiguous).  strideA = 0 shares A.
constexpr int GT = 64, GK = 8;
__global__ void __launch_bounds__(256)
g_cgemm_nt(const float2 *__restrict__ A, size_t strideA, const float2 *__restrict__ B, size_t strideB, float2 *__restrict__ C,
           size_t strideC, int I, int J, int Kd) {
  __shared__ float2 As[GK][GT + 1], Bs[GK][GT + 1];
  const int bz = blockIdx.z;
  A += (size_t)bz * strideA; B += (size_t)bz * strideB; C += (size_t)bz * strideC;
  const int i0 = blockIdx.y * GT, j0 = blockIdx.x * GT;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float2 acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = make_float2(0.f, 0.f);
  for (int k0 = 0; k0 < Kd; k0 += GK) {
    for (int e = threadIdx.x; e < GT * GK; e += 256) {
      const int r = e / GK, k = e % GK;
      As[k][r] = (i0 + r < I && k0 + k < Kd) ? __ldg(A + (size_t)(i0 + r) * Kd + k0 + k) : make_float2(0.f, 0.f);
      Bs[k][r] = (j0 + r < J && k0 + k < Kd) ? __ldg(B + (size_t)(j0 + r) * Kd + k0 + k) : make_float2(0.f, 0.f);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < GK; ++k) {
      float2 a[4], b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { a[u] = As[k][ty + 16 * u]; b[u] = Bs[k][tx + 16 * u]; }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          acc[u][v].x = fmaf(a[u].x, b[v].x, fmaf(-a[u].y, b[v].y, acc[u][v].x));
          acc[u][v].y = fmaf(a[u].x, b[v].y, fmaf(a[u].y, b[v].x, acc[u][v].y));
        }
    }
    __syncthreads();
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const int i = i0 + ty + 16 * u, j = j0 + tx + 16 * v;
      if (i < I && j < J) C[(size_t)i * J + j] = acc[u][v];
    }
}

// H = w_c G conj(E), in place on E: [Cg][zc][M][M]
__global__ void g_weight(float2 *__restrict__ E, const float *__restrict__ G, int Cg, int zc, size_t MM, int z0, const float w0,
                         const float w1, const float w2, const float w3, const float w4, const float w5) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int zl = blockIdx.y;
  if (i >= MM) return;
  const float g = __ldg(G + (size_t)(z0 + zl) * MM + i);
  const float w[6] = {w0, w1, w2, w3, w4, w5};
  for (int c = 0; c < Cg; ++c) {
    float2 *e = E + ((size_t)c * zc + zl) * MM + i;
    const float2 v = *e;
    *e = make_float2(w[c] * g * v.x, -w[c] * g * v.y);
  }
}

// S[p] = -2 sum_c Im(Q_c[p] B_c[p]);  dL/dz_b += sum_p kappa_p S[p];  dL/dc[b][j] += sum_p Z_j[p] S[p]
__global__ void __launch_bounds__(256)
g_reduce(const float2 *__restrict__ Q, const float2 *__restrict__ B, const float2 *__restrict__ kt, const float *__restrict__ zb,
         double *__restrict__ dz, double *__restrict__ dc, int Cg, int zc, int K, size_t NN, int z0) {
  __shared__ double red[256];
  const int zl = blockIdx.y;
  constexpr int KMAX = 64;
  double accz = 0.0;
  float accc[KMAX];
  for (int j = 0; j < K; ++j) accc[j] = 0.f;
  // each thread covers a strided slice short enough for fp32 partial sums (<= 64 samples at N = 512)
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < NN; i += (size_t)gridDim.x * blockDim.x) {
    float s = 0.f;
    for (int c = 0; c < Cg; ++c) {
      const float2 q = __ldg(Q + ((size_t)c * zc + zl) * NN + i), b = __ldg(B + ((size_t)c * zc + zl) * NN + i);
      s -= 2.f * (q.x * b.y + q.y * b.x);
    }
    const float2 k = __ldg(kt + i);
    accz += 6.283185307179586 * ((double)k.x + (double)k.y) * (double)s;
    for (int j = 0; j < K; ++j) accc[j] = fmaf(__ldg(zb + (size_t)j * NN + i), s, accc[j]);
  }
  for (int j = -1; j < K; ++j) {
    red[threadIdx.x] = j < 0 ? accz : (double)accc[j];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) atomicAdd(j < 0 ? dz + z0 + zl : dc + (size_t)(z0 + zl) * K + j, red[0]);
    __syncthreads();
  }
}

// ---- tensor-core route ----------------------------------------------------------------------------------------------
__global__ void g_absmax(const float *__restrict__ G, size_t n, unsigned *__restrict__ out) {
  float m = 0.f;
  const size_t n4 = n >> 2;                      // G is 16-byte aligned (psf.h)
  const float4 *G4 = reinterpret_cast<const float4 *>(G);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
    const float4 v = __ldg(G4 + i);
    m = fmaxf(fmaxf(m, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
  }
  for (size_t i = (n4 << 2) + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) m = fmaxf(m, fabsf(__ldg(G + i)));
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));       // non-negative floats order like their bit patterns
}

struct WFArgs {
  const float2 *E;      // [C][Z][M][M]
  const float *G;       // [Z][M][M]
  const unsigned *gmax;
  float4 *hfold;        // [Z][2][C][np][np]
  int C, Z, M, mB, np;
  float w[5];
  float sQ;
};
// H_c = w_c (G / max|G|) conj(E_c), folded about both axes of the image grid into the four parity classes, written in the
// order the stage-1 pair producers read their base pupil (kernels_tc.cu, tc_setup): one thread per folded sample.
__global__ void __launch_bounds__(256) g_weight_fold(const WFArgs A) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int z = blockIdx.y;
  if (i >= A.mB * A.mB) return;
  const int qy = i / A.mB, qx = i - qy * A.mB;
  const int M = A.M, ry = M - 1 - qy, rx = M - 1 - qx;
  const bool selfx = rx == qx, selfy = ry == qy;
  const float gm = __uint_as_float(*A.gmax);
  const float inv = gm > 0.f ? 1.f / gm : 0.f;
  const size_t MM = (size_t)M * M;
  const float *Gz = A.G + (size_t)z * MM;
  const float g00 = __ldg(Gz + (size_t)qy * M + qx) * inv, g01 = __ldg(Gz + (size_t)qy * M + rx) * inv;
  const float g10 = __ldg(Gz + (size_t)ry * M + qx) * inv, g11 = __ldg(Gz + (size_t)ry * M + rx) * inv;
  const int nk = A.np / 64;
  const int jt = qy >> 6, half = (qy >> 5) & 1, ql = qy & 31, kc = qx >> 6, cgp = (qx >> 3) & 7, e = qx & 7;
  const size_t idx = ((size_t)(jt * nk + kc) * 2 + half) * 2048 + (size_t)e * 256 + ql * 8 + cgp;
  const size_t npp = (size_t)A.np * A.np;
  for (int c = 0; c < A.C; ++c) {
    const float2 *Ec = A.E + ((size_t)c * A.Z + z) * MM;
    const float w = A.w[c];
    auto H = [&](int y, int x, float g) { const float2 v = __ldg(Ec + (size_t)y * M + x); return make_float2(w * g * v.x, -w * g * v.y); };
    const float2 p00 = H(qy, qx, g00);
    const float2 p01 = selfx ? make_float2(0.f, 0.f) : H(qy, rx, g01);
    const float2 p10 = selfy ? make_float2(0.f, 0.f) : H(ry, qx, g10);
    const float2 p11 = (selfx || selfy) ? make_float2(0.f, 0.f) : H(ry, rx, g11);
    const float2 e0 = make_float2(p00.x + p01.x, p00.y + p01.y), o0 = selfx ? make_float2(0.f, 0.f) : make_float2(p00.x - p01.x, p00.y - p01.y);
    const float2 e1 = make_float2(p10.x + p11.x, p10.y + p11.y), o1 = selfx ? make_float2(0.f, 0.f) : make_float2(p10.x - p11.x, p10.y - p11.y);
    const float s = A.sQ;
    const float2 ee = make_float2(e0.x + e1.x, e0.y + e1.y), eo = make_float2(o0.x + o1.x, o0.y + o1.y);
    const float2 oe = selfy ? make_float2(0.f, 0.f) : make_float2(e0.x - e1.x, e0.y - e1.y);
    const float2 oo = selfy ? make_float2(0.f, 0.f) : make_float2(o0.x - o1.x, o0.y - o1.y);
    float4 *dst = A.hfold + ((size_t)z * 2 * A.C) * npp;
    dst[(size_t)(0 * A.C + c) * npp + idx] = make_float4(s * ee.x, s * ee.y, s * oe.x, s * oe.y);     // x-even group: ee, oe
    dst[(size_t)(1 * A.C + c) * npp + idx] = make_float4(s * eo.x, s * eo.y, s * oo.x, s * oo.y);     // x-odd group:  eo, oo
  }
}

// Pupil-side sensitivity S[z][p] = -2 max|G| sum_c Im(Q_c[p] B_c[p]), Q_c[p] = base_c[p] exp(i kappa_p z) regenerated here.
__global__ void __launch_bounds__(256)
g_dphi(const float2 *__restrict__ base, const float2 *__restrict__ B, const float2 *__restrict__ kt, const float4 *__restrict__ planes,
       const unsigned *__restrict__ gmax, float *__restrict__ S, int C, int Z, size_t NN) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int z = blockIdx.y;
  if (i >= NN) return;
  const float4 pl = __ldg(planes + z);
  float sn, cs;
  sincospif(2.0f * kz_turns(__ldg(kt + i), pl.x, pl.y), &sn, &cs);
  float s = 0.f;
  for (int c = 0; c < C; ++c) {
    const float2 q = cmul(__ldg(base + (size_t)c * NN + i), make_float2(cs, sn));
    const float2 b = __ldg(B + ((size_t)c * Z + z) * NN + i);
    s -= 2.f * (q.x * b.y + q.y * b.x);
  }
  S[(size_t)z * NN + i] = s * __uint_as_float(*gmax);
}

// dL/dz_b = sum_p kappa_p S[b][p],  dL/dc[b][j] = sum_p Z_j[p] S[b][p]: a skinny product [Z x N^2] . [N^2 x (K + 1)].
// Block = 16 planes x one chunk of 4096 samples, in tiles of 256 samples through shared memory; thread = (plane, j mod 16);
// fp32 sums inside a tile, fp64 across tiles, one atomicAdd per (block, plane, j).
constexpr int SR_ZT = 16, SR_TILE = 256, SR_CHUNK = 4096, SR_PITCH = SR_TILE + 1, SR_JMAX = 5;
__global__ void __launch_bounds__(256)
g_sred(const float *__restrict__ S, const float2 *__restrict__ kt, const float *__restrict__ zb, double *__restrict__ dz,
       double *__restrict__ dc, int Z, int K, size_t NN) {
  extern __shared__ float sr_smem[];
  float *Ss = sr_smem;                         // [SR_ZT][SR_PITCH]
  float *Ws = sr_smem + SR_ZT * SR_PITCH;      // [K + 1][SR_PITCH]: row 0 = kappa, row 1 + j = Z_j
  const int KW = K + 1;
  const int z0 = blockIdx.y * SR_ZT;
  const int tz = threadIdx.x >> 4, tj = threadIdx.x & 15;
  double acc[SR_JMAX] = {0.0, 0.0, 0.0, 0.0, 0.0};
  const size_t i0 = (size_t)blockIdx.x * SR_CHUNK;
  for (int t = 0; t < SR_CHUNK / SR_TILE; ++t) {
    const size_t ib = i0 + (size_t)t * SR_TILE;
    if (ib >= NN) break;
    __syncthreads();
    for (int e = threadIdx.x; e < SR_ZT * SR_TILE; e += 256) {
      const int zz = e / SR_TILE, ii = e % SR_TILE;
      Ss[zz * SR_PITCH + ii] = (z0 + zz < Z && ib + ii < NN) ? __ldg(S + (size_t)(z0 + zz) * NN + ib + ii) : 0.f;
    }
    for (int e = threadIdx.x; e < KW * SR_TILE; e += 256) {
      const int jj = e / SR_TILE, ii = e % SR_TILE;
      float w = 0.f;
      if (ib + ii < NN) {
        if (jj == 0) { const float2 k = __ldg(kt + ib + ii); w = 6.283185307179586f * (k.x + k.y); }
        else w = __ldg(zb + (size_t)(jj - 1) * NN + ib + ii);
      }
      Ws[jj * SR_PITCH + ii] = w;
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < SR_JMAX; ++u) {
      const int j = tj + 16 * u;
      if (j < KW) {
        float a = 0.f;
        const float *sr = Ss + tz * SR_PITCH, *wr = Ws + j * SR_PITCH;
#pragma unroll 8
        for (int ii = 0; ii < SR_TILE; ++ii) a = fmaf(sr[ii], wr[ii], a);
        acc[u] += (double)a;
      }
    }
  }
  if (z0 + tz < Z) {
#pragma unroll
    for (int u = 0; u < SR_JMAX; ++u) {
      const int j = tj + 16 * u;
      if (j < KW) {
        if (j == 0) atomicAdd(dz + z0 + tz, acc[u]);
        else if (dc) atomicAdd(dc + (size_t)(z0 + tz) * K + (j - 1), acc[u]);
      }
    }
  }
}

}  // namespace

void grad_free(psf_plan *p) {
  GradState *g = p->grad;
  if (!g) return;
  if (g->planB) { psf_plan_destroy(g->planB); g->planB = nullptr; }
  void *tbufs[] = {g->d_base5, g->d_fieldE, g->d_fieldB, g->d_hfold, g->d_dummyI, g->d_gmax};
  for (void *q : tbufs)
    if (q) cudaFree(q);
  void *bufs[] = {g->d_base, g->d_kt, g->d_zb, g->d_ax, g->d_axt, g->d_Q, g->d_T, g->d_E, g->d_B};
  for (void *q : bufs)
    if (q) cudaFree(q);
  delete g;
  p->grad = nullptr;
}

// (Re)builds the device tables of the adjoint from the plan's current host tables; allocates the per-pass scratch.
bool grad_needs_setup(const psf_plan *p) { return !(p->grad && p->grad->version == p->table_version); }

psf_status grad_setup(psf_plan *p) {
  const psf_plan_desc &d = p->desc;
  const DevPlan &D = p->dp;
  const int N = D.N, M = D.M;
  const size_t NN = (size_t)N * N, MM = (size_t)M * M, MN = (size_t)M * N;
  if (p->grad && p->grad->version == p->table_version) return PSF_OK;
  if (p->grad && p->grad->tensor && p->grad->static_version == p->static_version) {
    // only the shared pupil phase changed since the last full setup (device-side refresh): the back-projection plan, the
    // scratch and every static table stand; what moves is the unfolded pupil and, if the term list changed, the basis
    GradState *g = p->grad;
    const int K = (int)p->zern_shared.size();
    if (K != g->K || (K > 0 && p->zb_first != g->zb_first)) {
      std::vector<float> zb((size_t)K * NN);
      for (size_t i = 0; i < zb.size(); ++i) zb[i] = (float)p->zbasis[i];
      if (g->d_zb) { cudaFree(g->d_zb); g->d_zb = nullptr; }
      if (K > 0 && (cudaMalloc(&g->d_zb, zb.size() * sizeof(float)) != cudaSuccess ||
                    cudaMemcpy(g->d_zb, zb.data(), zb.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)) {
        p->err = "gradients: basis upload failed";
        grad_free(p);
        return PSF_ERR_ALLOC;
      }
      g->K = K;
      g->zb_first = p->zb_first;
    }
    g->base5 = tc_device_pupil(p);
    if (!g->base5) {                       // cannot happen while static_version stands, but stay correct if it does
      grad_free(p);
      return grad_setup(p);
    }
    g->version = p->table_version;
    return PSF_OK;
  }
  grad_free(p);
  GradState *g = new GradState();
  p->grad = g;
  auto fail = [&](const char *msg) { p->err = msg; grad_free(p); return PSF_ERR_ALLOC; };
  // pupils: scalar 1, coherent 3, unpolarised = x input (a, b, c_x) and y input (b, d, c_y), weight 1/2 each
  const HostPupil &hp = p->hp0;
  const bool unpol = hp.C == 5;
  g->Cg = unpol ? 6 : hp.C;
  const int pick[6] = {0, 1, 3, 1, 2, 4};
  for (int c = 0; c < g->Cg; ++c) g->w[c] = unpol ? 0.5f : 1.0f;
  std::vector<float2> base((size_t)g->Cg * NN);
  for (int c = 0; c < g->Cg; ++c) {
    const cplx *src = host_base(p).data() + (size_t)(unpol ? pick[c] : c) * NN;
    for (size_t i = 0; i < NN; ++i) base[(size_t)c * NN + i] = make_float2((float)src[i].real(), (float)src[i].imag());
  }
  std::vector<float2> kt(NN);
  const double twopi = 6.283185307179586476925287;
  for (size_t i = 0; i < NN; ++i) {
    const double t = hp.kappa[i] / twopi;
    const float hi = (float)t;
    kt[i] = make_float2(hi, (float)(t - (double)hi));
  }
  g->K = p->zern_shared.empty() ? p->K_rows : (int)p->zern_shared.size();
  g->zb_first = p->zb_first;
  g->static_version = p->static_version;
  std::vector<float> zb((size_t)g->K * NN);
  for (size_t i = 0; i < zb.size(); ++i) zb[i] = (float)p->zbasis[i];
  std::vector<float2> ax(MN), axt(MN);
  const double kk = twopi * d.NA / d.wavelength_um;
  for (int m = 0; m < M; ++m) {
    const double x = (m - 0.5 * (M - 1)) * d.pixel_um;
    for (int q = 0; q < N; ++q) {
      const double ph = kk * ((double)(2L * q + 1 - N) / N) * x;
      const float2 v = make_float2((float)std::cos(ph), (float)std::sin(ph));
      ax[(size_t)m * N + q] = v;
      axt[(size_t)q * M + m] = v;
    }
  }
  auto up = [&](void **dst, const void *src, size_t bytes) {
    if (bytes == 0) return true;
    return cudaMalloc(dst, bytes) == cudaSuccess && cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!up(&g->d_base, base.data(), base.size() * sizeof(float2)) || !up(&g->d_kt, kt.data(), kt.size() * sizeof(float2)) ||
      !up(&g->d_zb, zb.data(), zb.size() * sizeof(float)) || !up(&g->d_ax, ax.data(), ax.size() * sizeof(float2)) ||
      !up(&g->d_axt, axt.data(), axt.size() * sizeof(float2)))
    return fail("gradients: table upload failed");
  // tensor-core route: static mode on the 3xFP16 path, if the back-projection plan also lands there
  if (p->tune_grad_tensor && p->path == 2 && p->tc && !D.per_plane && tc_pair_stage1(p)) {
    const int C5 = hp.C;
    double hmax = 0.0;
    std::vector<float2> base5((size_t)C5 * NN);
    for (int c = 0; c < C5; ++c) {
      double l1 = 0.0;
      const cplx *src = host_base(p).data() + (size_t)c * NN;
      for (size_t i = 0; i < NN; ++i) { l1 += std::abs(src[i]); base5[(size_t)c * NN + i] = make_float2((float)src[i].real(), (float)src[i].imag()); }
      hmax = std::max(hmax, hp.weight[c] * l1);                 // |H_c| = w_c |G / max G| |E_c| <= w_c sum_p |base_c[p]|
    }
    psf_plan_desc db = d;
    std::vector<double> zeros(D.Z, 0.0);
    db.pupil_n = M; db.out_m = N; db.pixel_um = d.pixel_um * (double)M / (double)N;
    db.n_planes = D.Z; db.z_um = zeros.data(); db.precision = PSF_PREC_3XF16; db.device = p->device;
    psf_plan *pb = nullptr;
    if (psf_plan_create(&db, &pb) == PSF_OK && pb) {
      const int mB = (M + 1) / 2;
      pb->tune_fused = p->tune_fused;
      if (pb->path == 2 && tc_pair_stage1(pb) && plan_set_materialised(pb, 4.0 * hmax, 4.0 * hmax * mB) == PSF_OK && tc_pair_stage1(pb)) {
        const int np = tc_n_pad(pb);
        const size_t big = (size_t)D.Z * (MM > NN ? MM : NN);
        const size_t hf = (size_t)D.Z * 2 * C5 * np * np;
        if (cudaMalloc(&g->d_base5, base5.size() * sizeof(float2)) == cudaSuccess &&
            cudaMemcpy(g->d_base5, base5.data(), base5.size() * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess &&
            cudaMalloc(&g->d_fieldE, (size_t)C5 * D.Z * MM * sizeof(float2)) == cudaSuccess &&
            cudaMalloc(&g->d_fieldB, (size_t)C5 * D.Z * NN * sizeof(float2)) == cudaSuccess &&
            cudaMalloc(&g->d_hfold, hf * sizeof(float4)) == cudaSuccess && cudaMemset(g->d_hfold, 0, hf * sizeof(float4)) == cudaSuccess &&
            cudaMalloc(&g->d_dummyI, big * sizeof(float)) == cudaSuccess && cudaMalloc(&g->d_gmax, sizeof(unsigned)) == cudaSuccess) {
          cudaFuncSetAttribute(g_sred, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((SR_ZT + 65) * SR_PITCH * sizeof(float)));
          g->tensor = true;
          g->base5 = (const float2 *)g->d_base5;
          g->planB = pb;
          g->C5 = C5;
          for (int c = 0; c < C5; ++c) g->w5[c] = (float)hp.weight[c];
        }
      }
      if (!g->tensor) {                                         // not this time: free what was taken, the FFMA route runs
        psf_plan_destroy(pb);
        void **tb[] = {&g->d_base5, &g->d_fieldE, &g->d_fieldB, &g->d_hfold, &g->d_dummyI, &g->d_gmax};
        for (void **q : tb)
          if (*q) { cudaFree(*q); *q = nullptr; }
        cudaGetLastError();
      }
    }
  }
  if (g->tensor) { g->version = p->table_version; return PSF_OK; }
  // scratch: Q, B [Cg][zc][N][N]; T (and V) [Cg][zc][M][N]; E [Cg][zc][M][M]
  const size_t per_plane = (size_t)g->Cg * (2 * NN + MN + MM) * sizeof(float2);
  size_t zc = ((size_t)1 << 30) / per_plane;
  if (zc < 1) zc = 1;
  if (zc > (size_t)D.Z) zc = D.Z;
  if (zc > 65535 / (size_t)g->Cg) zc = 65535 / (size_t)g->Cg;   // gridDim.z of the batched products is Cg * zc
  g->zc = (int)zc;
  if (cudaMalloc(&g->d_Q, zc * g->Cg * NN * sizeof(float2)) != cudaSuccess || cudaMalloc(&g->d_B, zc * g->Cg * NN * sizeof(float2)) != cudaSuccess ||
      cudaMalloc(&g->d_T, zc * g->Cg * MN * sizeof(float2)) != cudaSuccess || cudaMalloc(&g->d_E, zc * g->Cg * MM * sizeof(float2)) != cudaSuccess)
    return fail("gradients: scratch allocation failed");
  g->version = p->table_version;
  return PSF_OK;
}

cudaError_t launch_grad(const psf_plan *p, cudaStream_t st, const float *dL_dI, double *dL_dz, double *dL_dc) {
  const GradState *g = p->grad;
  const DevPlan &D = p->dp;
  const int N = D.N, M = D.M, Cg = g->Cg;
  const size_t NN = (size_t)N * N, MM = (size_t)M * M, MN = (size_t)M * N;
  cudaMemsetAsync(dL_dz, 0, (size_t)D.Z * sizeof(double), st);
  if (dL_dc && g->K > 0) cudaMemsetAsync(dL_dc, 0, (size_t)D.Z * g->K * sizeof(double), st);
  if (g->tensor) {
    const psf_plan *pb = g->planB;
    cudaError_t e = launch_tc(p, st, (float *)g->d_dummyI, (float2 *)g->d_fieldE);                 // E_c, all planes
    if (e != cudaSuccess) return e;
    cudaMemsetAsync(g->d_gmax, 0, sizeof(unsigned), st);
    g_absmax<<<148 * 8, 256, 0, st>>>(dL_dI, (size_t)D.Z * MM, (unsigned *)g->d_gmax);
    WFArgs A;
    A.E = (const float2 *)g->d_fieldE; A.G = dL_dI; A.gmax = (const unsigned *)g->d_gmax; A.hfold = (float4 *)g->d_hfold;
    A.C = g->C5; A.Z = D.Z; A.M = M; A.mB = (M + 1) / 2; A.np = tc_n_pad(pb); A.sQ = tc_pupil_scale(pb);
    for (int c = 0; c < 5; ++c) A.w[c] = g->w5[c];
    g_weight_fold<<<dim3((unsigned)((A.mB * A.mB + 255) / 256), D.Z), 256, 0, st>>>(A);
    e = launch_tc_mat(pb, st, (float *)g->d_dummyI, (float2 *)g->d_fieldB, (const float4 *)g->d_hfold);   // B_c = A_y^T H_c A_x
    if (e != cudaSuccess) return e;
    const int Kt = dL_dc ? g->K : 0;
    // sensitivity S (fp32, in the dummy-intensity buffer, free by now), then the skinny product against kappa and the basis
    float *S = (float *)g->d_dummyI;
    g_dphi<<<dim3((unsigned)((NN + 255) / 256), D.Z), 256, 0, st>>>(g->base5, (const float2 *)g->d_fieldB, (const float2 *)g->d_kt,
                                                                   D.planes, (const unsigned *)g->d_gmax, S, g->C5, D.Z, NN);
    const size_t sr_bytes = (size_t)(SR_ZT + Kt + 1) * SR_PITCH * sizeof(float);
    g_sred<<<dim3((unsigned)((NN + SR_CHUNK - 1) / SR_CHUNK), (D.Z + SR_ZT - 1) / SR_ZT), 256, sr_bytes, st>>>(
        S, (const float2 *)g->d_kt, (const float *)g->d_zb, dL_dz, Kt ? dL_dc : nullptr, D.Z, Kt, NN);
    return cudaGetLastError();
  }
  float2 *Q = (float2 *)g->d_Q, *T = (float2 *)g->d_T, *E = (float2 *)g->d_E, *B = (float2 *)g->d_B;
  const float2 *ax = (const float2 *)g->d_ax, *axt = (const float2 *)g->d_axt;
  auto tiles = [](int n) { return (unsigned)((n + GT - 1) / GT); };
  for (int z0 = 0; z0 < D.Z; z0 += g->zc) {
    const int zc = (D.Z - z0 < g->zc) ? (D.Z - z0) : g->zc;
    const unsigned nb = (unsigned)(Cg * zc);          // batches are laid out [c][zl] with the pass's own zc
    g_pupil<<<dim3((unsigned)((NN + 255) / 256), zc), 256, 0, st>>>(D, (const float2 *)g->d_base, (const float2 *)g->d_kt, Q, Cg, z0, zc);
    // forward: T^T[mx][py] = sum_px Ax[mx][px] Q[py][px];  E[my][mx] = sum_py Ay[my][py] T^T[mx][py]
    g_cgemm_nt<<<dim3(tiles(N), tiles(M), nb), 256, 0, st>>>(ax, 0, Q, NN, T, MN, M, N, N);
    g_cgemm_nt<<<dim3(tiles(M), tiles(M), nb), 256, 0, st>>>(ax, 0, T, MN, E, MM, M, M, N);
    g_weight<<<dim3((unsigned)((MM + 255) / 256), zc), 256, 0, st>>>(E, dL_dI, Cg, zc, MM, z0, g->w[0], g->w[1], g->w[2], g->w[3], g->w[4], g->w[5]);
    // adjoint: V[px][my] = sum_mx Ax^T[px][mx] H[my][mx];  B[py][px] = sum_my Ay^T[py][my] V[px][my]
    g_cgemm_nt<<<dim3(tiles(M), tiles(N), nb), 256, 0, st>>>(axt, 0, E, MM, T, MN, N, M, M);
    g_cgemm_nt<<<dim3(tiles(N), tiles(N), nb), 256, 0, st>>>(axt, 0, T, MN, B, NN, N, N, M);
    g_reduce<<<dim3(16, zc), 256, 0, st>>>(Q, B, (const float2 *)g->d_kt, (const float *)g->d_zb, dL_dz, dL_dc, Cg, zc,
                                           dL_dc ? g->K : 0, NN, z0);
  }
  return cudaGetLastError();
}

int grad_terms(const psf_plan *p) { return p->grad ? p->grad->K : 0; }
const char *grad_route(const psf_plan *p) { return !p->grad ? "" : p->grad->tensor ? "adjoint_tc3xf16" : "adjoint_ffma"; }

}  // namespace psf
