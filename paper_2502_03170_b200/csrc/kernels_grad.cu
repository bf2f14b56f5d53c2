// Adjoint of the hot path (the paper's motivation for a differentiable PSF):
// gradients of L = sum_{b,y,x} G[b,y,x] I[b,y,x] with respect to the defocus z_b of every plane and to the Zernike
// coefficients, given G = dL/dI.  With Q_c[p] the pupil field of plane b (base pupil x phasor) and A(x, p) the zoomed-DFT
// kernel exp(i k s_max (u_px x + u_py y)),
//     E_c(x)      = sum_p Q_c[p] A(x, p)                         forward, two products (rows, columns)
//     B_c[p]      = sum_x w_c G(x) conj(E_c(x)) A(x, p)          back-projection: the same two products, transposed
//     dL/dphi[p]  = -2 sum_c Im(Q_c[p] B_c[p])                   pupil-side sensitivity
//     dL/dz_b     = sum_p k cos(theta_p) dL/dphi[p],    dL/dc_bj = sum_p Z_j[p] dL/dphi[p].
// First correct version: unfolded complex fp32 FFMA products (one generic batched kernel C = A B^T used four times), own
// forward pass (the optimised kernels keep neither the unfolded pupil nor the fields of unpolarised light).  The tensor
// path is the next step; this file is the correctness vehicle and the API.
#include <cmath>
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

}  // namespace

void grad_free(psf_plan *p) {
  GradState *g = p->grad;
  if (!g) return;
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
    const cplx *src = p->h_base.data() + (size_t)(unpol ? pick[c] : c) * NN;
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

}  // namespace psf
