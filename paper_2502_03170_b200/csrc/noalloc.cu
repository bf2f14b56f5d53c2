// psf_propagate_static (include/psf.h): the zoomed Fourier sum of PAPER.md:116 Eq. 9 for pupils the caller already holds on
// the device, for callers that cannot allocate device memory at all (no plan: psf_plan_create allocates).  It is the
// two-stage fp32 route of kernels_ffma.cu (rows, then columns with |E|^2 in the epilogue) in its plainest form - unfolded
// complex products - with the stage-1 -> stage-2 scratch T^T and the DFT table in ONE file-scope device array instead of
// plan-owned cudaMalloc memory.
//
//   * The array is `static __device__`: every device that loads this module holds NA_SCRATCH_BYTES until the process exits.
//   * In host code its name is a host-side stand-in, not a device address.  The address is looked up once per device, with
//     that device current, by cudaGetSymbolAddress (scratch_of_current_device), and that pointer is what the kernels get.
//   * All calls on a device share the array and it keeps the last call's contents.  Nothing here needs to start at zero:
//     the table is rewritten by every call and stage 2 reads only what stage 1 of the same pass wrote (tile loads are
//     bounds-checked, out-of-range operands are zero).  Calls that overlap on the GPU (two streams, two threads) race on it.
//   * No cudaMalloc / cudaFree / allocating library routine: launches only, plus the one-off symbol look-up.
#include <cmath>
#include <mutex>

#include "plan.hpp"

namespace psf {
void set_thread_error(const char *msg) noexcept;   // api.cu: the message psf_last_error(NULL) returns on this thread
}

namespace {

constexpr size_t NA_SCRATCH_BYTES = (size_t)PSF_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[NA_SCRATCH_BYTES];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_scratch_mu;
void *g_scratch_ptr[NA_MAX_DEVICES] = {};

// Device address of g_static_scratch on the current device (looked up once per device).
cudaError_t scratch_of_current_device(void **out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

// A[m][q] = exp(2 pi i t),  t = (NA pixel / lambda) u_q (m - (M - 1) / 2),  u_q = (2 q + 1 - N) / N  (readings A4, A6);
// the phase in turns in fp64, reduced, then rounded once to fp32 (the plan-time tables are made the same way).
__global__ void na_table(float2 *__restrict__ A, int M, int N, double turns_per_pixel) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M * N) return;
  const int m = i / N, q = i - m * N;
  double t = turns_per_pixel * ((double)(2 * q + 1 - N) / (double)N) * ((double)m - 0.5 * (double)(M - 1));
  t -= rint(t);
  double s, c;
  sincospi(2.0 * t, &s, &c);
  A[i] = make_float2((float)c, (float)s);
}

constexpr int NA_TILE = 64, NA_KT = 16, NA_LD = NA_TILE + 2;

struct NaArgs {
  const float2 *A;        // [I][K]  the table (no batch stride)
  const float2 *B;        // [batch][J][K]
  float2 *T;              // !FINAL: out [batch][I][J]
  float *Iout;            // FINAL:  out [batch][I][J], sum over the C components of a batch entry
  int I, J, K, C;
  float w[5];
};

// out[i][j] = sum_k A[i][k] B[j][k] (complex, fp32).  64 x 64 tile, 256 threads, 4 x 4 outputs per thread.
// FINAL: B holds C matrices per batch entry; the output is sum_c w_c |out_c|^2.
template <bool FINAL>
__global__ void __launch_bounds__(256) na_cgemm_nt(const NaArgs P) {
  __shared__ __align__(16) float2 As[NA_KT][NA_LD], Bs[NA_KT][NA_LD];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int i0 = blockIdx.y * NA_TILE, j0 = blockIdx.x * NA_TILE;
  const int lrow = threadIdx.x >> 2, lk = (threadIdx.x & 3) * 4;
  const size_t JK = (size_t)P.J * P.K;
  float inten[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) inten[a][b] = 0.f;
  const int ncomp = FINAL ? P.C : 1;
  for (int c = 0; c < ncomp; ++c) {
    const float2 *Bm = P.B + ((size_t)blockIdx.z * ncomp + c) * JK;
    float2 acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) acc[a][b] = make_float2(0.f, 0.f);
    for (int k0 = 0; k0 < P.K; k0 += NA_KT) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int k = k0 + lk + e;
        const int ia = i0 + lrow, jb = j0 + lrow;
        As[lk + e][lrow] = (ia < P.I && k < P.K) ? __ldg(P.A + (size_t)ia * P.K + k) : make_float2(0.f, 0.f);
        Bs[lk + e][lrow] = (jb < P.J && k < P.K) ? __ldg(Bm + (size_t)jb * P.K + k) : make_float2(0.f, 0.f);
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < NA_KT; ++k) {
        float2 a[4], b[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) { a[e] = As[k][ty * 4 + e]; b[e] = Bs[k][tx * 4 + e]; }
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            acc[ii][jj].x = fmaf(a[ii].x, b[jj].x, fmaf(-a[ii].y, b[jj].y, acc[ii][jj].x));
            acc[ii][jj].y = fmaf(a[ii].x, b[jj].y, fmaf(a[ii].y, b[jj].x, acc[ii][jj].y));
          }
      }
      __syncthreads();
    }
    if (FINAL) {
      const float w = P.w[c];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
          inten[ii][jj] = fmaf(w, acc[ii][jj].x * acc[ii][jj].x + acc[ii][jj].y * acc[ii][jj].y, inten[ii][jj]);
    } else {
      float2 *out = P.T + (size_t)blockIdx.z * P.I * P.J;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int i = i0 + ty * 4 + ii, j = j0 + tx * 4 + jj;
          if (i < P.I && j < P.J) out[(size_t)i * P.J + j] = acc[ii][jj];
        }
    }
  }
  if (FINAL) {
    float *out = P.Iout + (size_t)blockIdx.z * P.I * P.J;
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        const int i = i0 + ty * 4 + ii, j = j0 + tx * 4 + jj;
        if (i < P.I && j < P.J) out[(size_t)i * P.J + j] = inten[ii][jj];
      }
  }
}

psf_status na_fail(psf_status s, const std::string &msg) noexcept {
  psf::set_thread_error(msg.c_str());
  return s;
}

}  // namespace

extern "C" psf_status psf_propagate_static(void *cuda_stream, const void *pupil, int n_planes, int n_components, int pupil_n, int out_m,
                                           double NA, double wavelength_um, double pixel_um, const float *weights, float *intensity) {
  try {
    const int Z = n_planes, C = n_components, N = pupil_n, M = out_m;
    if (!pupil || !intensity || !weights) return na_fail(PSF_ERR_INVALID_ARG, "psf_propagate_static: pupil, weights and intensity must not be NULL");
    if (((uintptr_t)pupil & 7) || ((uintptr_t)intensity & 3))
      return na_fail(PSF_ERR_INVALID_ARG, "psf_propagate_static: pupil must be 8-byte aligned, intensity 4-byte aligned");
    if (Z < 1 || C < 1 || C > 5 || N < 1 || M < 1)
      return na_fail(PSF_ERR_INVALID_ARG, "psf_propagate_static: need n_planes >= 1, 1 <= n_components <= 5, pupil_n >= 1, out_m >= 1");
    if (!(NA > 0) || !(wavelength_um > 0) || !(pixel_um > 0) || !std::isfinite(NA) || !std::isfinite(wavelength_um) || !std::isfinite(pixel_um))
      return na_fail(PSF_ERR_INVALID_ARG, "psf_propagate_static: NA, wavelength_um and pixel_um must be finite and positive");
    NaArgs base = {};
    for (int c = 0; c < C; ++c) {
      if (!std::isfinite(weights[c])) return na_fail(PSF_ERR_INVALID_ARG, "psf_propagate_static: non-finite weight");
      base.w[c] = weights[c];
    }
    // the static scratch holds the table [M][N] and T^T [zc][C][M][N] (float2), zc >= 1 planes per pass
    auto up256 = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t tab_bytes = up256((size_t)M * N * sizeof(float2));
    const size_t plane_bytes = (size_t)C * M * N * sizeof(float2);
    if ((size_t)M > 32768 || (size_t)N > 32768 || tab_bytes + plane_bytes > NA_SCRATCH_BYTES)
      return na_fail(PSF_ERR_UNSUPPORTED,
                     "psf_propagate_static: (n_components + 1) * out_m * pupil_n * 8 bytes = " + std::to_string(tab_bytes + plane_bytes) +
                         " exceed the static scratch of " + std::to_string(NA_SCRATCH_BYTES) +
                         " bytes (PSF_STATIC_SCRATCH_BYTES); use a plan (psf_plan_create / psf_compute) for this size");
    void *scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess)
      return na_fail(PSF_ERR_CUDA, std::string("psf_propagate_static: cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float2 *tab = (float2 *)scratch;
    float2 *T = (float2 *)((unsigned char *)scratch + tab_bytes);
    size_t zc = (NA_SCRATCH_BYTES - tab_bytes) / plane_bytes;
    if (zc > (size_t)Z) zc = Z;
    if (zc > 65535 / (size_t)C) zc = 65535 / (size_t)C;          // gridDim.z of stage 1 is zc * C
    na_table<<<(unsigned)(((size_t)M * N + 255) / 256), 256, 0, st>>>(tab, M, N, NA * pixel_um / wavelength_um);
    const unsigned tm = (unsigned)((M + NA_TILE - 1) / NA_TILE), tn = (unsigned)((N + NA_TILE - 1) / NA_TILE);
    const float2 *P = (const float2 *)pupil;
    for (int z0 = 0; z0 < Z; z0 += (int)zc) {
      const int zn = (Z - z0 < (int)zc) ? (Z - z0) : (int)zc;
      // rows:    T^T[c][mx][py] = sum_px A[mx][px] P[c][py][px]
      NaArgs a1 = base;
      a1.A = tab; a1.B = P + (size_t)z0 * C * N * N; a1.T = T; a1.I = M; a1.J = N; a1.K = N; a1.C = 1;
      na_cgemm_nt<false><<<dim3(tn, tm, (unsigned)(zn * C)), 256, 0, st>>>(a1);
      // columns: E_c[my][mx] = sum_py A[my][py] T^T[c][mx][py];  I = sum_c w_c |E_c|^2
      NaArgs a2 = base;
      a2.A = tab; a2.B = T; a2.Iout = intensity + (size_t)z0 * M * M; a2.I = M; a2.J = M; a2.K = N; a2.C = C;
      na_cgemm_nt<true><<<dim3(tm, tm, (unsigned)zn), 256, 0, st>>>(a2);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(PSF_ERR_CUDA, std::string("psf_propagate_static: kernel launch: ") + cudaGetErrorString(e));
    return PSF_OK;
  } catch (...) {
    psf::set_thread_error("psf_propagate_static: out of host memory (or another C++ exception)");
    return PSF_ERR_ALLOC;
  }
}
