// Chirp-Z path (PSF_PREC_CZT_FFT): the paper's own formulation of the zoomed DFT (PAPER.md:47, :217 -- "a custom variant of
// the 2D FFT ... chirp Z-transform ... three FFTs ... size doubled"), with hand-written shared-memory FFTs (no cuFFT).
// built to measure the matrix-vs-FFT crossover in N against the tensor-core product form.
//
// The finite sum of one axis,  E[m] = sum_p a[p] exp(i beta p' m'),  p' = p - (N-1)/2,  m' = m - (M-1)/2,
// beta = k s_max (2/N) pixel, is an exact re-association (Bluestein):  p' m' = (p'^2 + m'^2 - (m' - p')^2) / 2,
//     E[m] = v[m] * sum_p (a[p] w[p]) h[m - p],     w[p] = exp(i beta p'^2 / 2),  v[m] = exp(i beta m'^2 / 2),
//                                                   h[d] = exp(-i beta (d - (M - N)/2)^2 / 2),  d = m - p,
// i.e. a linear convolution of length N + M - 1, evaluated as a circular one of length L = 2^ceil(log2(N + M - 1)):
//     y = IFFT_L( FFT_L(a w, zero padded) * FFT_L(h, wrapped) ).
// FFT_L(h) / L is tabulated at plan time (fp64), so each 1-D transform costs two FFTs on the device.  Both chirps of the
// input side (w[p_x] w[p_y]) are folded into the static base pupil; the output chirps v have modulus 1 and only enter
// the optional field output.  Everything that is tabulated (chirps, twiddles, FFT of h) is evaluated in fp64 on the host.
//
//   czt_rows : CTA = RB pupil rows p_y of one (plane, component): pupil producer (base x exp(i kappa z)) straight into
//              shared memory, FFT, x H, inverse FFT, first M outputs -> T^T[m_x][p_y] (complex fp32 scratch).
//   czt_cols : CTA = RB output columns m_x of one plane; loops over the components: rows of T^T (contiguous in p_y),
//              FFT, x H, inverse FFT, |E|^2 accumulated over the components in registers; optional field store.
// FFT: Stockham autosort, radix 4 (one radix-2 pass first when log2 L is odd), ping-pong between two shared buffers,
// twiddles exp(-2 pi i k / L) from a table.
#include <cmath>
#include <complex>

#include "plan.hpp"
#include "pupil_gen.cuh"

namespace psf {

struct CztState {
  int L = 0, logL = 0, RB = 1, C = 0, zchunk = 1;
  void *d_base = nullptr;   // [C][N][N] float2: static pupil x w[p_x] w[p_y]
  void *d_kt = nullptr;     // [N][N] float2: kappa / 2 pi (hi, lo), turns per um
  void *d_tw = nullptr;     // [L] float2: exp(-2 pi i k / L)
  void *d_hf = nullptr;     // [L] float2: FFT_L(h) / L
  void *d_v = nullptr;      // [M] float2: output chirp v[m]
  void *d_T = nullptr;      // [zchunk][C][M][N] float2
  float weight[5] = {0, 0, 0, 0, 0};
  long long version = -1;
};

namespace {

constexpr int CZ_THREADS = 256;
constexpr int CZ_ELEMS = 8192;               // complex elements per shared buffer: RB * L (two buffers = 128 KB)
constexpr int CZ_SMEM = 2 * CZ_ELEMS * 8;

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// R independent length-L transforms stored back to back in `a`; result pointer returned (a or b).  INV: conjugate kernel.
template <bool INV>
__device__ float2 *fft_smem(float2 *a, float2 *b, int L, int logL, int R, const float2 *__restrict__ tw) {
  const int tid = threadIdx.x;
  int Ns = 1;
  if (logL & 1) {                               // one radix-2 pass
    const int half = L >> 1;
    for (int idx = tid; idx < R * half; idx += CZ_THREADS) {
      const int r = idx / half, j = idx - r * half;
      const float2 *in = a + r * L;
      float2 *out = b + r * L;
      const float2 v0 = in[j], v1 = in[j + half];
      out[2 * j] = cadd(v0, v1);                // Ns = 1: k = 0, twiddle 1
      out[2 * j + 1] = csub(v0, v1);
    }
    __syncthreads();
    float2 *t = a; a = b; b = t;
    Ns = 2;
  }
  const int quarter = L >> 2;
  for (; Ns < L; Ns <<= 2) {
    const int tstep = L / (Ns * 4);             // table stride of exp(-2 pi i k / (4 Ns))
    for (int idx = tid; idx < R * quarter; idx += CZ_THREADS) {
      const int r = idx / quarter, j = idx - r * quarter;
      const float2 *in = a + r * L;
      float2 *out = b + r * L;
      const int k = j & (Ns - 1);
      float2 v0 = in[j], v1 = in[j + quarter], v2 = in[j + 2 * quarter], v3 = in[j + 3 * quarter];
      if (k) {
        float2 w1 = __ldg(tw + k * tstep), w2 = __ldg(tw + 2 * k * tstep), w3 = __ldg(tw + 3 * k * tstep);
        if (INV) { w1.y = -w1.y; w2.y = -w2.y; w3.y = -w3.y; }
        v1 = cmul(v1, w1); v2 = cmul(v2, w2); v3 = cmul(v3, w3);
      }
      const float2 t0 = cadd(v0, v2), t1 = csub(v0, v2), t2 = cadd(v1, v3), d = csub(v1, v3);
      const float2 t3 = INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);   // (+-i) (v1 - v3)
      const int j0 = ((j - k) << 2) + k;        // (j / Ns) * 4 Ns + k
      out[j0] = cadd(t0, t2);
      out[j0 + Ns] = cadd(t1, t3);
      out[j0 + 2 * Ns] = csub(t0, t2);
      out[j0 + 3 * Ns] = csub(t1, t3);
    }
    __syncthreads();
    float2 *t = a; a = b; b = t;
  }
  return a;
}

// y = IFFT(FFT(x) * Hf) for the R transforms in `a`; returns the buffer holding y (unnormalised: Hf carries 1 / L)
__device__ float2 *convolve_smem(float2 *a, float2 *b, int L, int logL, int R, const float2 *__restrict__ tw, const float2 *__restrict__ hf) {
  float2 *f = fft_smem<false>(a, b, L, logL, R, tw);
  float2 *o = (f == a) ? b : a;
  for (int idx = threadIdx.x; idx < R * L; idx += CZ_THREADS) f[idx] = cmul(f[idx], __ldg(hf + (idx & (L - 1))));
  __syncthreads();
  return fft_smem<true>(f, o, L, logL, R, tw);
}

struct CzArgs {
  const float2 *base, *kt, *tw, *hf, *v;
  const float4 *planes;
  float2 *T;            // [zc][C][M][N]
  float *intensity;     // [Z][M][M]
  float2 *field;        // [C][Z][M][M] or nullptr
  int N, M, L, logL, RB, C, Z, z0;
  float weight[5];
};

__global__ void __launch_bounds__(CZ_THREADS) czt_rows(const CzArgs P) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  float2 *a = reinterpret_cast<float2 *>(smem_raw), *b = a + CZ_ELEMS;
  const int N = P.N, M = P.M, L = P.L, RB = P.RB;
  const int py0 = blockIdx.x * RB;
  const int zl = blockIdx.y / P.C, c = blockIdx.y - zl * P.C;
  const float4 pl = __ldg(P.planes + P.z0 + zl);
  // pupil producer: base x exp(i kappa z), zero outside the disc and in the padding
  for (int idx = threadIdx.x; idx < RB * L; idx += CZ_THREADS) {
    const int r = idx / L, px = idx - r * L, py = py0 + r;
    float2 val = make_float2(0.f, 0.f);
    if (px < N && py < N) {
      const size_t s = (size_t)py * N + px;
      const float2 bq = __ldg(P.base + (size_t)c * N * N + s);
      if (bq.x != 0.f || bq.y != 0.f) {
        float sn, cs;
        sincospif(2.0f * kz_turns(__ldg(P.kt + s), pl.x, pl.y), &sn, &cs);
        val = make_float2(bq.x * cs - bq.y * sn, bq.x * sn + bq.y * cs);
      }
    }
    a[idx] = val;
  }
  __syncthreads();
  const float2 *y = convolve_smem(a, b, L, P.logL, RB, P.tw, P.hf);
  float2 *Tt = P.T + ((size_t)zl * P.C + c) * (size_t)M * N;
  for (int idx = threadIdx.x; idx < RB * M; idx += CZ_THREADS) {
    const int r = idx % RB, mx = idx / RB, py = py0 + r;                  // r fastest: consecutive p_y of one m_x row
    if (py < N) Tt[(size_t)mx * N + py] = y[r * L + mx];
  }
}

template <bool FIELD>
__global__ void __launch_bounds__(CZ_THREADS) czt_cols(const CzArgs P) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  float2 *a = reinterpret_cast<float2 *>(smem_raw), *b = a + CZ_ELEMS;
  const int N = P.N, M = P.M, L = P.L, RB = P.RB;
  const int mx0 = blockIdx.x * RB, zl = blockIdx.y, z = P.z0 + zl;
  constexpr int PER = CZ_ELEMS / CZ_THREADS;    // RB * M <= RB * L = CZ_ELEMS output pixels per CTA
  float inten[PER];
#pragma unroll
  for (int k = 0; k < PER; ++k) inten[k] = 0.f;
  for (int c = 0; c < P.C; ++c) {
    const float2 *Tt = P.T + ((size_t)zl * P.C + c) * (size_t)M * N;
    __syncthreads();                            // the buffers of the previous component are free
    for (int idx = threadIdx.x; idx < RB * L; idx += CZ_THREADS) {
      const int r = idx / L, py = idx - r * L, mx = mx0 + r;
      a[idx] = (py < N && mx < M) ? __ldg(Tt + (size_t)mx * N + py) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const float2 *y = convolve_smem(a, b, L, P.logL, RB, P.tw, P.hf);
    const float w = P.weight[c];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
      const int idx = threadIdx.x + k * CZ_THREADS;
      const int r = idx % RB, my = idx / RB;                               // r fastest: consecutive m_x of one image row
      if (my < M && mx0 + r < M) {
        const float2 e = y[r * L + my];
        inten[k] = fmaf(w, e.x * e.x + e.y * e.y, inten[k]);
        if (FIELD) {
          const float2 ph = cmul(__ldg(P.v + my), __ldg(P.v + mx0 + r));  // output chirps v[m_y] v[m_x]
          P.field[((size_t)c * P.Z + z) * (size_t)M * M + (size_t)my * M + mx0 + r] = cmul(e, ph);
        }
      }
    }
  }
  float *Ib = P.intensity + (size_t)z * M * M;
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const int idx = threadIdx.x + k * CZ_THREADS;
    const int r = idx % RB, my = idx / RB;
    if (my < M && mx0 + r < M) Ib[(size_t)my * M + mx0 + r] = inten[k];
  }
}

// host-side reference FFT (fp64, recursive radix 2) for the plan-time transform of the chirp h
void fft_host(std::vector<std::complex<double>> &x) {
  const size_t n = x.size();
  if (n <= 1) return;
  std::vector<std::complex<double>> e(n / 2), o(n / 2);
  for (size_t i = 0; i < n / 2; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
  fft_host(e);
  fft_host(o);
  const double twopi = 6.283185307179586476925287;
  for (size_t k = 0; k < n / 2; ++k) {
    const std::complex<double> t = std::polar(1.0, -twopi * (double)k / (double)n) * o[k];
    x[k] = e[k] + t;
    x[k + n / 2] = e[k] - t;
  }
}

template <typename T>
bool up(void **d, const std::vector<T> &h, long long *acc) {
  if (*d) { cudaFree(*d); *d = nullptr; }
  if (cudaMalloc(d, h.size() * sizeof(T)) != cudaSuccess) return false;
  if (cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
  if (acc) *acc += (long long)(h.size() * sizeof(T));
  return true;
}

}  // namespace

bool czt_supported(const psf_plan *p, std::string &why) {
  const long long need = (long long)p->dp.N + p->dp.M - 1;
  if (need > CZ_ELEMS) { why = "PSF_PREC_CZT_FFT: N + M - 1 must be <= 8192 (one transform per shared-memory buffer)"; return false; }
  if (p->dp.per_plane) { why = "PSF_PREC_CZT_FFT supports the static mode only (shared Zernike terms, no per-plane rows or shifts)"; return false; }
  return true;
}

void czt_free(psf_plan *p) {
  CztState *t = p->czt;
  if (!t) return;
  void *bufs[] = {t->d_base, t->d_kt, t->d_tw, t->d_hf, t->d_v, t->d_T};
  for (void *b : bufs)
    if (b) cudaFree(b);
  delete t;
  p->czt = nullptr;
}

// (Re)builds the chirp-Z tables from the plan's static pupil p->h_base (which already holds the shared Zernike term).
psf_status czt_setup(psf_plan *p) {
  const psf_plan_desc &d = p->desc;
  const DevPlan &D = p->dp;
  const HostPupil &hp = p->hp0;
  const bool fresh = p->czt == nullptr;
  if (fresh) p->czt = new CztState();
  CztState *t = p->czt;
  auto fail = [&](const char *msg, psf_status s) { p->err = msg; return s; };
  const int N = D.N, M = D.M, C = hp.C;
  const size_t NN = (size_t)N * N;
  int L = 1, logL = 0;
  while (L < N + M - 1) { L <<= 1; ++logL; }
  if (L < 4) { L = 4; logL = 2; }
  t->L = L; t->logL = logL; t->C = C;
  t->RB = CZ_ELEMS / L;
  for (int c = 0; c < 5; ++c) t->weight[c] = (float)hp.weight[c];
  const double twopi = 6.283185307179586476925287;
  const double beta = twopi * d.NA / d.wavelength_um * (2.0 / N) * d.pixel_um;      // k s_max (2 / N) pixel
  const double p0 = 0.5 * (N - 1), m0 = 0.5 * (M - 1);
  std::vector<std::complex<double>> w(N);
  for (int q = 0; q < N; ++q) w[q] = std::polar(1.0, 0.5 * beta * (q - p0) * (q - p0));
  // static pupil x input chirps, and kappa in turns (hi, lo)
  std::vector<float2> base((size_t)C * NN), kt(NN);
#pragma omp parallel for schedule(static)
  for (int py = 0; py < N; ++py)
    for (int px = 0; px < N; ++px) {
      const size_t s = (size_t)py * N + px;
      const double kap = hp.kappa[s] / twopi;
      const float hi = (float)kap;
      kt[s] = make_float2(hi, (float)(kap - (double)hi));
      for (int c = 0; c < C; ++c) {
        const std::complex<double> v = p->h_base[(size_t)c * NN + s] * w[px] * w[py];
        base[(size_t)c * NN + s] = make_float2((float)v.real(), (float)v.imag());
      }
    }
  if (!up(&t->d_base, base, &p->upload_bytes) || !up(&t->d_kt, kt, &p->upload_bytes)) return fail("czt: table upload failed", PSF_ERR_ALLOC);
  t->version = p->table_version;
  if (!fresh) return PSF_OK;

  std::vector<float2> tw(L), hf(L), v(M);
  for (int k = 0; k < L; ++k) {
    const double a = -twopi * (double)k / (double)L;
    tw[k] = make_float2((float)std::cos(a), (float)std::sin(a));
  }
  std::vector<std::complex<double>> h(L, std::complex<double>(0.0, 0.0));
  const double delta = m0 - p0;
  for (int dd = -(N - 1); dd <= M - 1; ++dd) {
    const double x = (double)dd - delta;
    h[(size_t)((dd + L) % L)] = std::polar(1.0, -0.5 * beta * x * x);
  }
  fft_host(h);
  for (int k = 0; k < L; ++k) hf[k] = make_float2((float)(h[k].real() / L), (float)(h[k].imag() / L));
  for (int m = 0; m < M; ++m) {
    const std::complex<double> e = std::polar(1.0, 0.5 * beta * (m - m0) * (m - m0));
    v[m] = make_float2((float)e.real(), (float)e.imag());
  }
  if (!up(&t->d_tw, tw, &p->upload_bytes) || !up(&t->d_hf, hf, &p->upload_bytes) || !up(&t->d_v, v, &p->upload_bytes))
    return fail("czt: table upload failed", PSF_ERR_ALLOC);
  // scratch T^T [zchunk][C][M][N] complex fp32, at most 2 GB
  const size_t per_plane = (size_t)C * M * N * sizeof(float2);
  size_t zc = ((size_t)2 << 30) / per_plane;
  if (zc < 1) zc = 1;
  if (zc > (size_t)D.Z) zc = D.Z;
  if (zc > 65535 / (size_t)C) zc = 65535 / (size_t)C;          // gridDim.y of czt_rows
  t->zchunk = (int)zc;
  if (cudaMalloc(&t->d_T, zc * per_plane) != cudaSuccess) return fail("czt: cudaMalloc of the scratch failed", PSF_ERR_ALLOC);
  if (cudaFuncSetAttribute(czt_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, CZ_SMEM) != cudaSuccess ||
      cudaFuncSetAttribute(czt_cols<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CZ_SMEM) != cudaSuccess ||
      cudaFuncSetAttribute(czt_cols<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CZ_SMEM) != cudaSuccess)
    return fail("czt: cudaFuncSetAttribute failed", PSF_ERR_CUDA);
  return PSF_OK;
}

int czt_launches(const psf_plan *p) { return 2 * ((p->dp.Z + p->czt->zchunk - 1) / p->czt->zchunk); }

cudaError_t launch_czt(const psf_plan *p, cudaStream_t st, float *intensity, float2 *field) {
  const DevPlan &D = p->dp;
  const CztState *t = p->czt;
  CzArgs a;
  a.base = (const float2 *)t->d_base; a.kt = (const float2 *)t->d_kt; a.tw = (const float2 *)t->d_tw;
  a.hf = (const float2 *)t->d_hf; a.v = (const float2 *)t->d_v; a.planes = D.planes; a.T = (float2 *)t->d_T;
  a.intensity = intensity; a.field = field;
  a.N = D.N; a.M = D.M; a.L = t->L; a.logL = t->logL; a.RB = t->RB; a.C = t->C; a.Z = D.Z;
  for (int c = 0; c < 5; ++c) a.weight[c] = t->weight[c];
  for (int z0 = 0; z0 < D.Z; z0 += t->zchunk) {
    const int zc = (D.Z - z0 < t->zchunk) ? (D.Z - z0) : t->zchunk;
    a.z0 = z0;
    czt_rows<<<dim3((D.N + t->RB - 1) / t->RB, zc * t->C), CZ_THREADS, CZ_SMEM, st>>>(a);
    prof_mark(p, st, 0);
    const dim3 g2((D.M + t->RB - 1) / t->RB, zc);
    if (field) czt_cols<true><<<g2, CZ_THREADS, CZ_SMEM, st>>>(a);
    else czt_cols<false><<<g2, CZ_THREADS, CZ_SMEM, st>>>(a);
    prof_mark(p, st, 1);
  }
  return cudaGetLastError();
}

}  // namespace psf
