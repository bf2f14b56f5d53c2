// C-ABI implementation (include/psf.h): validation, plan-time table upload, launch sequencing.
#include <cmath>
#include <cstring>
#include <new>

#include "plan.hpp"

using namespace psf;

namespace {

thread_local std::string g_create_err = "";

const size_t kScratchBudget = (size_t)48 << 20;   // T scratch ring: small enough to live in the 126 MB L2

#define CU_TRY(p, call)                                                                         \
  do {                                                                                          \
    cudaError_t e_ = (call);                                                                    \
    if (e_ != cudaSuccess) {                                                                    \
      (p)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                            \
      return PSF_ERR_CUDA;                                                                      \
    }                                                                                           \
  } while (0)

void set_err(psf_plan *p, const char *msg) noexcept {
  try { if (p) p->err = msg; else g_create_err = msg; } catch (...) {}
}

// Every extern "C" body runs inside this guard: nothing throws across the ABI (psf.h).
template <typename F>
psf_status guarded(psf_plan *p, F &&body) noexcept {
  try {
    return body();
  } catch (const std::bad_alloc &) {
    set_err(p, "out of host memory");
    return PSF_ERR_ALLOC;
  } catch (const std::exception &e) {
    set_err(p, e.what());
    return PSF_ERR_CUDA;
  } catch (...) {
    set_err(p, "unknown C++ exception");
    return PSF_ERR_CUDA;
  }
}

// Tables on the device may still be read by launches of an earlier compute call on the caller's stream (any stream:
// a non-blocking stream does not serialise with the copies below).  Every compute call records `done_ev` behind its
// last launch; whoever is about to overwrite or free a table waits for it first.
cudaError_t wait_inflight(psf_plan *p) { return p->done_ev ? cudaEventSynchronize(p->done_ev) : cudaSuccess; }
void mark_inflight(psf_plan *p, cudaStream_t st) { if (p->done_ev) cudaEventRecord(p->done_ev, st); }

template <typename T>
psf_status upload(psf_plan *p, void **dptr, size_t *cap, const std::vector<T> &h) {
  const size_t bytes = h.size() * sizeof(T);
  if (bytes == 0) return PSF_OK;
  if (bytes > *cap) {
    if (*dptr) { cudaFree(*dptr); *dptr = nullptr; *cap = 0; }
    cudaError_t e = cudaMalloc(dptr, bytes);
    if (e != cudaSuccess) { p->err = std::string("cudaMalloc: ") + cudaGetErrorString(e); *dptr = nullptr; return PSF_ERR_ALLOC; }
    *cap = bytes;
  }
  CU_TRY(p, cudaMemcpy(*dptr, h.data(), bytes, cudaMemcpyHostToDevice));
  p->upload_bytes += (long long)bytes;
  return PSF_OK;
}

// (hi, lo) float pair of a double
inline void split2(double v, float &hi, float &lo) { hi = (float)v; lo = (float)(v - (double)hi); }

// Device copies of the folded base pupil and kappa table of the FFMA kernels, from the plan's host copies.
psf_status upload_ffma_tables(psf_plan *p) {
  psf_status s;
  if ((s = upload(p, &p->d_bfold, &p->cap_bfold, p->h_bfold)) != PSF_OK) return s;
  if ((s = upload(p, &p->d_kt, &p->cap_kt, p->h_kt)) != PSF_OK) return s;
  p->dp.bfold = (const float4 *)p->d_bfold;
  p->dp.kt = (const float2 *)p->d_kt;
  return PSF_OK;
}

// Plane table: defocus (hi, lo) and the tilt of the lateral shift, per plane / emitter.
psf_status upload_planes(psf_plan *p) {
  const psf_plan_desc &d = p->desc;
  DevPlan &P = p->dp;
  std::vector<float4> planes(d.n_planes);
  const double tscale = d.NA / d.wavelength_um;   // k s_max / 2 pi
  P.has_shift = p->shifts.empty() ? 0 : 1;
  for (int b = 0; b < d.n_planes; ++b) {
    float zh, zl;
    split2(p->z[b], zh, zl);
    float tx = 0.f, ty = 0.f;
    if (P.has_shift) { tx = (float)(tscale * (double)p->shifts[2 * b]); ty = (float)(tscale * (double)p->shifts[2 * b + 1]); }
    planes[b] = make_float4(zh, zl, tx, ty);
  }
  psf_status s = upload(p, &p->d_planes, &p->cap_planes, planes);
  if (s != PSF_OK) return s;
  P.planes = (const float4 *)p->d_planes;
  return PSF_OK;
}

// Per-plane Zernike rows: as given (the tiled FFMA kernels, the adjoint) and in the parity-sorted term order p->zorder
// (k_small, k_smlm).
psf_status upload_coef_rows(psf_plan *p) {
  const int K = p->K_rows, Z = p->desc.n_planes;
  std::vector<float> coefq(p->zern_rows.size(), 0.f);
  for (int k = 0; k < K; ++k) {
    const int j = p->zorder[k];
    for (int b = 0; b < Z; ++b) coefq[(size_t)b * K + k] = p->zern_rows[(size_t)b * K + j];
  }
  psf_status s;
  if ((s = upload(p, &p->d_coef, &p->cap_coef, p->zern_rows)) != PSF_OK) return s;
  if ((s = upload(p, &p->d_coefq, &p->cap_coefq, coefq)) != PSF_OK) return s;
  p->dp.coef = (const float *)p->d_coef;
  p->dp.coefq = (const float *)p->d_coefq;
  return PSF_OK;
}

// Folds the static pupil about both axes into the four parity classes and uploads every static table.
psf_status upload_static(psf_plan *p) {
  const psf_plan_desc &d = p->desc;
  const HostPupil &hp = p->hp0;
  const int Kneed = p->zern_shared.empty() ? p->K_rows : (int)p->zern_shared.size();
  if (Kneed > 0 && (p->zb_first != p->noll_first || p->zb_K != Kneed)) {
    build_zernike_basis(hp, p->noll_first, Kneed, p->zbasis);
    p->zb_first = p->noll_first;
    p->zb_K = Kneed;
  }
  PhaseTimer tm;
  std::vector<cplx> &base_z = p->h_base;
  apply_shared_zernike(hp, p->zern_shared.empty() ? nullptr : p->zern_shared.data(), (int)p->zern_shared.size(), p->zbasis,
                       p->phase_mask.empty() ? nullptr : p->phase_mask.data(), base_z);
  p->host_base_stale = false;
  const int N = d.pupil_n, n = (N + 1) / 2, C = hp.C;
  const size_t NN = (size_t)N * N, nn = (size_t)n * n;
  DevPlan &P = p->dp;
  P.C = C;
  for (int c = 0; c < 5; ++c) P.weight[c] = (float)hp.weight[c];

  tm.mark("apply_shared_zernike");
  if (d.precision == PSF_PREC_CZT_FFT) {          // chirp-Z path: unfolded pupil with the input chirps folded in, plane table
    std::string why;
    if (!czt_supported(p, why)) { p->err = why; return PSF_ERR_UNSUPPORTED; }
    std::vector<float4> planes(d.n_planes);
    for (int b = 0; b < d.n_planes; ++b) {
      float zh, zl;
      split2(p->z[b], zh, zl);
      planes[b] = make_float4(zh, zl, 0.f, 0.f);
    }
    psf_status sc;
    if ((sc = upload(p, &p->d_planes, &p->cap_planes, planes)) != PSF_OK) return sc;
    P.planes = (const float4 *)p->d_planes;
    p->path = 4;
    return czt_setup(p);
  }
  std::vector<float4> &bfold = p->h_bfold;
  std::vector<float2> &kt = p->h_kt;
  bfold.resize((size_t)C * nn * 2);
  kt.resize(nn);
  const double twopi = 6.283185307179586476925287;
#pragma omp parallel for schedule(static)
  for (int qy = 0; qy < n; ++qy) {
    for (int qx = 0; qx < n; ++qx) {
      const int ry = N - 1 - qy, rx = N - 1 - qx;
      const bool sy = ry == qy, sx = rx == qx;
      float hi, lo;
      split2(hp.kappa[(size_t)qy * N + qx] / twopi, hi, lo);
      kt[(size_t)qy * n + qx] = make_float2(hi, lo);
      for (int c = 0; c < C; ++c) {
        const cplx *B = base_z.data() + (size_t)c * NN;
        const cplx p00 = B[(size_t)qy * N + qx];
        const cplx p01 = sx ? cplx(0, 0) : B[(size_t)qy * N + rx];
        const cplx p10 = sy ? cplx(0, 0) : B[(size_t)ry * N + qx];
        const cplx p11 = (sx || sy) ? cplx(0, 0) : B[(size_t)ry * N + rx];
        const cplx e0 = p00 + p01, o0 = sx ? cplx(0, 0) : p00 - p01;     // row qy:      even / odd in x
        const cplx e1 = p10 + p11, o1 = sx ? cplx(0, 0) : p10 - p11;     // mirror row
        const cplx ee = e0 + e1, eo = o0 + o1;
        const cplx oe = sy ? cplx(0, 0) : e0 - e1, oo = sy ? cplx(0, 0) : o0 - o1;
        float4 *o = &bfold[((size_t)c * nn + (size_t)qy * n + qx) * 2];
        o[0] = make_float4((float)ee.real(), (float)ee.imag(), (float)eo.real(), (float)eo.imag());
        o[1] = make_float4((float)oe.real(), (float)oe.imag(), (float)oo.real(), (float)oo.imag());
      }
    }
  }
  tm.mark("fold");
  psf_status s;
  // The folded tables feed the FFMA kernels only; a plan on the tensor path (whose stage-2 epilogue also writes the field
  // output) never reads them: no upload (10 MB at N = 512).
  const bool tensor_path = d.precision != PSF_PREC_FP32 && !P.per_plane &&
                           (d.precision == PSF_PREC_3XTF32 || d.precision == PSF_PREC_3XF16 || tc_eligible(p));
  if (!tensor_path && (s = upload_ffma_tables(p)) != PSF_OK) return s;
  tm.mark("upload bfold, kt");

  if (P.per_plane) {
    std::vector<float2> bunf((size_t)C * NN);
    for (size_t i = 0; i < bunf.size(); ++i) bunf[i] = make_float2((float)base_z[i].real(), (float)base_z[i].imag());
    if ((s = upload(p, &p->d_bunf, &p->cap_bunf, bunf)) != PSF_OK) return s;
    P.bunf = (const float2 *)p->d_bunf;
    const int K = p->K_rows;
    std::vector<float> zb((size_t)K * NN, 0.f);
    for (size_t i = 0; i < zb.size(); ++i) zb[i] = (float)(p->zbasis[i] / twopi);
    if ((s = upload(p, &p->d_zb, &p->cap_zb, zb)) != PSF_OK) return s;
    P.zb = (const float *)p->d_zb;
    P.K = K;
    // folded, parity-sorted copy for the fused small-grid kernel: Z_j(-x, y) = +-Z_j(x, y), Z_j(x, -y) = +-Z_j(x, y)
    //   m = 0: even/even;  cos(m phi): even in y, odd in x iff m odd;  sin(m phi): odd in y, odd in x iff m even
    std::vector<int> order;
    for (int i = 0; i < 4; ++i) P.zcnt[i] = 0;
    for (int cls = 0; cls < 4; ++cls)
      for (int j = 0; j < K; ++j) {
        int zn, zm, kind;
        noll_to_nm(p->noll_first + j, zn, zm, kind);
        const int xo = (kind == 0) ? 0 : (kind == 1 ? (zm & 1) : ((zm + 1) & 1));
        const int yo = (kind == 2) ? 1 : 0;
        if (xo + 2 * yo == cls) { order.push_back(j); P.zcnt[cls]++; }
      }
    p->zorder = order;
    std::vector<float> zbq((size_t)K * nn, 0.f);
    for (int k = 0; k < K; ++k) {
      const int j = order[k];
      for (int qy = 0; qy < n; ++qy)
        for (int qx = 0; qx < n; ++qx) zbq[(size_t)k * nn + (size_t)qy * n + qx] = (float)(p->zbasis[(size_t)j * NN + (size_t)qy * N + qx] / twopi);
    }
    if ((s = upload(p, &p->d_zbq, &p->cap_zbq, zbq)) != PSF_OK) return s;
    if ((s = upload_coef_rows(p)) != PSF_OK) return s;
    P.zbq = (const float *)p->d_zbq;
    // the emitter-batch kernel for small grids (falls back to k_small when the plan does not qualify)
    smlm_free(p);
    if (p->tune_smlm && small_eligible(p) && d.precision != PSF_PREC_CZT_FFT && (s = smlm_setup(p, zbq)) != PSF_OK) return s;
  } else {
    P.K = 0;
    for (int i = 0; i < 4; ++i) P.zcnt[i] = 0;
    smlm_free(p);
  }
  if ((s = upload_planes(p)) != PSF_OK) return s;
  // path: tensor cores for the static (shared-pupil) mode when asked for or when the problem is large enough
  const psf_precision prec = d.precision;
  const bool want_tc = prec != PSF_PREC_FP32 && !P.per_plane && (prec == PSF_PREC_3XTF32 || prec == PSF_PREC_3XF16 || tc_eligible(p));
  p->path = want_tc ? (prec == PSF_PREC_3XTF32 ? 1 : 2) : 0;     // AUTO: the fp16 split (same accuracy, about twice as fast)
  if (!want_tc && small_eligible(p)) p->path = 3;                // whole path fused in one CTA per plane
  tm.mark("planes, path");
  if (want_tc && (s = tc_setup(p, bfold, kt, p->phi, p->path == 2)) != PSF_OK) return s;
  tm.mark("tc_setup");
  return PSF_OK;
}

psf_status upload_dft(psf_plan *p) {
  const std::vector<double> &phi = p->phi;
  std::vector<float> c(phi.size()), s(phi.size());
  for (size_t i = 0; i < phi.size(); ++i) { c[i] = (float)std::cos(phi[i]); s[i] = (float)std::sin(phi[i]); }
  psf_status st;
  if ((st = upload(p, &p->d_cos, &p->cap_cos, c)) != PSF_OK) return st;
  if ((st = upload(p, &p->d_sin, &p->cap_sin, s)) != PSF_OK) return st;
  p->dp.cosT = (const float *)p->d_cos;
  p->dp.sinT = (const float *)p->d_sin;
  return PSF_OK;
}

psf_status alloc_scratch(psf_plan *p) {
  const DevPlan &P = p->dp;
  if (p->path == 4) return PSF_OK;              // the chirp-Z path owns its scratch
  const size_t per_plane = (size_t)P.C * 8 * P.n * P.m * sizeof(float);
  size_t zc = kScratchBudget / per_plane;
  if (zc < 1) zc = 1;
  if (zc > (size_t)P.Z) zc = P.Z;
  if (zc > 65535 / (size_t)P.C) zc = 65535 / P.C;       // gridDim.z limit of the stage-1 launch
  p->zchunk = (int)zc;
  const size_t need = zc * per_plane;
  if (need > p->T_bytes) {
    if (p->d_T) { cudaFree(p->d_T); p->d_T = nullptr; p->T_bytes = 0; }
    cudaError_t e = cudaMalloc(&p->d_T, need);
    if (e != cudaSuccess) { p->err = std::string("cudaMalloc(T scratch): ") + cudaGetErrorString(e); return PSF_ERR_ALLOC; }
    p->T_bytes = need;
  }
  return PSF_OK;
}

// cudaMemcpy from pageable host memory returns once the data is staged; the DMA to the device may still be in flight, ordered
// only against the legacy stream and blocking streams.  The caller's stream may be non-blocking, so every call that uploads
// tables ends with this fence.
psf_status uploads_fence(psf_plan *p) {
  if (cudaStreamSynchronize(cudaStreamLegacy) != cudaSuccess) { p->err = "cudaStreamSynchronize after the table uploads failed"; return PSF_ERR_CUDA; }
  return PSF_OK;
}

psf_status refresh(psf_plan *p) {
  if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
  if (tc_fused_aborted(p)) {
    p->err = "an earlier psf_compute of this plan (fused launch) gave up waiting for a stage-1 / stage-2 dependency: its stack is invalid";
    return PSF_ERR_CUDA;
  }
  p->upload_bytes = 0;
  ++p->table_version;
  ++p->static_version;
  psf_status s = upload_static(p);
  if (s != PSF_OK) return s;
  if ((s = alloc_scratch(p)) != PSF_OK) return s;     // C is fixed per plan, but keep the scratch consistent with it
  return uploads_fence(p);
}

// A change of the shared pupil phase only (shared Zernike coefficients, phase mask) on a plan whose tables are already in place:
// plans on the 3xFP16 pair kernels redo the phase, the fold and the operand scales on the device (tc_refresh_device, ~0.1 ms
// instead of 2.5 ms of host work and an 11 MB upload at config 5); every other plan takes the host path.
psf_status refresh_phase(psf_plan *p) {
  if (!p->tune_dev_refresh || !tc_refresh_device_ok(p) || p->desc.precision == PSF_PREC_CZT_FFT) return refresh(p);
  if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
  if (tc_fused_aborted(p)) {
    p->err = "an earlier psf_compute of this plan (fused launch) gave up waiting for a stage-1 / stage-2 dependency: its stack is invalid";
    return PSF_ERR_CUDA;
  }
  const int Kneed = (int)p->zern_shared.size();
  if (Kneed > 0 && (p->zb_first != p->noll_first || p->zb_K != Kneed)) {
    build_zernike_basis(p->hp0, p->noll_first, Kneed, p->zbasis);
    p->zb_first = p->noll_first;
    p->zb_K = Kneed;
  }
  p->upload_bytes = 0;
  ++p->table_version;
  p->host_base_stale = true;
  return tc_refresh_device(p);
}

void free_all(psf_plan *p) {
  void **bufs[] = {&p->d_bfold, &p->d_kt, &p->d_bunf, &p->d_zb, &p->d_coef, &p->d_planes, &p->d_cos, &p->d_sin, &p->d_T,
                   &p->d_zbq, &p->d_coefq};
  for (void **b : bufs)
    if (*b) { cudaFree(*b); *b = nullptr; }
  for (cudaEvent_t e : p->prof_ev) cudaEventDestroy(e);
  p->prof_ev.clear();
  if (p->done_ev) { cudaEventDestroy(p->done_ev); p->done_ev = nullptr; }
  tc_free(p);
  czt_free(p);
  smlm_free(p);
  bessel_free(p);
  grad_free(p);
}

}  // namespace

namespace psf {
// for entry points without a plan in other files (noalloc.cu): the message psf_last_error(NULL) returns on this thread
void set_thread_error(const char *msg) noexcept { set_err(nullptr, msg); }

const std::vector<cplx> &host_base(psf_plan *p) {
  if (p->host_base_stale) {
    apply_shared_zernike(p->hp0, p->zern_shared.empty() ? nullptr : p->zern_shared.data(), (int)p->zern_shared.size(), p->zbasis,
                         p->phase_mask.empty() ? nullptr : p->phase_mask.data(), p->h_base);
    p->host_base_stale = false;      // h_bfold stays behind: only upload_static reads it, right after rebuilding it
  }
  return p->h_base;
}
psf_status plan_set_materialised(psf_plan *p, double qmax, double rmax) {
  p->mat_mode = 1;
  p->mat_qmax = qmax;
  p->mat_rmax = rmax;
  if (cudaSetDevice(p->device) != cudaSuccess) { p->err = "cudaSetDevice failed"; return PSF_ERR_CUDA; }
  tc_free(p);
  return refresh(p);
}
}  // namespace psf

extern "C" {

psf_status psf_plan_create(const psf_plan_desc *desc, psf_plan **out) {
  psf_plan *p = nullptr;
  try {
  if (out) *out = nullptr;
  if (!out) { g_create_err = "out is NULL"; return PSF_ERR_INVALID_ARG; }
  std::string err;
  psf_status s = validate_desc(desc, err);
  if (s != PSF_OK) { g_create_err = err; return s; }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    g_create_err = std::string("no CUDA device: ") + cudaGetErrorString(e) + " (libpsf_b200 has no CPU fallback)";
    return PSF_ERR_CUDA;
  }
  if (desc->device < 0 || desc->device >= ndev) { g_create_err = "device ordinal out of range"; return PSF_ERR_INVALID_ARG; }
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, desc->device)) != cudaSuccess) {
    g_create_err = std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e);
    return PSF_ERR_CUDA;
  }
  if (prop.major != 10) {
    g_create_err = "device is not sm_100 (compute capability 10.x): this library is built for B200 only";
    return PSF_ERR_UNSUPPORTED;
  }
  p = new (std::nothrow) psf_plan();
  if (!p) { g_create_err = "out of host memory"; return PSF_ERR_ALLOC; }
  p->desc = *desc;
  p->z.assign(desc->z_um, desc->z_um + desc->n_planes);
  p->desc.z_um = p->z.data();
  if (std::isnan(p->desc.n_immersion_design)) p->desc.n_immersion_design = desc->n_immersion;
  p->device = desc->device;
  p->sm_count = prop.multiProcessorCount;
  DevPlan &P = p->dp;
  P.N = desc->pupil_n; P.M = desc->out_m; P.n = (P.N + 1) / 2; P.m = (P.M + 1) / 2; P.Z = desc->n_planes;
  P.per_plane = 0; P.K = 0; P.has_shift = 0;
  if ((e = cudaSetDevice(p->device)) != cudaSuccess || (e = cudaEventCreateWithFlags(&p->done_ev, cudaEventDisableTiming)) != cudaSuccess ||
      (e = small_setup()) != cudaSuccess) {
    g_create_err = std::string("plan set-up (device, event, function attributes): ") + cudaGetErrorString(e);
    free_all(p);
    delete p;
    return PSF_ERR_CUDA;
  }
  p->path = 0;
  build_host_pupil(p->desc, nullptr, 1, 0, p->hp0);
  const bool czt = p->desc.precision == PSF_PREC_CZT_FFT;
  if (!czt) build_dft_phase(p->desc, p->phi);
  if ((s = refresh(p)) != PSF_OK || (!czt && (s = upload_dft(p)) != PSF_OK) || (s = uploads_fence(p)) != PSF_OK) {
    g_create_err = p->err;
    free_all(p);
    delete p;
    return s;
  }
  *out = p;
  return PSF_OK;
  } catch (...) {                       // std::bad_alloc from the host tables, or anything else: never across the ABI
    if (p) { try { free_all(p); } catch (...) {} delete p; }
    if (out) *out = nullptr;
    set_err(nullptr, "out of host memory (or another C++ exception) while building the plan");
    return PSF_ERR_ALLOC;
  }
}

psf_status psf_set_zernike(psf_plan *p, const float *coeffs, int noll_first, int n_coeffs, int per_plane) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (n_coeffs < 0) { p->err = "n_coeffs < 0"; return PSF_ERR_INVALID_ARG; }
  if (n_coeffs > 0 && coeffs && noll_first < 1) { p->err = "noll_first must be >= 1"; return PSF_ERR_INVALID_ARG; }
  if (n_coeffs > 64) { p->err = "at most 64 Zernike terms"; return PSF_ERR_INVALID_ARG; }
  const size_t cnt = (size_t)n_coeffs * (per_plane ? p->dp.Z : 1);
  if (coeffs)
    for (size_t i = 0; i < cnt; ++i)
      if (!std::isfinite(coeffs[i])) { p->err = "non-finite Zernike coefficient"; return PSF_ERR_INVALID_ARG; }
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  // new per-plane rows for the terms already set: only the two coefficient tables change (no table refresh, derived state stands)
  if (per_plane && coeffs && n_coeffs > 0 && p->dp.per_plane && p->K_rows == n_coeffs && p->noll_first == noll_first &&
      p->zern_shared.empty() && (int)p->zorder.size() == n_coeffs && (p->path == 0 || p->path == 3)) {
    if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
    p->zern_rows.assign(coeffs, coeffs + cnt);
    p->upload_bytes = 0;
    psf_status s = upload_coef_rows(p);
    return s != PSF_OK ? s : uploads_fence(p);
  }
  p->zern_shared.clear();
  p->zern_rows.clear();
  p->K_rows = 0;
  if (coeffs && n_coeffs > 0) {
    p->noll_first = noll_first;
    if (per_plane) { p->zern_rows.assign(coeffs, coeffs + cnt); p->K_rows = n_coeffs; }
    else p->zern_shared.assign(coeffs, coeffs + n_coeffs);
  }
  const int was_per_plane = p->dp.per_plane;
  p->dp.per_plane = (p->K_rows > 0 || !p->shifts.empty()) ? 1 : 0;
  return (was_per_plane || p->dp.per_plane) ? refresh(p) : refresh_phase(p);
  });
}

psf_status psf_set_phase_mask(psf_plan *p, const float *w0_rad) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  const size_t NN = (size_t)p->desc.pupil_n * p->desc.pupil_n;
  if (w0_rad)
    for (size_t i = 0; i < NN; ++i)
      if (!std::isfinite(w0_rad[i])) { p->err = "non-finite phase-mask value"; return PSF_ERR_INVALID_ARG; }
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  p->phase_mask.clear();
  if (w0_rad) p->phase_mask.assign(w0_rad, w0_rad + NN);
  ++p->phase_mask_version;
  return refresh_phase(p);
  });
}

psf_status psf_set_shifts(psf_plan *p, const float *xy_um) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (xy_um)
    for (int i = 0; i < 2 * p->dp.Z; ++i)
      if (!std::isfinite(xy_um[i])) { p->err = "non-finite shift"; return PSF_ERR_INVALID_ARG; }
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  // new shifts where shifts are already set: only the plane table changes
  if (xy_um && !p->shifts.empty() && p->dp.per_plane && (p->path == 0 || p->path == 3)) {
    if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
    p->shifts.assign(xy_um, xy_um + 2 * (size_t)p->dp.Z);
    p->upload_bytes = 0;
    psf_status s = upload_planes(p);
    return s != PSF_OK ? s : uploads_fence(p);
  }
  p->shifts.clear();
  if (xy_um) p->shifts.assign(xy_um, xy_um + 2 * (size_t)p->dp.Z);
  p->dp.per_plane = (p->K_rows > 0 || !p->shifts.empty()) ? 1 : 0;
  return refresh(p);
  });
}

psf_status psf_compute(psf_plan *p, void *cuda_stream, float *intensity, void *field) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (!intensity) { p->err = "intensity is NULL"; return PSF_ERR_INVALID_ARG; }
  if (((uintptr_t)intensity & 15) || ((uintptr_t)field & 15)) { p->err = "output pointers must be 16-byte aligned"; return PSF_ERR_INVALID_ARG; }
  if (field && p->desc.pol == PSF_POL_UNPOLARIZED && p->desc.model == PSF_MODEL_VECTORIAL) {
    p->err = "field output is undefined for PSF_POL_UNPOLARIZED (two incoherent fields)";
    return PSF_ERR_UNSUPPORTED;
  }
  if (cudaSetDevice(p->device) != cudaSuccess) { p->err = "cudaSetDevice failed"; return PSF_ERR_CUDA; }
  if (p->prof) {
    p->prof_n = 0;
    p->prof_valid = true;
    cudaEventRecord(p->prof_ev[0], (cudaStream_t)cuda_stream);
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool tc = p->path == 1 || p->path == 2;
  cudaError_t e = tc ? launch_tc(p, st, intensity, (float2 *)field)
                     : p->path == 4 ? launch_czt(p, st, intensity, (float2 *)field)
                     : (p->path == 3 && p->smlm && !field) ? launch_smlm(p, st, intensity)
                     : p->path == 3 ? launch_small(p, st, intensity, (float2 *)field)
                                    : launch_ffma(p, st, intensity, (float2 *)field);
  mark_inflight(p, st);
  if (e != cudaSuccess) { p->err = std::string("kernel launch: ") + cudaGetErrorString(e); return PSF_ERR_CUDA; }
  return PSF_OK;
  });
}

// ---- spherical (Bessel) parametrisation: axisymmetric pupils only ---------------------------------------------------
static bool axisymmetric(psf_plan *p) {
  if (!p->zern_shared.empty() || p->K_rows > 0 || !p->shifts.empty() || !p->phase_mask.empty()) {
    p->err = "the spherical parametrisation needs an axisymmetric pupil: clear Zernike terms, shifts and the phase mask";
    return false;
  }
  return true;
}

psf_status psf_spherical_prepare(psf_plan *p, int n_nodes) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (n_nodes < 3 || !(n_nodes & 1) || n_nodes > (1 << 20)) { p->err = "n_nodes must be odd, >= 3 (composite Simpson)"; return PSF_ERR_INVALID_ARG; }
  if (!axisymmetric(p)) return PSF_ERR_STATE;
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
  psf_status sb = bessel_setup(p, n_nodes);
  return sb != PSF_OK ? sb : uploads_fence(p);
  });
}

psf_status psf_compute_spherical(psf_plan *p, void *cuda_stream, float *intensity) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (!intensity || ((uintptr_t)intensity & 15)) { p->err = "intensity must be a 16-byte aligned device pointer"; return PSF_ERR_INVALID_ARG; }
  if (!p->bessel) { p->err = "psf_spherical_prepare has not been called"; return PSF_ERR_STATE; }
  if (!axisymmetric(p)) return PSF_ERR_STATE;
  if (cudaSetDevice(p->device) != cudaSuccess) { p->err = "cudaSetDevice failed"; return PSF_ERR_CUDA; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (p->prof) {
    p->prof_n = 0;
    p->prof_valid = true;
    cudaEventRecord(p->prof_ev[0], st);
  }
  cudaError_t e = launch_bessel(p, st, intensity);
  mark_inflight(p, st);
  if (e != cudaSuccess) { p->err = std::string("kernel launch: ") + cudaGetErrorString(e); return PSF_ERR_CUDA; }
  return PSF_OK;
  });
}

// ---- adjoint ---------------------------------------------------------------------------------------------------------
psf_status psf_gradients(psf_plan *p, void *cuda_stream, const float *dL_dI, double *dL_dz, double *dL_dc) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (!dL_dI || !dL_dz) { p->err = "dL_dI and dL_dz must be device pointers"; return PSF_ERR_INVALID_ARG; }
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  if (grad_needs_setup(p) && wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
  const bool setup = grad_needs_setup(p);
  psf_status s = grad_setup(p);               // first call, or the tables changed: (re)build the adjoint's copies
  if (s == PSF_OK && setup) s = uploads_fence(p);
  if (s != PSF_OK) return s;
  if (dL_dc && grad_terms(p) == 0) { p->err = "dL_dc asked for, but no Zernike terms are set"; return PSF_ERR_STATE; }
  e = launch_grad(p, (cudaStream_t)cuda_stream, dL_dI, dL_dz, dL_dc);
  mark_inflight(p, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) { p->err = std::string("kernel launch: ") + cudaGetErrorString(e); return PSF_ERR_CUDA; }
  return PSF_OK;
  });
}

psf_status psf_plan_destroy(psf_plan *p) {
  if (!p) return PSF_ERR_INVALID_ARG;
  cudaSetDevice(p->device);
  wait_inflight(p);                            // launches of this plan still in flight read its tables
  try { free_all(p); } catch (...) {}
  delete p;
  return PSF_OK;
}

psf_status psf_plan_tune(psf_plan *p, int knob, long long value) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
    if (knob == PSF_TUNE_TC_PAIR_MASK) {
      if (value < 0 || value > 3) { p->err = "PSF_TUNE_TC_PAIR_MASK: 0..3"; return PSF_ERR_INVALID_ARG; }
      p->tune_pair_mask = (int)value;
    } else if (knob == PSF_TUNE_TC_SCRATCH_MB) {
      if (value < 0 || value > (1 << 20)) { p->err = "PSF_TUNE_TC_SCRATCH_MB: 0 (default) .. 2^20"; return PSF_ERR_INVALID_ARG; }
      p->tune_scratch_mb = (int)value;
    } else if (knob == PSF_TUNE_TC_FUSED) {
      if (value < 0 || value > 8) { p->err = "PSF_TUNE_TC_FUSED: 0 (off), 1 (on), 2..8 (on, ring depth forced)"; return PSF_ERR_INVALID_ARG; }
      p->tune_fused = (int)value;
    } else if (knob == PSF_TUNE_GRAD_TENSOR) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_GRAD_TENSOR: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_grad_tensor = (int)value;
    } else if (knob == PSF_TUNE_FUSED_WINDOW) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_FUSED_WINDOW: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_fused_window = (int)value;
    } else if (knob == PSF_TUNE_K1P_ASPLIT) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_K1P_ASPLIT: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_k1p_asplit = (int)value;
    } else if (knob == PSF_TUNE_SMLM) {
      if (value < 0 || value > 2) { p->err = "PSF_TUNE_SMLM: 0..2"; return PSF_ERR_INVALID_ARG; }
      p->tune_smlm = (int)value;
    } else if (knob == PSF_TUNE_K1P_WAITFIRST) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_K1P_WAITFIRST: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_k1p_waitfirst = (int)value;
    } else if (knob == PSF_TUNE_PDL) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_PDL: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_pdl = (int)value;
    } else if (knob == PSF_TUNE_DEVICE_REFRESH) {
      if (value < 0 || value > 1) { p->err = "PSF_TUNE_DEVICE_REFRESH: 0..1"; return PSF_ERR_INVALID_ARG; }
      p->tune_dev_refresh = (int)value;
    } else if (knob == PSF_TUNE_K1P_HANDOFF) {
      if (value < 0 || value > 3) { p->err = "PSF_TUNE_K1P_HANDOFF: 0..3"; return PSF_ERR_INVALID_ARG; }
      p->tune_k1p_handoff = (int)value;
    } else if (knob == PSF_TUNE_K1P_DEFER) {
      if (value < 0 || value > 4) { p->err = "PSF_TUNE_K1P_DEFER: 0..4"; return PSF_ERR_INVALID_ARG; }
      p->tune_k1p_defer = (int)value;
    } else {
      p->err = "unknown tuning knob";
      return PSF_ERR_INVALID_ARG;
    }
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
    if (wait_inflight(p) != cudaSuccess) { p->err = "cudaEventSynchronize (launches in flight) failed"; return PSF_ERR_CUDA; }
    tc_free(p);                                // the tensor path rebuilds its tables, scratch and tensor maps with the new knobs
    return refresh(p);
  });
}

const char *psf_grad_path_name(const psf_plan *p) { return p ? grad_route(p) : ""; }

int psf_grad_terms(const psf_plan *p) {
  if (!p) return 0;
  return p->K_rows > 0 ? p->K_rows : (int)p->zern_shared.size();
}

const char *psf_last_error(const psf_plan *p) { return p ? p->err.c_str() : g_create_err.c_str(); }

int psf_launches_per_compute(const psf_plan *p) {
  if (!p) return 0;
  if (p->path == 3) return 1;
  if (p->path == 4) return p->czt ? czt_launches(p) : 0;
  return (p->path >= 1 && p->tc) ? tc_launches(p) : ffma_launches(p);
}

const char *psf_path_name(const psf_plan *p) { return !p ? "ffma" : p->path == 4 ? "czt_fft" : p->path == 3 ? (smlm_on_tensor_cores(p) ? "fused_tc3xf16" : "ffma_fused") : p->path == 2 ? "tc3xf16" : p->path == 1 ? "tc3xtf32" : "ffma"; }

psf_status psf_profile_enable(psf_plan *p, int enable) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { p->err = cudaGetErrorString(e); return PSF_ERR_CUDA; }
  p->prof = false;
  p->prof_valid = false;
  if (!enable) return PSF_OK;
  size_t need = (size_t)ffma_launches(p) + 1;
  if (p->tc && (size_t)tc_launches(p) + 1 > need) need = (size_t)tc_launches(p) + 1;
  if (p->czt && (size_t)czt_launches(p) + 1 > need) need = (size_t)czt_launches(p) + 1;
  while (p->prof_ev.size() < need) {
    cudaEvent_t ev;
    if ((e = cudaEventCreate(&ev)) != cudaSuccess) { p->err = std::string("cudaEventCreate: ") + cudaGetErrorString(e); return PSF_ERR_CUDA; }
    p->prof_ev.push_back(ev);
  }
  p->prof_stage.assign(p->prof_ev.size(), 0);
  p->prof = true;
  return PSF_OK;
  });
}

psf_status psf_profile_read(psf_plan *p, float *stage_ms, int *launches) {
  if (!p) return PSF_ERR_INVALID_ARG;
  return guarded(p, [&]() -> psf_status {
  if (!stage_ms || !launches) { p->err = "NULL output"; return PSF_ERR_INVALID_ARG; }
  if (!p->prof || !p->prof_valid) { p->err = "profiling is not enabled or no psf_compute ran since"; return PSF_ERR_STATE; }
  for (int i = 0; i < 4; ++i) { stage_ms[i] = 0.f; launches[i] = 0; }
  for (int i = 0; i < p->prof_n; ++i) {
    float ms = 0.f;
    cudaError_t e = cudaEventElapsedTime(&ms, p->prof_ev[i], p->prof_ev[i + 1]);
    if (e != cudaSuccess) { p->err = std::string("cudaEventElapsedTime: ") + cudaGetErrorString(e); return PSF_ERR_CUDA; }
    const int st = p->prof_stage[i] & 3;
    stage_ms[st] += ms;
    launches[st] += 1;
  }
  return PSF_OK;
  });
}

long long psf_last_upload_bytes(const psf_plan *p) { return p ? p->upload_bytes : 0; }

const char *psf_kernel_names(psf_plan *p) {
  if (!p) return "";
  try {
    if (p->path == 3) p->kernel_names = p->smlm ? (smlm_on_tensor_cores(p) ? "k_smlm_tc" : "k_smlm") : "k_small";
    else if (p->path == 4) p->kernel_names = "czt_rows,czt_cols";
    else if ((p->path == 1 || p->path == 2) && p->tc) p->kernel_names = tc_kernel_names(p);
    else p->kernel_names = "k1_stage1,k2_stage2";
    return p->kernel_names.c_str();
  } catch (...) {
    return "";
  }
}

psf_status psf_host_tables(const psf_plan_desc *desc, const float *coeffs, int noll_first, int n_coeffs, int *n_components,
                           double *weights, double *base, double *kappa, unsigned char *mask) {
  return guarded(nullptr, [&]() -> psf_status {
  std::string err;
  psf_status s = validate_desc(desc, err);
  if (s != PSF_OK) { g_create_err = err; return s; }
  if (coeffs && n_coeffs > 0 && noll_first < 1) { g_create_err = "noll_first must be >= 1"; return PSF_ERR_INVALID_ARG; }
  psf_plan_desc d = *desc;
  if (std::isnan(d.n_immersion_design)) d.n_immersion_design = d.n_immersion;
  HostPupil hp;
  build_host_pupil(d, coeffs, noll_first, coeffs ? n_coeffs : 0, hp);
  const size_t NN = (size_t)d.pupil_n * d.pupil_n;
  if (n_components) *n_components = hp.C;
  if (weights) for (int c = 0; c < 5; ++c) weights[c] = hp.weight[c];
  if (base)
    for (size_t i = 0; i < (size_t)hp.C * NN; ++i) { base[2 * i] = hp.base[i].real(); base[2 * i + 1] = hp.base[i].imag(); }
  if (kappa) std::memcpy(kappa, hp.kappa.data(), NN * sizeof(double));
  if (mask) std::memcpy(mask, hp.mask.data(), NN);
  return PSF_OK;
  });
}

}  // extern "C"
