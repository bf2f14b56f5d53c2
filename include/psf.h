/* psf.h -- C ABI of libpsf_b200: Fourier-parametrised vectorial Richards-Wolf propagation of a z-stack
 * on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations are PAPER.md = arXiv 2502.03170, line : equation):
 *   for every plane b of a stack (or every emitter of a batch) and every pixel (x, y) of an M x M grid,
 *
 *     E_c(x,y;b) = -(i f k / 2 pi) * sum over the pupil disc s_x^2+s_y^2 <= s_max^2 of
 *                    a(s) exp{i W(s)} e_inf,c(s) / s_z * exp{i k s_z z_b} exp{i k (s_x x + s_y y)} ds_x ds_y
 *                                                 (Eq. 9 with the corrections of :146 Eq. 15)
 *     I(x,y;b)   = |E_x|^2 + |E_y|^2 + |E_z|^2
 *
 *   with  k = 2 pi n_i / lambda, s_max = NA / n_i, f = 1;
 *         e_inf = polarisation-rotation matrix applied to the input Jones vector (Eq. 6);
 *         a(s)  = sqrt(cos theta) apodisation (Eq. 19) when PSF_FLAG_APODIZE;
 *         W(s)  = Gibson-Lanni phase (Eq. 16 with t_i from :167 Eq. 17) when
 *                 PSF_FLAG_GIBSON_LANNI, plus sum_j c_j Z_j(s) in Noll-indexed Zernike polynomials
 *                 (Eq. 18), plus an optional per-plane tilt -k (s_x x_b + s_y y_b);
 *   discretised on the N x N midpoint pupil grid u_p = (2p+1-N)/N, s = s_max u, weight (s_max 2/N)^2,
 *   output coordinates x_m = (m - (M-1)/2) * pixel.  The readings taken where the paper is silent are
 *   listed in DESIGN.md.  The zoomed DFT is evaluated as two real-matrix product stages (rows, then
 *   columns) on the GPU; the per-plane pupil is generated inside the first product and never stored.
 *
 * Conventions
 *   - all lengths in micrometres; all `const T *` arguments marked "host" are read before the call returns;
 *   - device pointers are CUDA device memory of the plan's device, 16-byte aligned, owned by the caller;
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - every call returns a psf_status; nothing throws or aborts across the ABI; on error outputs are
 *     unspecified and *out is NULL; the message is available from psf_last_error();
 *   - psf_plan_create / psf_set_* may allocate device memory and synchronise; psf_compute only enqueues
 *     kernels (and one event record) on `cuda_stream`: it never allocates, never synchronises, never copies
 *     and never touches host memory;
 *   - ordering guarantee: every call that overwrites or frees device tables (psf_set_*, psf_plan_tune,
 *     psf_spherical_prepare, the table rebuild inside psf_gradients, psf_plan_destroy) first waits, on the host,
 *     for the launches of this plan's earlier psf_compute / psf_compute_spherical / psf_gradients calls, on
 *     whatever stream they were enqueued (blocking or non-blocking): compute(stream) followed at once by
 *     psf_set_zernike is safe, and the earlier call still sees the old tables;
 *   - every call makes the plan's device current (cudaSetDevice) and leaves it current;
 *   - a plan is not thread-safe; distinct plans are independent (also across threads and devices);
 *   - there is no CPU fallback: without a CUDA device of compute capability 10.x, psf_plan_create fails.
 */
#ifndef PSF_B200_H
#define PSF_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psf_plan psf_plan; /* opaque, owned by the library */

typedef enum {
  PSF_OK = 0,
  PSF_ERR_INVALID_ARG = 1, /* NA<=0, NA>=n_immersion, lambda<=0, N<2, M<1, pixel<=0, n_planes<1, non-finite z,
                              noll_first<1, null pointers, misaligned outputs                                 */
  PSF_ERR_UNSUPPORTED = 2, /* field output with PSF_POL_UNPOLARIZED, device without sm_100                            */
  PSF_ERR_ALLOC = 3,       /* host or device allocation failed                                                 */
  PSF_ERR_CUDA = 4,        /* any CUDA runtime failure (message via psf_last_error)                            */
  PSF_ERR_STATE = 5        /* call order violated (e.g. shifts given for another n_planes)                     */
} psf_status;

typedef enum {
  PSF_POL_X = 0,          /* (1, 0)                                                                             */
  PSF_POL_Y = 1,          /* (0, 1)                                                                             */
  PSF_POL_CIRC_L = 2,     /* (1, +i)/sqrt(2)                                                                    */
  PSF_POL_CIRC_R = 3,     /* (1, -i)/sqrt(2)                                                                    */
  PSF_POL_JONES = 4,      /* custom complex (px, py) from psf_plan_desc.jones, used as given                    */
  PSF_POL_UNPOLARIZED = 5 /* 1/2 (I_x + I_y): x and y inputs summed incoherently, unit input power              */
} psf_pol;

enum {
  PSF_FLAG_APODIZE = 1,      /* a(s) = sqrt(cos theta), Eq. 19                                     */
  PSF_FLAG_GIBSON_LANNI = 2, /* W(s) of PAPER.md:154 Eq. 16                                                     */
  PSF_FLAG_FRESNEL = 4,      /* q_s, q_p of PAPER.md:102-107 Eq. 7-8 over immersion -> glass (n_glass) -> sample,
                                complex past a critical angle; ignored by PSF_MODEL_SCALAR                       */
  PSF_FLAG_GAUSSIAN_ENVELOPE = 8 /* a(s) *= exp(-sin^2 theta / envelope_s^2), Eq. 20              */
};

typedef enum {
  PSF_MODEL_VECTORIAL = 0, /* PAPER.md:116 Eq. 9: three field components through the rotation matrix of Eq. 6   */
  PSF_MODEL_SCALAR = 1     /* PAPER.md:70 Eq. 3: e_inf = e_inc = 1, one component; `pol` and `jones` are ignored */
} psf_model;

typedef enum {
  PSF_PREC_AUTO = 0,   /* the library picks per problem size: 3XF16 when the tensor tiles fill, FP32 otherwise  */
  PSF_PREC_3XTF32 = 1, /* tcgen05 tensor cores, both operands split hi/lo in TF32 (fp32-level accuracy)         */
  PSF_PREC_FP32 = 2,   /* plain fp32 FFMA tiles                                                                 */
  PSF_PREC_3XF16 = 3,  /* tcgen05 tensor cores, both operands pre-scaled by powers of two and split hi/lo in FP16:
                          same 11-bit parts as 3XTF32, half the bytes, twice the tensor rate     */
  PSF_PREC_CZT_FFT = 4 /* the paper's own formulation of the zoomed DFT: chirp-Z transform per row and
                          column by hand-written shared-memory fp32 FFTs of length 2^ceil(log2(N + M - 1)) (Bluestein; an
                          exact re-association of the same finite sum).  Static mode only (no per-plane Zernike rows or
                          shifts: PSF_ERR_UNSUPPORTED), N + M - 1 <= 8192.  Never chosen by PSF_PREC_AUTO: on B200 the
                          tensor-core product form is faster at every measured size (profiles/r2_czt_crossover.md)      */
} psf_precision;

typedef struct {
  double NA, wavelength_um, n_immersion, n_sample;
  /* Gibson-Lanni, PAPER.md:154-167 (read iff PSF_FLAG_GIBSON_LANNI) */
  double particle_depth_um;                         /* t_s                                                      */
  double n_glass, t_glass_um;                       /* n_g, t_g                                                 */
  double n_glass_design, t_glass_design_um;         /* n_g*, t_g*                                               */
  double n_immersion_design, t_immersion_design_um; /* n_i*, t_i*                                               */
  double t_immersion_um;                            /* t_i; NaN -> derived from Eq. 17 as printed               */
  int pupil_n;                                      /* N: the pupil grid is N x N                               */
  int out_m;                                        /* M: the image grid is M x M                               */
  double pixel_um;                                  /* output pixel size                                        */
  int n_planes;                                     /* Z: number of planes (or emitters)                        */
  const double *z_um;                               /* host, length n_planes, copied                            */
  psf_pol pol;
  double jones[4];                                  /* re px, im px, re py, im py (PSF_POL_JONES only)          */
  unsigned flags;                                   /* PSF_FLAG_*                                               */
  psf_precision precision;
  int device;                                       /* CUDA device ordinal                                      */
  psf_model model;                                  /* vectorial (0) or scalar                                  */
  double envelope_s;                                /* s_env > 0, read iff PSF_FLAG_GAUSSIAN_ENVELOPE           */
} psf_plan_desc;

/* Build a plan: validates `desc`, evaluates every z-independent factor of the integrand in fp64 on the host
 * (disc mask in integers, rotation matrix x Jones vector, apodisation / s_z, Gibson-Lanni phase incl. the
 * evanescent branch, wavenumber tables, zoomed-DFT matrices), rounds to fp32 and uploads.  *out owns all
 * device memory of the plan (tables + scratch) until psf_plan_destroy. */
psf_status psf_plan_create(const psf_plan_desc *desc, psf_plan **out);

/* Zernike phase W = sum_{i<n_coeffs} coeffs[i] * Z_{noll_first+i}, radians, Noll-normalised (Eq. 18).
 * per_plane == 0: coeffs[n_coeffs] shared by all planes (folded into the static pupil);
 * per_plane == 1: coeffs[n_planes][n_coeffs], row b for plane b (evaluated in the pupil producer).
 * coeffs == NULL or n_coeffs == 0 clears the Zernike term.  coeffs is host memory, copied.
 * Cost: a change of the term list, or of the mode, rebuilds and uploads the plan's tables (host, fp64).  Two cases are cheap,
 * as they are the inner loop of a fit: new shared values on a plan that runs the 3xFP16 pair kernels are folded into the
 * operand tables on the device (K doubles uploaded, two small launches; see PSF_TUNE_DEVICE_REFRESH), and new per-plane rows for
 * the terms already set upload the rows only (2 * n_planes * n_coeffs floats).  psf_last_upload_bytes reports what a call moved. */
psf_status psf_set_zernike(psf_plan *plan, const float *coeffs, int noll_first, int n_coeffs, int per_plane);

/* Free phase mask W_0 of PAPER.md:176 Eq. 18 (vortex ramp, half-moon, measured wavefront ...): w0_rad is host
 * [N][N] radians on the pupil grid (row = p_y, sample (p_y, p_x) at s = s_max (2p + 1 - N)/N), added to the static
 * phase of every plane; values outside the disc are ignored.  NULL clears.  Copied. */
psf_status psf_set_phase_mask(psf_plan *plan, const float *w0_rad);

/* Per-plane lateral emitter position (x_b, y_b): plane b becomes I(x - x_b, y - y_b; z_b), applied as the pupil
 * tilt phase -k (s_x x_b + s_y y_b).  xy_um is host [n_planes][2]; NULL clears.  Setting shifts for the first time (or
 * clearing them) switches the plan between static and per-plane mode and rebuilds its tables; new values where shifts are
 * already set upload the plane table only (16 bytes per plane). */
psf_status psf_set_shifts(psf_plan *plan, const float *xy_um);

/* Enqueue the whole stack on `cuda_stream`:
 *   intensity : device fp32 [n_planes][M][M], x fastest (required);
 *   field     : device complex64 (interleaved re, im) [3][n_planes][M][M] = (E_x, E_y, E_z), or NULL
 *               ([1][n_planes][M][M] for PSF_MODEL_SCALAR).
 * Asynchronous; results are valid once the stream has passed this point.  Enqueue-only on every kernel path: the
 * tensor-core stage-2 kernels write the field from their epilogue, no table is uploaded here. */
psf_status psf_compute(psf_plan *plan, void *cuda_stream, float *intensity, void *field);

/* Spherical (Bessel) parametrisation of the same integral, Eq. 11-14 (Eq. 5 for PSF_MODEL_SCALAR):
 * three 1-D integrals over theta per (radius, plane) by composite Simpson with `n_nodes` (odd, >= 3) nodes, then Eq. 11
 * with the plan's Jones vector.  Valid for axisymmetric pupils only: PSF_ERR_STATE while Zernike terms, shifts or a
 * phase mask are set.  It is a different discretisation of the integral than psf_compute (quadrature in theta instead of
 * the N x N pupil grid): the two agree to the quadrature error of the pupil grid, not to rounding.
 *   psf_spherical_prepare : host tables for n_nodes, device scratch [n_planes][m (m + 1) / 2][3] complex64 (may allocate);
 *   psf_compute_spherical : enqueue on `cuda_stream`; intensity is device fp32 [n_planes][M][M] as for psf_compute. */
psf_status psf_spherical_prepare(psf_plan *plan, int n_nodes);
psf_status psf_compute_spherical(psf_plan *plan, void *cuda_stream, float *intensity);

/* Adjoint of psf_compute (the paper's differentiable-PSF use): for L = sum dL_dI[b][y][x] *
 * I[b][y][x] the gradients with respect to the plane parameters the pupil phase depends on,
 *   dL_dz : device fp64 [n_planes]            dL / d z_b (per micrometre);
 *   dL_dc : device fp64 [n_planes][K] or NULL  dL / d c_bj for the K Zernike terms currently set (radians^-1); row b is
 *           the contribution of plane b: for shared coefficients the gradient is the column sum over the planes.
 * dL_dI is device fp32 [n_planes][M][M].  All polarisations incl. PSF_POL_UNPOLARIZED, both models, every correction
 * factor.  The first call (and the first call after any psf_set_*) builds device copies of the unfolded tables and
 * allocates scratch, so it may allocate and synchronise; later calls only enqueue on `cuda_stream`.
 * On a plan that runs on the tensor cores (3xFP16, static mode) both transforms of the adjoint run there too: the field
 * from the forward kernels, then the back-projection as the same zoomed transform with the two grids swapped (a second,
 * internal plan), scratch 8 bytes x (C Z M^2 + C Z N^2) + 32 bytes x C Z ceil(M/2)^2 (padded). */
psf_status psf_gradients(psf_plan *plan, void *cuda_stream, const float *dL_dI, double *dL_dz, double *dL_dc);

psf_status psf_plan_destroy(psf_plan *plan);

/* Route the last psf_gradients of this plan took: "adjoint_tc3xf16" (both transforms on the tensor cores: static mode on the
 * 3xFP16 path), "adjoint_ffma" (fp32 FFMA products: every other case), "" before the first call (static string). */
const char *psf_grad_path_name(const psf_plan *plan);

/* Number of Zernike terms currently set (shared or per plane) = the row length K of psf_gradients' dL_dc. */
int psf_grad_terms(const psf_plan *plan);

/* Test / A-B knobs of the tensor-core path (never needed for normal use; the library reads no environment variable
 * for them).  Rebuilds the tensor path's tables and scratch: may allocate and synchronise.
 *   PSF_TUNE_TC_PAIR_MASK  : value ANDed with the plan's choice; bit 0 = stage 1 on CTA pairs (cta_group::2),
 *                            bit 1 = stage 2 on CTA pairs; 0 forces the single-CTA tcgen05 kernels (default 3);
 *   PSF_TUNE_TC_SCRATCH_MB : budget in MB of the stage-1 -> stage-2 scratch (default 0 = 4096): a smaller value splits a
 *                            stack into several launch pairs;
 *   PSF_TUNE_K1P_HANDOFF   : stage-1 pair kernel, how the non-leader CTA's producer warps signal the leader's barrier:
 *                            0 (default) plain remote arrive, 1 cluster-scope release per warp; 2 / 3 = diagnosis settings of
 *                            profiles/r5_soak.md (plain arrive; the operand slot of the leader / of the peer is released one K-step late,
 *                            the other's two, whatever PSF_TUNE_K1P_DEFER says): not for use;
 *   PSF_TUNE_K1P_DEFER     : producer-written operand slots are released that many K-steps (three UMMAs each) after the stage's
 *                            last UMMA: 2 (default), 1 (round 2's first setting: alone, one wrong plane in about 25000 calls),
 *                            0 = at once (alone, about one call in 100: the A/B setting of profiles/r2_race_k1_pair.md), up to 4.
 *                            The margin alone is not robust (two K-steps failed once in 150000 calls in one build): it is
 *                            combined with PSF_TUNE_K1P_WAITFIRST; profiles/r5_soak.md has the measured rates and costs;
 *   PSF_TUNE_TC_FUSED      : 1 (default) = where both stages run on CTA pairs and take about equal time, they are enqueued as
 *                            ONE kernel (k12_fused) whose stage-2 clusters consume the scratch right behind the stage-1
 *                            clusters, so that it stays in L2; 0 = always two kernels; 2..8 = fused with that ring depth.
 *                            Known issue (profiles/r5_soak.md): in soaks the fused launch produced one wrong plane in about one of
 *                            4e5 config-5 calls; the two-kernel path (0) was clean in 1.3e6;
 *   PSF_TUNE_SMLM          : 1 (default) = small grids in per-plane mode (emitter batches) run the emitter-batch kernels where the plan
 *                            qualifies: k_smlm_tc (tcgen05; output half-size <= 16, precision AUTO or 3XF16), else k_smlm (fp32 FMA);
 *                            2 = k_smlm, never the tensor-core variant; 0 = always k_small;
 *   PSF_TUNE_K1P_ASPLIT    : 1 (default) = in the stage-1 pair kernel the TMA-written table half of a stage buffer has its own barrier and
 *                            is released right behind its own stage (only the producer-written half needs the deferred release);
 *                            0 = one barrier for both halves (round 1);
 *   PSF_TUNE_FUSED_WINDOW  : 1 = the fused launch carries a persisting L2 access-policy window over its ring scratch (the library then
 *                            raises the device's cudaLimitPersistingL2CacheSize to the ring size); 0 (default) = none - measured, the
 *                            window doubles the DRAM writes and gains no time (profiles/r2_fused_cfg5.md);
 *   PSF_TUNE_GRAD_TENSOR   : 1 (default) = psf_gradients runs its two transforms on the tensor cores where the plan is on the 3xFP16
 *                            path in static mode; 0 = the fp32 FFMA route of round 1;
 *   PSF_TUNE_DEVICE_REFRESH: 1 (default) = on a plan that runs the 3xFP16 pair kernels, psf_set_zernike (shared coefficients) and
 *                            psf_set_phase_mask recompute the phase, the fold and the operand scales on the device from resident
 *                            fp64 copies of the static pupil and the Zernike basis (same arithmetic, same order as the host path);
 *                            0 = the host path (fp64 on the host cores + upload of the folded tables);
 *   PSF_TUNE_PDL           : 1 (default) = on the two-kernel tensor path the stage-2 kernel is a programmatic dependent launch of
 *                            stage 1: its CTAs take the SMs stage 1 leaves, run their prologue (barriers, TMEM, table loads) and
 *                            wait (griddepcontrol.wait) for the stage-1 grid to complete before the first read of its output;
 *                            0 = plain stream order;
 *   PSF_TUNE_K1P_WAITFIRST : 1 (default) = the stage-1 producers wait for their operand slot before they compute its rows, so that the
 *                            computation lies between the observed release and the first store into the slot; 0 = they compute
 *                            first and wait with the rows in registers (round 2's earlier order; profiles/r5_soak.md). */
enum { PSF_TUNE_TC_PAIR_MASK = 1, PSF_TUNE_TC_SCRATCH_MB = 2, PSF_TUNE_K1P_HANDOFF = 3, PSF_TUNE_K1P_DEFER = 4, PSF_TUNE_TC_FUSED = 5,
       PSF_TUNE_SMLM = 6, PSF_TUNE_GRAD_TENSOR = 7, PSF_TUNE_K1P_ASPLIT = 8,
       PSF_TUNE_FUSED_WINDOW = 9, PSF_TUNE_DEVICE_REFRESH = 10, PSF_TUNE_PDL = 11, PSF_TUNE_K1P_WAITFIRST = 12 };
psf_status psf_plan_tune(psf_plan *plan, int knob, long long value);

/* Last error message of `plan`, or (plan == NULL) of the calling thread's last failed psf_plan_create /
 * psf_host_tables / psf_propagate_static.  Never NULL; valid until the next call on the same plan / thread. */
const char *psf_last_error(const psf_plan *plan);

/* Number of kernel launches one psf_compute call of this plan enqueues (for benchmarking records). */
int psf_launches_per_compute(const psf_plan *plan);

/* Name of the kernel path the plan selected (static string): "ffma" (fp32 FFMA tiles), "ffma_fused" (small grids: the
 * whole path in one kernel, fp32 FMA: k_small, k_smlm), "fused_tc3xf16" (emitter batches on small grids: the whole path in one
 * kernel with both DFT stages on tcgen05, 3xFP16 split: k_smlm_tc), "tc3xtf32", "tc3xf16" (tcgen05 tensor cores, split precision,
 * one kernel per stage or both in k12_fused), "czt_fft" (chirp-Z by FFT). */
const char *psf_path_name(const psf_plan *plan);

/* Comma-separated names of the kernels one psf_compute of this plan launches, in launch order (stage 1, stage 2; one
 * name for the fused small-grid path), e.g. "k1_pair,k2_pair".  Owned by the plan, valid until the next call on it. */
const char *psf_kernel_names(psf_plan *plan);

/* Profiling aid for bench.py.  enable != 0: create CUDA events (this call may allocate) and make every later
 * psf_compute bracket each of its kernel launches with cudaEventRecord on the compute stream; enable == 0: stop. */
psf_status psf_profile_enable(psf_plan *plan, int enable);

/* After the caller has synchronised the stream of the last psf_compute: device time per stage of that call.
 *   stage_ms : host out [4], milliseconds summed over the launches of each stage
 *              (0 = stage-1 row DFT with the fused pupil producer, 1 = stage-2 column DFT + intensity,
 *               2 = Bessel integrals, 3 = Eq. 11 combination of psf_compute_spherical);
 *   launches : host out [4], number of launches of each stage.
 * PSF_ERR_STATE if profiling is not enabled or no psf_compute ran since. */
psf_status psf_profile_read(psf_plan *plan, float *stage_ms, int *launches);

/* Bytes copied host->device by the last psf_plan_create / psf_set_zernike / psf_set_shifts of this plan. */
long long psf_last_upload_bytes(const psf_plan *plan);

/* The zoomed Fourier sum of PAPER.md:116 Eq. 9 WITHOUT a plan and without any allocation, for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it; psf_plan_create allocates):
 *   E_c[z][my][mx] = sum_{py,px} pupil[z][c][py][px] exp(+i k s_max (u_px x_mx + u_py y_my)),   I[z] = sum_c weights[c] |E_c[z]|^2,
 *   u_p = (2p + 1 - N)/N, x_m = (m - (M-1)/2) pixel_um, k s_max = 2 pi NA / wavelength_um (readings A4, A6, A9).
 * The caller passes everything: `pupil` = DEVICE float2 [n_planes][n_components][pupil_n][pupil_n] (row = p_y), the complete
 * pupil field of every plane with every phase, prefactor and quadrature weight in it (e.g. psf_host_tables' base times
 * exp(i kappa z)), 8-byte aligned; `weights` = HOST float [n_components], read before the call returns; `intensity` = DEVICE
 * float [n_planes][out_m][out_m], written in stream order.  fp32 complex products (two kernels: rows, then columns with |E|^2
 * in the epilogue); the row -> column scratch and the DFT table live in a file-scope `static __device__` array of
 * PSF_STATIC_SCRATCH_BYTES that every GPU using this entry point holds until the process exits.
 * Limit: (n_components + 1) * out_m * pupil_n * 8 bytes (the table's share rounded up to 256) must fit the array, e.g. three
 * components at 512 x 512 or five at 256 x 512; n_planes is free (planes go through in passes that fit).  Larger sizes return PSF_ERR_UNSUPPORTED with the byte counts
 * in psf_last_error(NULL); nothing is launched.  n_components is 1..5.
 * The call only enqueues kernels on `cuda_stream` (NULL = the legacy default stream) of the CURRENT device: no cudaMalloc, cudaFree,
 * copy or synchronisation.  The first call on a device looks the array's device address up (cudaGetSymbolAddress, once per
 * device): make one call outside a stream capture first.
 * All calls on a device share the array, which keeps the last call's contents (nothing in it needs clearing: every call rewrites
 * what it reads).  Calls that overlap on the GPU - two streams, or two host threads on one device - race on it: serialise them
 * (one stream, or events).  Errors: PSF_ERR_INVALID_ARG (NULL / misaligned pointers, non-positive sizes or optics, non-finite
 * weights), PSF_ERR_UNSUPPORTED (too large), PSF_ERR_CUDA; the message is psf_last_error(NULL) of the calling thread. */
#define PSF_STATIC_SCRATCH_BYTES (16u << 20)
psf_status psf_propagate_static(void *cuda_stream, const void *pupil, int n_planes, int n_components, int pupil_n, int out_m,
                                double NA, double wavelength_um, double pixel_um, const float *weights, float *intensity);

/* Host-only diagnostic (no device needed): the plan-time static pupil in fp64, before folding and rounding.
 *   n_components : out, 3 (coherent input), 5 (unpolarised: the distinct scalar pupils a, b, d, c_x, c_y) or 1 (scalar);
 *   weights      : out [5], intensity weight of each component;
 *   base         : out [n_components][N][N][2] (re, im) = prefactor * a / s_z * e_inf,c * exp(i W_static), 0 outside
 *                  the disc; W_static includes the shared Zernike term given here (coeffs may be NULL);
 *   kappa        : out [N][N], k cos(theta) in rad/um;     mask : out [N][N], 1 inside the disc.
 * Any output pointer may be NULL.  base must hold 5*N*N*2 doubles. */
psf_status psf_host_tables(const psf_plan_desc *desc, const float *coeffs, int noll_first, int n_coeffs,
                           int *n_components, double *weights, double *base, double *kappa, unsigned char *mask);

#ifdef __cplusplus
}
#endif
#endif /* PSF_B200_H */
