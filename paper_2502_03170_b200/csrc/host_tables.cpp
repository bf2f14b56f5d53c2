// fp64 plan-time tables.  See host_tables.hpp.  Readings of the paper (G1, A1-A10, Z) are listed in DESIGN.md.
#include "host_tables.hpp"

#include <cmath>

namespace psf {

static const double kPi = 3.14159265358979323846;

psf_status validate_desc(const psf_plan_desc *d, std::string &err) {
  if (!d) { err = "desc is NULL"; return PSF_ERR_INVALID_ARG; }
  auto bad = [&](const char *m) { err = m; return PSF_ERR_INVALID_ARG; };
  if (!(d->NA > 0) || !std::isfinite(d->NA)) return bad("NA must be > 0");
  if (!(d->n_immersion > 0) || !std::isfinite(d->n_immersion)) return bad("n_immersion must be > 0");
  if (!(d->NA < d->n_immersion)) return bad("NA must be < n_immersion (s_max = NA/n_i < 1)");
  if (!(d->wavelength_um > 0) || !std::isfinite(d->wavelength_um)) return bad("wavelength_um must be > 0");
  if (!(d->n_sample > 0) || !std::isfinite(d->n_sample)) return bad("n_sample must be > 0");
  if (d->pupil_n < 2) return bad("pupil_n must be >= 2");
  if (d->pupil_n > 8192) return bad("pupil_n must be <= 8192");
  if (d->out_m < 1) return bad("out_m must be >= 1");
  if (d->out_m > 8192) return bad("out_m must be <= 8192");
  if (!(d->pixel_um > 0) || !std::isfinite(d->pixel_um)) return bad("pixel_um must be > 0");
  if (d->n_planes < 1) return bad("n_planes must be >= 1");
  if (!d->z_um) return bad("z_um is NULL");
  for (int i = 0; i < d->n_planes; ++i)
    if (!std::isfinite(d->z_um[i])) return bad("z_um holds a non-finite value");
  if ((int)d->pol < 0 || (int)d->pol > (int)PSF_POL_UNPOLARIZED) return bad("unknown polarisation");
  if (d->pol == PSF_POL_JONES)
    for (int i = 0; i < 4; ++i)
      if (!std::isfinite(d->jones[i])) return bad("jones holds a non-finite value");
  if ((int)d->precision < 0 || (int)d->precision > (int)PSF_PREC_CZT_FFT) return bad("unknown precision");
  if (d->flags & ~(unsigned)(PSF_FLAG_APODIZE | PSF_FLAG_GIBSON_LANNI | PSF_FLAG_FRESNEL | PSF_FLAG_GAUSSIAN_ENVELOPE))
    return bad("unknown flag bit");
  if ((int)d->model != (int)PSF_MODEL_VECTORIAL && (int)d->model != (int)PSF_MODEL_SCALAR) return bad("unknown model");
  if ((d->flags & PSF_FLAG_GAUSSIAN_ENVELOPE) && !(d->envelope_s > 0 && std::isfinite(d->envelope_s)))
    return bad("envelope_s must be > 0 with PSF_FLAG_GAUSSIAN_ENVELOPE");
  if ((d->flags & PSF_FLAG_FRESNEL) && !(d->n_glass > 0 && std::isfinite(d->n_glass)))
    return bad("n_glass must be > 0 with PSF_FLAG_FRESNEL (interfaces immersion -> glass -> sample)");
  if (d->flags & PSF_FLAG_GIBSON_LANNI) {
    const double v[] = {d->particle_depth_um, d->n_glass, d->t_glass_um, d->n_glass_design, d->t_glass_design_um,
                        d->t_immersion_design_um};
    for (double x : v)
      if (!std::isfinite(x)) return bad("Gibson-Lanni parameter is not finite");
    if (!(d->n_glass > 0) || !(d->n_glass_design > 0)) return bad("Gibson-Lanni refractive indices must be > 0");
    // n_immersion_design: NaN means "same as n_immersion"
    if (!std::isnan(d->n_immersion_design) && !(d->n_immersion_design > 0 && std::isfinite(d->n_immersion_design)))
      return bad("n_immersion_design must be > 0 or NaN");
    if (std::isinf(d->t_immersion_um)) return bad("t_immersion_um must be finite or NaN");
  }
  return PSF_OK;
}

void noll_to_nm(int j, int &n, int &m, int &kind) {
  n = 0;
  while ((n + 1) * (n + 2) / 2 < j) ++n;       // largest n with n(n+1)/2 < j
  const int k = j - n * (n + 1) / 2;            // 1 .. n+1
  m = (n % 2 == 0) ? 2 * (k / 2) : 2 * ((k - 1) / 2) + 1;
  kind = (m == 0) ? 0 : ((j % 2 == 0) ? 1 : 2);
}

static double factorial(int v) {
  double r = 1.0;
  for (int i = 2; i <= v; ++i) r *= i;
  return r;
}

double zernike_noll(int j, double rho, double cosphi, double sinphi) {
  int n, m, kind;
  noll_to_nm(j, n, m, kind);
  // radial polynomial R_n^m by Horner in rho^2 from the highest power down
  double R = 0.0;
  const int smax = (n - m) / 2;
  for (int s = 0; s <= smax; ++s) {
    const double c = ((s & 1) ? -1.0 : 1.0) * factorial(n - s) /
                     (factorial(s) * factorial((n + m) / 2 - s) * factorial((n - m) / 2 - s));
    R += c * std::pow(rho, n - 2 * s);
  }
  if (kind == 0) return std::sqrt(n + 1.0) * R;
  // cos(m phi), sin(m phi) by the angle-addition recurrence from (cos phi, sin phi)
  double cm = 1.0, sm = 0.0;
  for (int i = 0; i < m; ++i) {
    const double c2 = cm * cosphi - sm * sinphi;
    sm = sm * cosphi + cm * sinphi;
    cm = c2;
  }
  return std::sqrt(2.0 * (n + 1.0)) * R * (kind == 1 ? cm : sm);
}

// principal square root of a real number as a complex one: +i sqrt(|v|) for v < 0 (evanescent branch, A3b)
static cplx csqrt_real(double v) { return v >= 0 ? cplx(std::sqrt(v), 0.0) : cplx(0.0, std::sqrt(-v)); }

// q_s, q_p of PAPER.md:102-107 Eq. 7-8 (readings G2, A2): product over the interfaces immersion -> glass -> sample,
// Snell's law n_j sin(theta_j) = n_i sin(theta), principal complex root for cos(theta_j) past a critical angle
static void fresnel_q(const psf_plan_desc &d, double sinth, cplx &qs, cplx &qp) {
  const double n[3] = {d.n_immersion, d.n_glass, d.n_sample};
  const double a = d.n_immersion * sinth;
  cplx c[3];
  for (int j = 0; j < 3; ++j) c[j] = csqrt_real(1.0 - (a / n[j]) * (a / n[j]));
  qs = cplx(1, 0);
  qp = cplx(1, 0);
  for (int j = 0; j < 2; ++j) {
    qs *= 2.0 * n[j] * c[j] / (n[j] * c[j] + n[j + 1] * c[j + 1]);
    qp *= 2.0 * n[j] * c[j] / (n[j + 1] * c[j] + n[j] * c[j + 1]);
  }
}

static cplx gibson_lanni_W(const psf_plan_desc &d, double sinth) {
  const double k0 = 2.0 * kPi / d.wavelength_um;
  const double ni = d.n_immersion, nis = d.n_immersion_design;
  double ti = d.t_immersion_um;
  if (std::isnan(ti))   // PAPER.md:167 Eq. 17 as printed (leading bare t_s)
    ti = d.particle_depth_um + ni * (-d.particle_depth_um / d.n_sample - d.t_glass_um / d.n_glass +
                                     d.t_glass_design_um / d.n_glass_design + d.t_immersion_design_um / nis);
  const double a2 = ni * ni * sinth * sinth;
  cplx opd = d.particle_depth_um * csqrt_real(d.n_sample * d.n_sample - a2);
  opd += ti * csqrt_real(ni * ni - a2);
  opd -= d.t_immersion_design_um * csqrt_real(nis * nis - a2);
  opd += d.t_glass_um * csqrt_real(d.n_glass * d.n_glass - a2);
  opd -= d.t_glass_design_um * csqrt_real(d.n_glass_design * d.n_glass_design - a2);
  return k0 * opd;   // PAPER.md:154 Eq. 16
}

void build_host_pupil(const psf_plan_desc &d, const float *coeffs, int noll_first, int n_coeffs, HostPupil &P) {
  const int N = d.pupil_n;
  P.N = N;
  P.k = 2.0 * kPi * d.n_immersion / d.wavelength_um;
  P.s_max = d.NA / d.n_immersion;
  const bool scalar = d.model == PSF_MODEL_SCALAR;               // PAPER.md:70 Eq. 3: e_inf = e_inc = 1
  const bool unpol = !scalar && d.pol == PSF_POL_UNPOLARIZED;
  P.C = scalar ? 1 : (unpol ? 5 : 3);
  for (int c = 0; c < 5; ++c) P.weight[c] = 0.0;
  if (unpol) {   // I = 1/2 (|A|^2 + 2|B|^2 + |D|^2 + |C_x|^2 + |C_y|^2): the two inputs share the off-diagonal entry
    const double w[5] = {0.5, 1.0, 0.5, 0.5, 0.5};
    for (int c = 0; c < 5; ++c) P.weight[c] = w[c];
  } else {
    for (int c = 0; c < P.C; ++c) P.weight[c] = 1.0;
  }
  cplx jx(1, 0), jy(0, 0);
  const double r2 = std::sqrt(0.5);
  switch (d.pol) {
    case PSF_POL_X: jx = cplx(1, 0); jy = cplx(0, 0); break;
    case PSF_POL_Y: jx = cplx(0, 0); jy = cplx(1, 0); break;
    case PSF_POL_CIRC_L: jx = cplx(r2, 0); jy = cplx(0, r2); break;
    case PSF_POL_CIRC_R: jx = cplx(r2, 0); jy = cplx(0, -r2); break;
    case PSF_POL_JONES: jx = cplx(d.jones[0], d.jones[1]); jy = cplx(d.jones[2], d.jones[3]); break;
    default: break;
  }
  const size_t NN = (size_t)N * N;
  P.mask.assign(NN, 0);
  P.kappa.assign(NN, 0.0);
  P.rho.assign(NN, 0.0);
  P.cosphi.assign(NN, 1.0);
  P.sinphi.assign(NN, 0.0);
  P.base.assign((size_t)P.C * NN, cplx(0, 0));
  const double du = 2.0 / N;
  const cplx pref = cplx(0.0, -P.k / (2.0 * kPi)) * (P.s_max * du) * (P.s_max * du);   // -(i k / 2 pi) (s_max du)^2, f = 1
  const bool apod = (d.flags & PSF_FLAG_APODIZE) != 0;
  const bool gl = (d.flags & PSF_FLAG_GIBSON_LANNI) != 0;
  const bool env = (d.flags & PSF_FLAG_GAUSSIAN_ENVELOPE) != 0;
  const bool fres = (d.flags & PSF_FLAG_FRESNEL) != 0;
  for (int py = 0; py < N; ++py) {
    for (int px = 0; px < N; ++px) {
      const long ax = 2L * px + 1 - N, ay = 2L * py + 1 - N;
      if (ax * ax + ay * ay > (long)N * N) continue;     // integer disc test, '<=' inside
      const size_t i = (size_t)py * N + px;
      P.mask[i] = 1;
      const double sx = P.s_max * (double)ax / N, sy = P.s_max * (double)ay / N;
      const double st = std::sqrt(sx * sx + sy * sy);
      const double ct = std::sqrt(1.0 - st * st);
      const double cp = st > 0 ? sx / st : 1.0, sp = st > 0 ? sy / st : 0.0;
      P.kappa[i] = P.k * ct;
      P.rho[i] = st / P.s_max;
      P.cosphi[i] = cp;
      P.sinphi[i] = sp;
      double amp = (apod ? std::sqrt(ct) : 1.0) / ct;           // Eq. 19 x the 1/s_z of Eq. 9
      if (env) amp *= std::exp(-(st * st) / (d.envelope_s * d.envelope_s));   // PAPER.md:194 Eq. 20
      cplx W(0, 0);
      if (gl) W += gibson_lanni_W(d, st);
      if (coeffs)
        for (int j = 0; j < n_coeffs; ++j) W += (double)coeffs[j] * zernike_noll(noll_first + j, P.rho[i], cp, sp);
      const cplx stat = pref * amp * std::exp(cplx(0, 1) * W);
      // PAPER.md:93-97 Eq. 6; q_s = q_p = 1 unless PSF_FLAG_FRESNEL
      cplx qs(1, 0), qp(1, 0);
      if (fres) fresnel_q(d, st, qs, qp);
      const double c2 = cp * cp - sp * sp, s2 = 2.0 * sp * cp;
      const cplx a = 0.5 * (qs * (1.0 - c2) + qp * ((1.0 + c2) * ct));
      const cplx b = 0.5 * (-qs + qp * ct) * s2;
      const cplx dd = 0.5 * (qs * (1.0 + c2) + qp * ((1.0 - c2) * ct));
      const cplx cx = -qp * (cp * st), cy = -qp * (sp * st);
      if (scalar) {
        P.base[i] = stat;
      } else if (unpol) {
        const cplx g[5] = {a, b, dd, cx, cy};
        for (int c = 0; c < 5; ++c) P.base[(size_t)c * NN + i] = stat * g[c];
      } else {
        P.base[0 * NN + i] = stat * (a * jx + b * jy);
        P.base[1 * NN + i] = stat * (b * jx + dd * jy);
        P.base[2 * NN + i] = stat * (cx * jx + cy * jy);
      }
    }
  }
}

void build_zernike_basis(const HostPupil &P, int noll_first, int K, std::vector<double> &out) {
  const size_t NN = (size_t)P.N * P.N;
  out.assign((size_t)K * NN, 0.0);
  for (int j = 0; j < K; ++j)
    for (size_t i = 0; i < NN; ++i)
      if (P.mask[i]) out[(size_t)j * NN + i] = zernike_noll(noll_first + j, P.rho[i], P.cosphi[i], P.sinphi[i]);
}

void apply_shared_zernike(const HostPupil &P0, const float *coeffs, int K, const std::vector<double> &basis,
                          const float *w0, std::vector<cplx> &base) {
  const size_t NN = (size_t)P0.N * P0.N;
  base.resize(P0.base.size());
  const bool zern = coeffs && K > 0;
#pragma omp parallel for schedule(static)
  for (long long i = 0; i < (long long)NN; ++i) {
    cplx e(1.0, 0.0);
    if ((zern || w0) && P0.mask[i]) {
      double W = w0 ? (double)w0[i] : 0.0;                     // free phase mask W_0 (Eq. 18)
      if (zern)
        for (int j = 0; j < K; ++j) W += (double)coeffs[j] * basis[(size_t)j * NN + i];
      e = cplx(std::cos(W), std::sin(W));
    }
    for (int c = 0; c < P0.C; ++c) {
      const cplx b = P0.base[(size_t)c * NN + i];
      base[(size_t)c * NN + i] = cplx(b.real() * e.real() - b.imag() * e.imag(), b.real() * e.imag() + b.imag() * e.real());
    }
  }
}

void build_bessel_nodes(const psf_plan_desc &d, int n_nodes, BesselNodes &B) {
  B.n = n_nodes;
  B.k = 2.0 * kPi * d.n_immersion / d.wavelength_um;
  const double th_max = std::asin(d.NA / d.n_immersion);
  const double h = th_max / (n_nodes - 1);
  const bool apod = (d.flags & PSF_FLAG_APODIZE) != 0;
  const bool gl = (d.flags & PSF_FLAG_GIBSON_LANNI) != 0;
  const bool env = (d.flags & PSF_FLAG_GAUSSIAN_ENVELOPE) != 0;
  B.sinth.resize(n_nodes);
  B.costh.resize(n_nodes);
  B.A.resize(n_nodes);
  for (int n = 0; n < 3; ++n) B.F[n].resize(n_nodes);
  const bool fres = (d.flags & PSF_FLAG_FRESNEL) != 0 && d.model == PSF_MODEL_VECTORIAL;
  for (int j = 0; j < n_nodes; ++j) {
    const double th = (j == n_nodes - 1) ? th_max : j * h;
    const double st = std::sin(th), ct = std::cos(th);
    const double w = ((j == 0 || j == n_nodes - 1) ? 1.0 : ((j & 1) ? 4.0 : 2.0)) * h / 3.0;   // composite Simpson
    double a = apod ? std::sqrt(ct) : 1.0;
    if (env) a *= std::exp(-(st * st) / (d.envelope_s * d.envelope_s));
    cplx e(1.0, 0.0);
    if (gl) e = std::exp(cplx(0, 1) * gibson_lanni_W(d, st));
    B.sinth[j] = st;
    B.costh[j] = ct;
    B.A[j] = w * a * st * e;
    cplx qs(1, 0), qp(1, 0);
    if (fres) fresnel_q(d, st, qs, qp);      // the phi integral of Eq. 6 with q_s, q_p kept (footnote 3 of the paper)
    B.F[0][j] = qs + qp * ct;
    B.F[1][j] = qp * st;
    B.F[2][j] = qp * ct - qs;
  }
}

void build_dft_phase(const psf_plan_desc &d, std::vector<double> &phi) {
  const int N = d.pupil_n, M = d.out_m;
  const int n = (N + 1) / 2, m = (M + 1) / 2;
  const double kk = 2.0 * kPi * d.NA / d.wavelength_um;   // k * s_max
  phi.assign((size_t)m * n, 0.0);
  for (int mi = 0; mi < m; ++mi) {
    const double x = (mi - 0.5 * (M - 1)) * d.pixel_um;
    for (int qi = 0; qi < n; ++qi) {
      const double u = (double)(2L * qi + 1 - N) / N;
      phi[(size_t)mi * n + qi] = kk * u * x;
    }
  }
}

}  // namespace psf
