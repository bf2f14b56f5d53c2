// Plan-time host tables (fp64): every z-independent factor of the integrand of PAPER.md:116 Eq. 9 / :146 Eq. 15.
// Host-only C++; no CUDA here so that it can be exercised on a machine without a GPU (psf_host_tables).
#pragma once
#include <complex>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/psf.h"

namespace psf {

typedef std::complex<double> cplx;

struct HostPupil {
  int N = 0;                       // pupil grid
  int C = 0;                       // scalar pupils pushed through the DFT stages: 3, 5 for unpolarised, 1 for the scalar model
  double weight[5] = {0, 0, 0, 0, 0};
  double k = 0;                    // 2 pi n_i / lambda
  double s_max = 0;                // NA / n_i
  std::vector<uint8_t> mask;       // [N][N]
  std::vector<double> kappa;       // [N][N]  k cos(theta)
  std::vector<double> rho;         // [N][N]  sin(theta)/s_max
  std::vector<double> cosphi, sinphi;
  std::vector<cplx> base;          // [C][N][N]  prefactor * amp * g_c * exp(i W_static)   (0 outside the disc)
};

// Validates the descriptor (everything that does not need a device). Returns PSF_OK or fills `err`.
psf_status validate_desc(const psf_plan_desc *d, std::string &err);

// Noll index -> (n, m, kind): kind 0 = m==0, 1 = cos, 2 = sin.
void noll_to_nm(int j, int &n, int &m, int &kind);
// Z_j(rho, phi) given (cos phi, sin phi), Noll-normalised.
double zernike_noll(int j, double rho, double cosphi, double sinphi);

// Builds the static pupil. `coeffs` (may be null) is a shared Zernike term folded into W_static.
void build_host_pupil(const psf_plan_desc &d, const float *coeffs, int noll_first, int n_coeffs, HostPupil &out);

// Zernike basis values Z_{noll_first+j} at every in-disc sample: out[j][N][N] (0 outside the disc).
void build_zernike_basis(const HostPupil &P, int noll_first, int K, std::vector<double> &out);

// base[c][i] = P0.base[c][i] * exp(i (sum_j coeffs[j] basis[j][i] + w0[i])): the shared Zernike term and the free
// phase mask w0 ([N][N] radians, may be null) folded into the static pupil.
void apply_shared_zernike(const HostPupil &P0, const float *coeffs, int K, const std::vector<double> &basis,
                          const float *w0, std::vector<cplx> &base);

// Nodes of the spherical (Bessel) parametrisation, Eq. 12-14 (Eq. 5 for the scalar model): composite
// Simpson over theta in [0, theta_max] with n (odd, >= 3) nodes.  A[j] = w_j a(theta_j) sin(theta_j) exp(i W_GL(theta_j))
// with a = apodisation x Gaussian envelope (no 1/s_z here: d Omega = sin(theta) d theta d phi).
struct BesselNodes {
  int n = 0;
  double k = 0;                    // 2 pi n_i / lambda
  std::vector<double> sinth, costh;
  std::vector<cplx> A;
  std::vector<cplx> F[3];          // theta factors of Eq. 12-14: (q_s + q_p cos), q_p sin, (q_p cos - q_s); q = 1 without Fresnel
};
void build_bessel_nodes(const psf_plan_desc &d, int n_nodes, BesselNodes &out);

// Zoomed-DFT phase table: phi[mi][qi] = k s_max u_qi x_mi for mi < m = ceil(M/2), qi < n = ceil(N/2).
void build_dft_phase(const psf_plan_desc &d, std::vector<double> &phi);

}  // namespace psf
