"""fp64 CPU oracle for the Fourier-parametrised vectorial Richards-Wolf z-stack.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` /
`--impl reference` legs of `bench.py` may import this module.  It shares no code with the CUDA
path (`paper_2502_03170_b200/`), and neither imports the other; only the seeded input records of
`psf_workloads` are common to both.

What it computes (plain definition): for every output voxel, the Riemann sum
over the in-disc samples of an N x N midpoint pupil grid of the Cartesian Richards-Wolf integral
(Eq. 9) with the correction factors of PAPER.md:146 Eq. 15:

    E_c(x,y; b) = -(i k / 2 pi) (s_max du)^2  sum_{p in D}  amp(theta) g_c(theta,phi)
                    exp( i [ W(p) + k cos(theta) z_b + k ( s_x (x - x_b) + s_y (y - y_b) ) ] )
    I = sum_c |E_c|^2

Tiers
  * `field_at` / `intensity_T1`  (T1, authoritative): the formula above, literally, one complex
    exponential per (voxel, pupil sample).
  * `stack_T2` (T2): the same finite sum summed over p_x first and p_y second with tabulated
    exp(i k s x) factors (two `numpy.matmul` calls per plane; no FFT, no chirp-z).  Must equal T1
    to ~1e-12; it is the timed CPU baseline.
  * `bessel_field` : the spherical parametrisation PAPER.md:126-138 Eq. 11-14 by composite
    Simpson quadrature -- used only to pin T1/T2 on axisymmetric cases (the paper's proven
    equivalence).

Pins: every function here is checked in tests/test_oracle_pins.py against something other than
itself (closed forms, the Bessel form, the Airy pattern, exact discrete symmetries, Parseval,
pure-Python brute force).  The combined non-axisymmetric aberrated result (the class of configs 2, 4, 5)
is pinned by an exact identity: Noll 2 / 3 terms inside the full combination (Gibson-Lanni with design !=
actual, circular input, further Zernike terms, defocus) are a lateral shift by 2 c / (k s_max), checked T2 on
the grid against T1 at the shifted points; `immersion_thickness` and every glass / design term of
`gibson_lanni_phase` by the paraxial curvature of Eq. 16 + Eq. 17, which is -k0 t_s / (2 n_i) for any design
values; the in-disc counts of SURVEY.md section 8 are asserted.

Further correction factors, each a factor of the static pupil: the scalar model
`case.model = "scalar"` (Eq. 3, e_inf = e_inc = 1, one component), the Gaussian envelope
`case.envelope_s` (Eq. 20, a factor of amp(theta)), and the free phase mask `case.phase_mask`
(W_0 of PAPER.md:176 Eq. 18, radians on the pupil grid, added to W).  Pins: Dawson-function closed form of the
on-axis focus amplitude and the Bessel form (envelope), exact zeros of vortex / half-moon masks, a mask equal
to a Zernike term (phase mask), Airy / sinc closed forms (scalar).

Readings of the paper taken where it is silent/garbled are those of SURVEY.md §8(c) (G1, A1-A10, Z)
and are listed in DESIGN.md.
"""
from __future__ import annotations

import math

import numpy as np

# --------------------------------------------------------------------------------------------
# Geometry
# --------------------------------------------------------------------------------------------

def pupil_numerators(N: int) -> np.ndarray:
    """Integer numerators 2p+1-N of the midpoint grid u_p = (2p+1-N)/N (reading A4)."""
    return 2 * np.arange(N, dtype=np.int64) + 1 - N


def disc_mask(N: int) -> np.ndarray:
    """In-disc mask [p_y, p_x]: s_x^2+s_y^2 <= s_max^2, tested in integers (A5)."""
    a = pupil_numerators(N)
    return (a[None, :] ** 2 + a[:, None] ** 2) <= N * N


def out_coords(M: int, pixel_um: float) -> np.ndarray:
    """Output coordinates x_m = (m - (M-1)/2) * pixel (reading A6)."""
    return (np.arange(M, dtype=np.float64) - (M - 1) / 2.0) * pixel_um


def jones_vector(case):
    """Unit Jones vector (px, py) of the incident field (reading A8)."""
    r = 1.0 / math.sqrt(2.0)
    if case.pol == "x":
        return 1.0 + 0j, 0.0 + 0j
    if case.pol == "y":
        return 0.0 + 0j, 1.0 + 0j
    if case.pol == "circ_l":
        return r + 0j, 1j * r
    if case.pol == "circ_r":
        return r + 0j, -1j * r
    if case.pol == "jones":
        j = case.jones
        return complex(j[0], j[1]), complex(j[2], j[3])
    raise ValueError(f"no single Jones vector for pol={case.pol!r}")


# --------------------------------------------------------------------------------------------
# Far field (Eq. 6, reading G1) and correction factors (Eq. 15-19)
# --------------------------------------------------------------------------------------------

def far_field_g(costh, sinth, cosphi, sinphi, px, py, q_s=1.0, q_p=1.0):
    """e_inf = g(theta, phi; px, py): the 3x2 polarisation-rotation matrix of Eq. 6 applied to (px, py).

    Third row of the y column is the detached '-2 q_p sin(phi) sin(theta)' of PAPER.md:97 (G1).
    Returns (g_x, g_y, g_z), complex arrays.
    """
    cos2phi = cosphi * cosphi - sinphi * sinphi
    sin2phi = 2.0 * sinphi * cosphi
    col_x = (q_s * (1.0 - cos2phi) + q_p * (1.0 + cos2phi) * costh,
             (-q_s + q_p * costh) * sin2phi,
             -2.0 * q_p * cosphi * sinth)
    col_y = ((-q_s + q_p * costh) * sin2phi,
             q_s * (1.0 + cos2phi) + q_p * (1.0 - cos2phi) * costh,
             -2.0 * q_p * sinphi * sinth)
    return tuple(0.5 * (cx * px + cy * py) for cx, cy in zip(col_x, col_y))


def fresnel_q(case, sinth):
    """(q_s, q_p) of PAPER.md:102-107 Eq. 7-8 (reading G2: Eq. 7 is q_s, Eq. 8 is q_p): the product over the interfaces
    immersion -> glass -> sample (focusing direction, reading A2) of
        q_s^j = 2 n_j cos(theta_j) / (n_j cos(theta_j) + n_{j+1} cos(theta_{j+1}))
        q_p^j = 2 n_j cos(theta_j) / (n_{j+1} cos(theta_j) + n_j cos(theta_{j+1}))
    with Snell's law n_j sin(theta_j) = n_i sin(theta) and the principal complex root for cos(theta_j) past a
    critical angle (the branch of A3b).  Complex arrays."""
    n = (case.n_immersion, case.n_glass, case.n_sample)
    a = case.n_immersion * np.asarray(sinth, dtype=np.float64)
    cos = [_csqrt(1.0 - (a / nj) ** 2) for nj in n]
    q_s = np.ones_like(cos[0])
    q_p = np.ones_like(cos[0])
    for j in range(len(n) - 1):
        q_s = q_s * (2.0 * n[j] * cos[j] / (n[j] * cos[j] + n[j + 1] * cos[j + 1]))
        q_p = q_p * (2.0 * n[j] * cos[j] / (n[j + 1] * cos[j] + n[j] * cos[j + 1]))
    return q_s, q_p


def _csqrt(v):
    """Principal complex square root of a real array: +i sqrt(|v|) for v < 0 (reading A3b)."""
    return np.sqrt(np.asarray(v, dtype=np.float64).astype(np.complex128))


def immersion_thickness(case) -> float:
    """t_i from the focusing condition PAPER.md:167 Eq. 17, as printed (leading bare t_s; A3d)."""
    if case.t_immersion_um is not None:
        return float(case.t_immersion_um)
    n_i = case.n_immersion
    n_i_star = n_i if case.n_immersion_design is None else case.n_immersion_design
    return case.particle_depth_um + n_i * (-case.particle_depth_um / case.n_sample
                                           - case.t_glass_um / case.n_glass
                                           + case.t_glass_design_um / case.n_glass_design
                                           + case.t_immersion_design_um / n_i_star)


def gibson_lanni_phase(case, sinth):
    """Complex W_GL(theta), Eq. 16 (all five terms), k0 = 2 pi / lambda.

    sin(theta) is in the immersion medium (A3a).  Square roots of negative arguments take the
    principal complex root, so exp(i W) carries the evanescent decay past the critical angle (A3b).
    """
    k0 = 2.0 * math.pi / case.wavelength_um
    n_i = case.n_immersion
    n_i_star = n_i if case.n_immersion_design is None else case.n_immersion_design
    t_i = immersion_thickness(case)
    a2 = (n_i * np.asarray(sinth, dtype=np.float64)) ** 2
    opd = (case.particle_depth_um * _csqrt(case.n_sample ** 2 - a2)
           + t_i * _csqrt(n_i ** 2 - a2)
           - case.t_immersion_design_um * _csqrt(n_i_star ** 2 - a2)
           + case.t_glass_um * _csqrt(case.n_glass ** 2 - a2)
           - case.t_glass_design_um * _csqrt(case.n_glass_design ** 2 - a2))
    return k0 * opd


def noll_to_nm(j: int):
    """Noll index j >= 1 -> (n, m, kind) with kind in {'0','cos','sin'} (reading Z)."""
    if j < 1:
        raise ValueError("Noll index starts at 1")
    n = int((math.isqrt(8 * (j - 1) + 1) - 1) // 2)
    k = j - n * (n + 1) // 2
    m = 2 * (k // 2) if n % 2 == 0 else 2 * ((k - 1) // 2) + 1
    if m == 0:
        return n, 0, "0"
    return n, m, ("cos" if j % 2 == 0 else "sin")


def zernike_noll(j: int, rho, cosphi, sinphi):
    """Z_j(rho, phi), Noll-normalised (unit rms on the unit disc; PAPER.md:174-176 'orthonormal')."""
    n, m, kind = noll_to_nm(j)
    rho = np.asarray(rho, dtype=np.float64)
    R = np.zeros_like(rho)
    for s in range((n - m) // 2 + 1):
        c = ((-1) ** s * math.factorial(n - s)
             / (math.factorial(s) * math.factorial((n + m) // 2 - s) * math.factorial((n - m) // 2 - s)))
        R = R + c * rho ** (n - 2 * s)
    if kind == "0":
        return math.sqrt(n + 1.0) * R
    e = (np.asarray(cosphi, dtype=np.float64) + 1j * np.asarray(sinphi, dtype=np.float64)) ** m
    ang = e.real if kind == "cos" else e.imag
    return math.sqrt(2.0 * (n + 1.0)) * R * ang


# --------------------------------------------------------------------------------------------
# Pupil samples: everything that multiplies the Fourier kernel, per in-disc sample
# --------------------------------------------------------------------------------------------

def _model(case, model):
    """`model` argument of the public functions: None -> the case's own model."""
    return getattr(case, "model", "vectorial") if model is None else model


class Pupil:
    """Per in-disc sample tables (fp64) for one case: the factors of Eq. 9/15 that do not depend on (x,y,z)."""

    def __init__(self, case, model=None, paraxial=False, jones=None):
        model = _model(case, model)
        N = case.pupil_n
        self.N = N
        self.k = 2.0 * math.pi * case.n_immersion / case.wavelength_um   # k = 2 pi n / lambda, n = n_i (A3a)
        self.s_max = case.NA / case.n_immersion
        a = pupil_numerators(N)
        mask = disc_mask(N)
        self.mask = mask
        py, px = np.nonzero(mask)
        self.py, self.px = py, px
        u = a.astype(np.float64) / N
        self.u = u
        self.s_x = self.s_max * u[px]
        self.s_y = self.s_max * u[py]
        sin2 = self.s_x ** 2 + self.s_y ** 2
        self.sinth = np.sqrt(sin2)
        self.costh = np.sqrt(1.0 - sin2)
        with np.errstate(invalid="ignore", divide="ignore"):
            self.cosphi = np.where(self.sinth > 0, self.s_x / self.sinth, 1.0)   # phi := 0 at the origin
            self.sinphi = np.where(self.sinth > 0, self.s_y / self.sinth, 0.0)
        self.rho = self.sinth / self.s_max
        # amplitude: apodisation (Eq. 19) x the 1/s_z Jacobian of Eq. 9 (always on, A10)
        amp = (np.sqrt(self.costh) if case.apodize else 1.0) / self.costh
        if paraxial:
            amp = amp * self.costh      # the extra s_z = cos(theta) of PAPER.md:253 (Airy benchmark)
        if getattr(case, "envelope_s", 0.0) > 0.0:
            amp = amp * np.exp(-sin2 / case.envelope_s ** 2)      # Gaussian envelope, Eq. 20
        self.amp = amp
        # far field
        if model == "vectorial":
            pxj, pyj = jones_vector(case) if jones is None else jones
            q_s, q_p = fresnel_q(case, self.sinth) if getattr(case, "fresnel", False) else (1.0, 1.0)
            self.g = far_field_g(self.costh, self.sinth, self.cosphi, self.sinphi, pxj, pyj, q_s, q_p)
        elif model == "scalar":             # PAPER.md:63 e_inf = e_inc (= 1)
            self.g = (np.ones_like(self.costh, dtype=np.complex128),)
        else:
            raise ValueError(model)
        # static phase W: Gibson-Lanni (complex) + shared Zernike
        W = np.zeros(len(px), dtype=np.complex128)
        if case.gibson_lanni:
            W = W + gibson_lanni_phase(case, self.sinth)
        if getattr(case, "phase_mask", None) is not None:          # W_0 of PAPER.md:176 Eq. 18, sampled on the pupil grid
            W = W + np.asarray(case.phase_mask, dtype=np.float64)[py, px]
        self.W_static = W
        self.case = case
        self._zbasis = None
        # prefactor -(i f k / 2 pi) with f = 1 (A1) times the quadrature weight (s_max du)^2, du = 2/N
        self.prefactor = -1j * self.k / (2.0 * math.pi) * (self.s_max * 2.0 / N) ** 2

    def zernike_basis(self):
        case = self.case
        if self._zbasis is None:
            K = case.zernike.shape[-1]
            self._zbasis = np.stack([zernike_noll(case.noll_first + i, self.rho, self.cosphi, self.sinphi)
                                     for i in range(K)], axis=0)      # [K, D]
        return self._zbasis

    def plane_phase(self, b: int):
        """Complex phase of plane b that does not depend on (x, y): W + k cos(theta) z_b - k(s_x x_b + s_y y_b)."""
        case = self.case
        ph = self.W_static + self.k * self.costh * float(case.z_um[b])
        if case.zernike is not None:
            c = case.zernike[b] if case.per_plane_zernike else case.zernike
            ph = ph + np.asarray(c, dtype=np.float64) @ self.zernike_basis()      # Eq. 18, radians
        if case.shifts_um is not None:
            xb, yb = (float(v) for v in case.shifts_um[b])
            ph = ph - self.k * (self.s_x * xb + self.s_y * yb)                    # A9
        return ph


def _pupils(case, model, paraxial):
    """One Pupil per incoherent input (unpolarised = x and y inputs, each weighted 1/2; A8)."""
    model = _model(case, model)
    if case.pol == "unpolarized" and model == "vectorial":
        return [(0.5, Pupil(case, model, paraxial, jones=(1.0 + 0j, 0j))),
                (0.5, Pupil(case, model, paraxial, jones=(0j, 1.0 + 0j)))]
    return [(1.0, Pupil(case, model, paraxial))]


# --------------------------------------------------------------------------------------------
# T1: literal sum
# --------------------------------------------------------------------------------------------

def field_at(case, plane, x_um, y_um, model=None, paraxial=False, jones=None, chunk=2048):
    """T1: E_c at arbitrary points (x, y) of plane(s) `plane` -- the literal double sum.

    plane, x_um, y_um broadcast to a common 1-D shape V.  Returns complex [C, V].
    One complex exponential per (voxel, in-disc pupil sample).
    """
    pup = Pupil(case, model, paraxial, jones)
    plane, x_um, y_um = np.broadcast_arrays(np.atleast_1d(plane), np.atleast_1d(x_um), np.atleast_1d(y_um))
    V = plane.size
    C = len(pup.g)
    out = np.zeros((C, V), dtype=np.complex128)
    A = np.stack([pup.amp * g for g in pup.g], axis=1)                  # [D, C]
    for b in np.unique(plane):
        sel = np.nonzero(plane == b)[0]
        phb = pup.plane_phase(int(b))                                   # [D] complex
        for s in range(0, len(sel), chunk):
            ii = sel[s:s + chunk]
            phase = (phb[None, :]
                     + pup.k * (x_um[ii, None] * pup.s_x[None, :] + y_um[ii, None] * pup.s_y[None, :]))
            out[:, ii] = (np.exp(1j * phase) @ A).T
    return pup.prefactor * out


def intensity_at(case, plane, x_um, y_um, **kw):
    """T1 intensity sum_c |E_c|^2 at points; unpolarised = 1/2 (I_x + I_y)."""
    model = _model(case, kw.get("model"))
    if case.pol == "unpolarized" and model == "vectorial":
        ix = np.sum(np.abs(field_at(case, plane, x_um, y_um, jones=(1.0 + 0j, 0j), **kw)) ** 2, axis=0)
        iy = np.sum(np.abs(field_at(case, plane, x_um, y_um, jones=(0j, 1.0 + 0j), **kw)) ** 2, axis=0)
        return 0.5 * (ix + iy)
    return np.sum(np.abs(field_at(case, plane, x_um, y_um, **kw)) ** 2, axis=0)


def intensity_T1(case, planes=None, **kw):
    """T1 on the full M x M output grid of the given planes -> [len(planes), M, M]."""
    M = case.out_m
    xs = out_coords(M, case.pixel_um)
    planes = range(case.n_planes) if planes is None else planes
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    out = []
    for b in planes:
        out.append(intensity_at(case, int(b), X.ravel(), Y.ravel(), **kw).reshape(M, M))
    return np.stack(out, axis=0)


def voxel_intensity(case, b, iy, ix, **kw):
    """T1 intensity at output-grid voxels (plane b, row iy, column ix) given by index arrays."""
    xs = out_coords(case.out_m, case.pixel_um)
    return intensity_at(case, np.asarray(b), xs[np.asarray(ix)], xs[np.asarray(iy)], **kw)


# --------------------------------------------------------------------------------------------
# T2: the same finite sum, summed over p_x then p_y (two matrix products per plane and component)
# --------------------------------------------------------------------------------------------

def field_T2(case, planes=None, model=None, paraxial=False, jones=None):
    """T2: E[c, b, m_y, m_x] for the given planes (complex128)."""
    pup = Pupil(case, model, paraxial, jones)
    N, M = case.pupil_n, case.out_m
    xs = out_coords(M, case.pixel_um)
    Ax = np.exp(1j * pup.k * pup.s_max * np.outer(xs, pup.u))          # [m, p]: exp(i k s_max u_p x_m)
    planes = list(range(case.n_planes)) if planes is None else list(planes)
    C = len(pup.g)
    E = np.empty((C, len(planes), M, M), dtype=np.complex128)
    for ib, b in enumerate(planes):
        e = np.exp(1j * pup.plane_phase(int(b)))
        for c in range(C):
            P = np.zeros((N, N), dtype=np.complex128)                    # zero outside the disc
            P[pup.py, pup.px] = pup.amp * pup.g[c] * e
            T = P @ Ax.T                                                 # sum over p_x -> [p_y, m_x]
            E[c, ib] = Ax @ T                                            # sum over p_y -> [m_y, m_x]
    return pup.prefactor * E


def stack_T2(case, planes=None, model=None, paraxial=False):
    """T2 intensity stack [len(planes), M, M] (float64)."""
    model = _model(case, model)
    if case.pol == "unpolarized" and model == "vectorial":
        ix = np.sum(np.abs(field_T2(case, planes, model, paraxial, jones=(1.0 + 0j, 0j))) ** 2, axis=0)
        iy = np.sum(np.abs(field_T2(case, planes, model, paraxial, jones=(0j, 1.0 + 0j))) ** 2, axis=0)
        return 0.5 * (ix + iy)
    return np.sum(np.abs(field_T2(case, planes, model, paraxial)) ** 2, axis=0)


# --------------------------------------------------------------------------------------------
# Spherical (Bessel) parametrisation, Eq. 11-14 -- cross-check only
# --------------------------------------------------------------------------------------------

def _simpson_weights(n_nodes: int, h: float) -> np.ndarray:
    if n_nodes % 2 == 0 or n_nodes < 3:
        raise ValueError("composite Simpson needs an odd number of nodes >= 3")
    w = np.ones(n_nodes)
    w[1:-1:2] = 4.0
    w[2:-1:2] = 2.0
    return w * h / 3.0


def bessel_integrals(case, r_um, z_um: float, model=None, paraxial=False, n_nodes=4001):
    """I_0, I_1, I_2 of PAPER.md:131-137 Eq. 12-14 (without e_inc) at radii r_um (1-D) and one defocus z,
    by composite Simpson over theta in [0, theta_max].  Scalar model: the single integral of Eq. 5.

    Axisymmetric corrections enter as a(theta) exp(i W(theta)) (Eq. 15, 209).
    """
    from scipy.special import jv
    model = _model(case, model)
    r_um = np.atleast_1d(np.asarray(r_um, dtype=np.float64))
    k = 2.0 * math.pi * case.n_immersion / case.wavelength_um
    th_max = math.asin(case.NA / case.n_immersion)
    th = np.linspace(0.0, th_max, n_nodes)
    w = _simpson_weights(n_nodes, th[1] - th[0])
    st, ct = np.sin(th), np.cos(th)
    a = (np.sqrt(ct) if case.apodize else np.ones_like(ct)).astype(np.complex128)
    if paraxial:
        a = a * ct
    if getattr(case, "envelope_s", 0.0) > 0.0:
        a = a * np.exp(-(st / case.envelope_s) ** 2)                       # PAPER.md:194 Eq. 20
    if case.gibson_lanni:
        a = a * np.exp(1j * gibson_lanni_phase(case, st))
    a = a * np.exp(1j * k * float(z_um) * ct)                              # exp(i k z cos(theta))
    arg = k * np.outer(r_um, st)                                           # k rho sin(theta)
    if model == "scalar":
        return (jv(0, arg) @ (w * a * st),)
    # with Fresnel coefficients the phi integral of Eq. 6 gives (q_s + q_p cos), q_p sin, (q_p cos - q_s) in place of
    # (1 + cos), sin, (cos - 1): footnote 3 applied to the entries of Eq. 6
    q_s, q_p = fresnel_q(case, st) if getattr(case, "fresnel", False) else (1.0, 1.0)
    I0 = jv(0, arg) @ (w * a * st * (q_s + q_p * ct))                      # Eq. 12
    I1 = jv(1, arg) @ (w * a * st * (q_p * st))                            # Eq. 13
    I2 = jv(2, arg) @ (w * a * st * (q_p * ct - q_s))                      # Eq. 14
    return I0, I1, I2


def bessel_field(case, r_um, varphi, z_um: float, model=None, paraxial=False, jones=None, n_nodes=4001):
    """E at cylindrical points (r, varphi) of the plane at defocus z from the Bessel integrals (Eq. 5 / Eq. 11).

    Valid for axisymmetric pupils only (no Zernike, no shifts).  f = 1 (A1).
    r_um, varphi broadcast to a common 1-D shape V.  Returns complex [C, V].
    """
    if case.zernike is not None or case.shifts_um is not None or getattr(case, "phase_mask", None) is not None:
        raise ValueError("Bessel form needs an axisymmetric pupil")
    model = _model(case, model)
    r_um, varphi = np.broadcast_arrays(np.atleast_1d(r_um).astype(float), np.atleast_1d(varphi).astype(float))
    k = 2.0 * math.pi * case.n_immersion / case.wavelength_um
    ru, inv = np.unique(np.round(r_um, 12), return_inverse=True)           # equal radii share their integrals
    ints = [v[inv] for v in bessel_integrals(case, ru, z_um, model, paraxial, n_nodes)]
    if model == "scalar":
        return (-1j * k * ints[0])[None, :]                                # Eq. 5
    I0, I1, I2 = ints
    pxj, pyj = jones_vector(case) if jones is None else jones
    c2, s2 = np.cos(2 * varphi), np.sin(2 * varphi)
    Ex = (I0 * pxj - I2 * pxj * c2) - I2 * pyj * s2                        # Eq. 11, row 1
    Ey = -I2 * pxj * s2 + (I0 * pyj + I2 * pyj * c2)                       # row 2
    Ez = -2j * I1 * pxj * np.cos(varphi) - 2j * I1 * pyj * np.sin(varphi)  # row 3
    return (-1j * k / 2.0) * np.stack([Ex, Ey, Ez], axis=0)


def bessel_stack(case, planes=None, model=None, paraxial=False, n_nodes=4001):
    """Bessel-form intensity on the output grid [len(planes), M, M]."""
    M = case.out_m
    xs = out_coords(M, case.pixel_um)
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    r = np.hypot(X, Y).ravel()
    vp = np.arctan2(Y, X).ravel()
    planes = range(case.n_planes) if planes is None else planes
    model = _model(case, model)
    out = []
    for b in planes:
        z = float(case.z_um[b])
        if case.pol == "unpolarized" and model == "vectorial":
            ix = np.sum(np.abs(bessel_field(case, r, vp, z, model, paraxial, (1.0 + 0j, 0j), n_nodes)) ** 2, 0)
            iy = np.sum(np.abs(bessel_field(case, r, vp, z, model, paraxial, (0j, 1.0 + 0j), n_nodes)) ** 2, 0)
            I = 0.5 * (ix + iy)
        else:
            I = np.sum(np.abs(bessel_field(case, r, vp, z, model, paraxial, None, n_nodes)) ** 2, axis=0)
        out.append(I.reshape(M, M))
    return np.stack(out, axis=0)


# --------------------------------------------------------------------------------------------
# Adjoint: gradients of a linear functional of the intensity
# --------------------------------------------------------------------------------------------

def grad_T2(case, G, planes=None, model=None):
    """Gradients of L = sum_{b,y,x} G[b,y,x] I[b,y,x] with respect to the per-plane pupil phase parameters, by the
    adjoint of the finite sum of `field_T2` (the paper's motivation for a differentiable PSF).

    With Q_c[p] = amp g_c exp(i phi_b[p]) the pupil of plane b and phi_b = W + k cos(theta) z_b + sum_j c_bj Z_j - ...,
        dI/dphi[p] = sum_c 2 Re( conj(E_c) i Q_c[p] A(x, p) ),   A(x, p) = prefactor exp(i k (s_x x + s_y y)),
        dL/dphi_b[p] = -2 sum_c Im( Q_c[p] B_c[p] ),   B_c[p] = sum_x G conj(E_c(x)) A(x, p)   (the back-projection),
        dL/dz_b = sum_p k cos(theta_p) dL/dphi_b[p],     dL/dc_bj = sum_p Z_j[p] dL/dphi_b[p].
    Unpolarised light: the two incoherent inputs, each with weight 1/2.
    Returns (dL_dz [len(planes)], dL_dc [len(planes), K] or None without Zernike terms).  A shared coefficient's
    gradient is the sum of its column over the planes."""
    model = _model(case, model)
    planes = list(range(case.n_planes)) if planes is None else list(planes)
    G = np.asarray(G, dtype=np.float64)
    N, M = case.pupil_n, case.out_m
    K = 0 if case.zernike is None else case.zernike.shape[-1]
    dz = np.zeros(len(planes))
    dc = np.zeros((len(planes), K)) if K else None
    for wgt, pup in _pupils(case, model, False):
        xs = out_coords(M, case.pixel_um)
        Ax = np.exp(1j * pup.k * pup.s_max * np.outer(xs, pup.u))          # [m, p]
        for ib, b in enumerate(planes):
            e = np.exp(1j * pup.plane_phase(int(b)))
            S = np.zeros(len(pup.px))
            for g in pup.g:
                Qd = pup.amp * g * e                                         # in-disc samples
                P = np.zeros((N, N), dtype=np.complex128)
                P[pup.py, pup.px] = Qd
                E = pup.prefactor * (Ax @ (P @ Ax.T))                        # [m_y, m_x]
                H = wgt * G[ib] * np.conj(E)
                B = pup.prefactor * (Ax.T @ H @ Ax)                          # [p_y, p_x] = sum_x H A(x, p)
                S += -2.0 * np.imag(Qd * B[pup.py, pup.px])
            dz[ib] += np.sum(pup.k * pup.costh * S)
            if K:
                dc[ib] += pup.zernike_basis() @ S
    return dz, dc
