"""Pins for the fp64 oracle (`oracle/psf_oracle.py`): each part is checked against something the paper
or the mathematics fixes, not against itself (SURVEY.md §8(c) "What pins each part").  CPU only."""
import math
from dataclasses import replace

import numpy as np
import pytest
from scipy.special import j1

import psf_workloads as W
from oracle import psf_oracle as O


def _case(**kw):
    base = dict(name="t", NA=1.4, wavelength_um=0.6, n_immersion=1.518, n_sample=1.518, pupil_n=64, out_m=17,
                pixel_um=0.04, z_um=np.array([0.0]), pol=W.POL_X)
    base.update(kw)
    return W.PsfCase(**base)


# ---- G1: rotation matrix (Eq. 6) ------------------------------------------------------------

def test_far_field_matches_textbook_construction():
    """e_inf = q_s (e.n_phi) n_phi + q_p (e.n_rho) n_theta  reproduces all six entries of Eq. 6 (reading G1)."""
    rng = np.random.default_rng(0)
    th = rng.uniform(0, 1.2, 200)
    ph = rng.uniform(-np.pi, np.pi, 200)
    px, py = 0.3 - 0.8j, -0.5 + 0.1j
    qs, qp = 0.9, 1.1
    n_phi = np.stack([-np.sin(ph), np.cos(ph), 0 * ph])
    n_rho = np.stack([np.cos(ph), np.sin(ph), 0 * ph])
    n_th = np.stack([np.cos(th) * np.cos(ph), np.cos(th) * np.sin(ph), -np.sin(th)])
    e = np.stack([px + 0 * ph, py + 0 * ph, 0 * ph])
    ref = qs * np.sum(e * n_phi, 0) * n_phi + qp * np.sum(e * n_rho, 0) * n_th
    g = np.stack(O.far_field_g(np.cos(th), np.sin(th), np.cos(ph), np.sin(ph), px, py, qs, qp))
    assert np.abs(g - ref).max() < 1e-14


def test_far_field_norm_and_axis_limit():
    rng = np.random.default_rng(1)
    th = rng.uniform(0, 1.3, 100)
    ph = rng.uniform(-np.pi, np.pi, 100)
    px, py = (0.6 + 0.2j), (0.1 - 0.7j)
    g = np.stack(O.far_field_g(np.cos(th), np.sin(th), np.cos(ph), np.sin(ph), px, py))
    assert np.allclose(np.sum(np.abs(g) ** 2, 0), abs(px) ** 2 + abs(py) ** 2, atol=1e-14)
    g0 = O.far_field_g(np.array([1.0]), np.array([0.0]), np.array([1.0]), np.array([0.0]), px, py)
    assert np.allclose([g0[0][0], g0[1][0], g0[2][0]], [px, py, 0.0])


# ---- Zernike (reading Z) ------------------------------------------------------------------------------------

def test_noll_table():
    # (n, m, kind) of Noll's ordering, j = 1..15
    exp = [(0, 0, "0"), (1, 1, "cos"), (1, 1, "sin"), (2, 0, "0"), (2, 2, "sin"), (2, 2, "cos"), (3, 1, "sin"),
           (3, 1, "cos"), (3, 3, "sin"), (3, 3, "cos"), (4, 0, "0"), (4, 2, "cos"), (4, 2, "sin"), (4, 4, "cos"),
           (4, 4, "sin")]
    assert [O.noll_to_nm(j) for j in range(1, 16)] == exp


def test_zernike_explicit_forms_and_rim_values():
    rho = np.linspace(0, 1, 11)
    one, zero = np.ones_like(rho), np.zeros_like(rho)
    assert np.allclose(O.zernike_noll(4, rho, one, zero), math.sqrt(3) * (2 * rho ** 2 - 1))
    assert np.allclose(O.zernike_noll(11, rho, one, zero), math.sqrt(5) * (6 * rho ** 4 - 6 * rho ** 2 + 1))
    ph = 0.7
    assert np.allclose(O.zernike_noll(5, rho, math.cos(ph) * one, math.sin(ph) * one),
                       math.sqrt(6) * rho ** 2 * math.sin(2 * ph))
    assert np.allclose(O.zernike_noll(8, rho, math.cos(ph) * one, math.sin(ph) * one),
                       math.sqrt(8) * (3 * rho ** 3 - 2 * rho) * math.cos(ph))
    for j in range(1, 29):
        n, m, kind = O.noll_to_nm(j)
        v = O.zernike_noll(j, np.array([1.0]), np.array([1.0]), np.array([0.0]))[0]
        want = math.sqrt(n + 1) if kind == "0" else (math.sqrt(2 * (n + 1)) if kind == "cos" else 0.0)
        assert abs(v - want) < 1e-12


def test_zernike_orthonormal_on_disc():
    """(1/pi) * integral over the unit disc of Z_j Z_j' = delta_jj' (Gauss-Legendre in rho, uniform in phi)."""
    xr, wr = np.polynomial.legendre.leggauss(40)
    rho = 0.5 * (xr + 1)
    wr = 0.5 * wr
    nphi = 64
    phi = 2 * np.pi * np.arange(nphi) / nphi
    R, P = np.meshgrid(rho, phi, indexing="ij")
    wgt = (wr * rho)[:, None] * (2 * np.pi / nphi) * np.ones_like(P)
    Z = np.stack([O.zernike_noll(j, R, np.cos(P), np.sin(P)) for j in range(1, 23)])
    G = np.einsum("iab,jab,ab->ij", Z, Z, wgt) / np.pi
    assert np.abs(G - np.eye(22)).max() < 1e-12


# ---- brute force on tiny grids: T1 and T2 vs a pure-Python loop ------------------------------------------------

def _brute_force(case, b, iy, ix, jones):
    """Pure-Python restatement of the sum of SURVEY §8(c) for one voxel (no numpy vectorisation)."""
    import cmath
    N, M = case.pupil_n, case.out_m
    k = 2 * math.pi * case.n_immersion / case.wavelength_um
    s_max = case.NA / case.n_immersion
    x = (ix - (M - 1) / 2) * case.pixel_um
    y = (iy - (M - 1) / 2) * case.pixel_um
    xb, yb = (case.shifts_um[b] if case.shifts_um is not None else (0.0, 0.0))
    z = case.z_um[b]
    coef = None
    if case.zernike is not None:
        coef = case.zernike[b] if case.zernike.ndim == 2 else case.zernike
    px, py = jones
    E = [0j, 0j, 0j]
    for qy in range(N):
        for qx in range(N):
            ax, ay = 2 * qx + 1 - N, 2 * qy + 1 - N
            if ax * ax + ay * ay > N * N:
                continue
            sx, sy = s_max * ax / N, s_max * ay / N
            st = math.hypot(sx, sy)
            ct = math.sqrt(1 - st * st)
            cp, sp = (sx / st, sy / st) if st > 0 else (1.0, 0.0)
            c2, s2 = cp * cp - sp * sp, 2 * sp * cp
            g = [0.5 * (((1 - c2) + (1 + c2) * ct) * px + (-1 + ct) * s2 * py),
                 0.5 * ((-1 + ct) * s2 * px + ((1 + c2) + (1 - c2) * ct) * py),
                 0.5 * (-2 * cp * st * px - 2 * sp * st * py)]
            amp = (math.sqrt(ct) if case.apodize else 1.0) / ct
            Wp = 0j
            if case.gibson_lanni:
                k0 = 2 * math.pi / case.wavelength_um
                ni = case.n_immersion
                nis = ni if case.n_immersion_design is None else case.n_immersion_design
                ti = case.particle_depth_um + ni * (-case.particle_depth_um / case.n_sample - case.t_glass_um / case.n_glass
                                                    + case.t_glass_design_um / case.n_glass_design
                                                    + case.t_immersion_design_um / nis)
                a2 = (ni * st) ** 2
                Wp += k0 * (case.particle_depth_um * cmath.sqrt(case.n_sample ** 2 - a2) + ti * cmath.sqrt(ni ** 2 - a2)
                            - case.t_immersion_design_um * cmath.sqrt(nis ** 2 - a2)
                            + case.t_glass_um * cmath.sqrt(case.n_glass ** 2 - a2)
                            - case.t_glass_design_um * cmath.sqrt(case.n_glass_design ** 2 - a2))
            if coef is not None:
                for i, cj in enumerate(coef):
                    Wp += float(cj) * float(O.zernike_noll(case.noll_first + i, np.array([st / s_max]),
                                                          np.array([cp]), np.array([sp]))[0])
            ph = Wp + k * ct * z + k * (sx * (x - float(xb)) + sy * (y - float(yb)))
            e = cmath.exp(1j * ph)
            for c in range(3):
                E[c] += amp * g[c] * e
    pref = -1j * k / (2 * math.pi) * (s_max * 2 / N) ** 2
    return [pref * v for v in E]


@pytest.mark.parametrize("seed,N,M", [(11, 8, 8), (12, 9, 7)])
def test_T1_T2_equal_brute_force_on_tiny_grid(seed, N, M):
    case = W.small_random_case(seed, pupil_n=N, out_m=M, n_planes=2)
    jones = O.jones_vector(case)
    E2 = O.field_T2(case)
    rng = np.random.default_rng(seed)
    for _ in range(6):
        b, iy, ix = int(rng.integers(2)), int(rng.integers(M)), int(rng.integers(M))
        ref = _brute_force(case, b, iy, ix, jones)
        xs = O.out_coords(M, case.pixel_um)
        E1 = O.field_at(case, b, xs[ix], xs[iy])[:, 0]
        scale = max(abs(v) for v in ref)
        assert np.abs(E1 - np.array(ref)).max() <= 1e-12 * scale
        assert np.abs(E2[:, b, iy, ix] - np.array(ref)).max() <= 1e-12 * scale


def test_T2_equals_T1_full_planes_all_options():
    for pol in (W.POL_JONES, W.POL_CIRC_L):
        case = W.small_random_case(5, pupil_n=16, out_m=11, n_planes=3, pol=pol)
        I1 = O.intensity_T1(case)
        I2 = O.stack_T2(case)
        assert np.abs(I1 - I2).max() <= 1e-12 * I1.max()
    case = replace(W.small_random_case(6, pupil_n=14, out_m=10, n_planes=2), pol=W.POL_UNPOLARIZED)
    assert np.abs(O.intensity_T1(case) - O.stack_T2(case)).max() <= 1e-12 * O.stack_T2(case).max()


# ---- closed forms ---------------------------------------------------------------------------------------------

def test_on_axis_focus_closed_form():
    """|E_x(0,0,0)| = (k/2) [2/3 (1-c^{3/2}) + 2/5 (1-c^{5/2})], c = cos(theta_max): from Eq. 12 with sqrt(cos) apodisation.

    The Bessel form is exact to quadrature precision; the Cartesian sum converges to it as N grows."""
    golden = float(open(__file__.replace("test_oracle_pins.py", "golden/on_axis_focus_cfg1.txt")).read().split()[0])
    k = 2 * math.pi * 1.518 / 0.6
    c = math.sqrt(1 - (1.4 / 1.518) ** 2)
    closed = (k / 2) * (2 / 3 * (1 - c ** 1.5) + 2 / 5 * (1 - c ** 2.5))
    assert abs(closed - golden) < 5e-6
    case = _case()
    Eb = O.bessel_field(case, 0.0, 0.0, 0.0)
    assert abs(abs(Eb[0, 0]) - closed) < 1e-10 * closed
    assert abs(Eb[1, 0]) < 1e-12 and abs(Eb[2, 0]) < 1e-12
    err = []
    for N in (64, 256):
        E = O.field_at(replace(case, pupil_n=N), 0, 0.0, 0.0)
        err.append(abs(abs(E[0, 0]) - closed) / closed)
    assert err[0] < 6e-3 and err[1] < err[0] / 4       # quadrature error, falls faster than 1/N


def test_defocus_on_axis_sinc_scalar():
    """Scalar, e_inf = 1, no apodisation, on axis: E(0,0,z) = -i k (e^{ikz} - e^{ikzc}) / (ikz)  (from Eq. 5)."""
    case = _case(apodize=False, z_um=np.array([-1.3, -0.2, 0.45, 2.0]))
    k = 2 * math.pi * 1.518 / 0.6
    c = math.sqrt(1 - (1.4 / 1.518) ** 2)
    for b, z in enumerate(case.z_um):
        closed = -1j * k * (np.exp(1j * k * z) - np.exp(1j * k * z * c)) / (1j * k * z)
        Eb = O.bessel_field(case, 0.0, 0.0, float(z), model="scalar")[0, 0]
        assert abs(Eb - closed) < 1e-9 * k
        Ec = O.field_at(replace(case, pupil_n=256), b, 0.0, 0.0, model="scalar")[0, 0]
        assert abs(Ec - closed) < 5e-3 * k * (1 - c)
    # intensity ~ sinc^2(k z (1-c)/2)
    z = 0.45
    E0 = -1j * k * (1 - c)
    Ez = O.bessel_field(case, 0.0, 0.0, z, model="scalar")[0, 0]
    x = k * z * (1 - c) / 2
    assert abs(abs(Ez / E0) ** 2 - (math.sin(x) / x) ** 2) < 1e-9


def test_vectorial_defocus_on_axis_elementary():
    """Vectorial x-pol without apodisation on axis: E_x = -(ik/2) int_c^1 (1+u) e^{ikzu} du (elementary)."""
    case = _case(apodize=False)
    k = 2 * math.pi * 1.518 / 0.6
    c = math.sqrt(1 - (1.4 / 1.518) ** 2)
    z = 0.37
    a = 1j * k * z
    prim = lambda u: np.exp(a * u) * ((1 + u) / a - 1 / a ** 2)
    closed = -(1j * k / 2) * (prim(1.0) - prim(c))
    Eb = O.bessel_field(case, 0.0, 0.0, z)[0, 0]
    assert abs(Eb - closed) < 1e-9 * abs(closed)
    Ec = O.field_at(replace(case, pupil_n=256, z_um=np.array([z])), 0, 0.0, 0.0)[0, 0]
    assert abs(Ec - closed) < 3e-3 * abs(closed)


def test_airy_limit_scalar_paraxial():
    """PAPER.md:245-253 Eq. 21: scalar, extra cos(theta) factor, z = 0 -> I(r)/I(0) = [2 J1(v)/v]^2, v = 2 pi NA r / lambda."""
    case = _case(apodize=False, NA=0.5, n_immersion=1.0, n_sample=1.0, wavelength_um=0.632, pupil_n=256)
    r = np.linspace(0.02, 2.5, 40)
    v = 2 * math.pi * case.NA * r / case.wavelength_um
    airy = (2 * j1(v) / v) ** 2
    Eb = O.bessel_field(case, np.concatenate([[0.0], r]), 0.0, 0.0, model="scalar", paraxial=True)[0]
    Ib = np.abs(Eb[1:]) ** 2 / abs(Eb[0]) ** 2
    assert np.abs(Ib - airy).max() < 1e-9                      # exact up to Simpson error
    Ec = O.field_at(case, 0, np.concatenate([[0.0], r]), 0.0, model="scalar", paraxial=True)[0]
    Ic = np.abs(Ec[1:]) ** 2 / abs(Ec[0]) ** 2
    assert np.abs(Ic - airy).max() < 2e-3                      # quadrature-limited at N = 256


def test_vectorial_low_NA_tends_to_airy():
    """scalar and vectorial agree at low NA."""
    errs = []
    for NA in (0.05, 0.3):
        case = _case(NA=NA, n_immersion=1.0, n_sample=1.0, wavelength_um=0.632)
        r = np.linspace(0.0, 1.2 * 0.632 / NA, 30)
        v = 2 * math.pi * NA * r / 0.632
        airy = np.where(v > 0, (2 * j1(np.where(v > 0, v, 1)) / np.where(v > 0, v, 1)) ** 2, 1.0)
        E = O.bessel_field(case, r, 0.3, 0.0)
        I = np.sum(np.abs(E) ** 2, 0)
        errs.append(np.abs(I / I[0] - airy).max())
    assert errs[0] < 1e-3 and errs[1] < 3e-2 and errs[0] < errs[1]


# ---- the paper's proven equivalence: Cartesian sum vs Bessel form ----------------------------------------------

def test_bessel_equivalence_config1_and_convergence():
    """Config 1 is axisymmetric end to end: the discrete Cartesian sum must agree with Eq. 11-14 up to the
    quadrature error of the pupil grid, and that error must fall with N."""
    c1 = W.config1()
    planes = [0, 7, 12]
    errs = {}
    for N in (64, 128, 256):
        case = replace(c1, pupil_n=N, out_m=24, pixel_um=0.08)
        Ic = O.stack_T2(case, planes)
        Ib = O.bessel_stack(case, planes, n_nodes=2001)
        errs[N] = max(np.abs(Ic[i] - Ib[i]).max() / Ib[i].max() for i in range(len(planes)))
    assert errs[64] < 2e-2 and errs[128] < 1e-2 and errs[256] < 5e-3
    assert errs[256] < errs[64] / 2


def test_bessel_equivalence_gibson_lanni_with_evanescent_rim():
    """Config-3 optics (GL, n_s < NA: supercritical rim with evanescent decay) at N = 128, three planes."""
    c3 = replace(W.config3(), pupil_n=128, out_m=20, pixel_um=0.1)
    planes = [20, 64, 110]
    Ic = O.stack_T2(c3, planes)
    Ib = O.bessel_stack(c3, planes, n_nodes=4001)
    for i in range(len(planes)):
        assert np.abs(Ic[i] - Ib[i]).max() / Ib.max() < 2e-2


# ---- exact discrete symmetries ------------------------------------------------------------------------------------

def test_discrete_symmetries():
    base = _case(pupil_n=20, out_m=12, z_um=np.array([-0.5, 0.5]))
    Ix = O.stack_T2(base)
    tol = 1e-12 * Ix.max()
    assert np.abs(Ix - Ix[:, :, ::-1]).max() < tol and np.abs(Ix - Ix[:, ::-1, :]).max() < tol   # mirror in x, y
    assert np.abs(Ix[0] - Ix[1]).max() < tol                                                        # I(z) = I(-z)
    Iy = O.stack_T2(replace(base, pol=W.POL_Y))
    assert np.abs(Ix - np.transpose(Iy, (0, 2, 1))).max() < tol                                      # I_x(x,y) = I_y(y,x)
    IL = O.stack_T2(replace(base, pol=W.POL_CIRC_L))
    IR = O.stack_T2(replace(base, pol=W.POL_CIRC_R))
    assert np.abs(IL - IL[:, ::-1, ::-1]).max() < tol                                                # point symmetry
    assert np.abs(IL - IR[:, :, ::-1]).max() < tol                                                   # L(x,y) = R(-x,y)
    assert np.abs(IL - np.transpose(IR, (0, 2, 1))).max() < tol                                      # L(x,y) = R(y,x)
    assert np.abs(0.5 * (Ix + Iy) - 0.5 * (IL + IR)).max() < tol
    IU = O.stack_T2(replace(base, pol=W.POL_UNPOLARIZED))
    assert np.abs(IU - 0.5 * (Ix + Iy)).max() < tol
    # circular mirror symmetry holds only in the continuum: small but non-zero on the square grid
    d = np.abs(IL - IL[:, :, ::-1]).max() / IL.max()
    assert 0 < d < 2e-2


def test_parseval_energy_conservation_across_z():
    """With pixel = lambda N / (2 NA M), M >= N, the zoomed DFT is a (shifted) unitary DFT: sum_xy I[z] =
    M^2 |prefactor|^2 sum_p |P|^2, identical for every z."""
    N, M = 16, 20
    lam, NA = 0.6, 1.4
    case = _case(pupil_n=N, out_m=M, pixel_um=lam * N / (2 * NA * M), z_um=np.linspace(-1.5, 1.5, 5),
                 pol=W.POL_CIRC_L, zernike=np.array([0.2, -0.1, 0.3], dtype=np.float32), noll_first=5)
    I = O.stack_T2(case)
    tot = I.sum(axis=(1, 2))
    assert np.ptp(tot) < 1e-12 * tot.mean()
    pup = O.Pupil(case)
    want = M * M * abs(pup.prefactor) ** 2 * sum(np.sum(np.abs(pup.amp * g) ** 2) for g in pup.g)
    assert abs(tot[0] - want) < 1e-12 * want


# ---- Gibson-Lanni -------------------------------------------------------------------------------------------------

def test_gibson_lanni_matched_indices_is_a_z_shift():
    """Matched indices and design = actual: Eq. 16-17 as printed reduce exactly to defocus by t_s (A3d)."""
    ts = 0.7
    z = np.array([-0.4, 0.1, 0.9])
    gl = _case(pupil_n=24, out_m=10, z_um=z, gibson_lanni=True, particle_depth_um=ts)
    ref = _case(pupil_n=24, out_m=10, z_um=z + ts)
    a, b = O.stack_T2(gl), O.stack_T2(ref)
    assert np.abs(a - b).max() < 1e-11 * b.max()


def test_gibson_lanni_on_axis_phase_closed_form():
    """W_GL(0) = k0 [t_s n_s + t_i n_i - t_i* n_i* + t_g n_g - t_g* n_g*]; and the supercritical branch decays."""
    case = W.small_random_case(3)
    k0 = 2 * math.pi / case.wavelength_um
    ti = O.immersion_thickness(case)
    want = k0 * (case.particle_depth_um * case.n_sample + ti * case.n_immersion
                 - case.t_immersion_design_um * case.n_immersion_design
                 + case.t_glass_um * case.n_glass - case.t_glass_design_um * case.n_glass_design)
    got = O.gibson_lanni_phase(case, np.array([0.0]))[0]
    assert abs(got - want) < 1e-9 * abs(want) and abs(got.imag) == 0
    c3 = W.config3()
    s = np.array([1.33 / 1.518 * 0.999, 1.4 / 1.518])      # just below critical, and the rim
    Wc = O.gibson_lanni_phase(c3, s)
    assert Wc[0].imag == 0 and Wc[1].imag > 0
    decay = math.exp(-2 * math.pi / 0.6 * 2.0 * math.sqrt(1.4 ** 2 - 1.33 ** 2))
    assert abs(math.exp(-Wc[1].imag) - decay) < 1e-12


def test_gl_eq17_paraxial_curvature_is_a_pure_defocus_by_t_s():
    """PAPER.md:154 Eq. 16 with t_i from PAPER.md:167 Eq. 17 as printed, design != actual (every glass / design term
    alive).  In a = n_i sin(theta) each term t sqrt(n^2 - a^2) has the quadratic coefficient -t / (2 n), so
        W_GL(a) = W_GL(0) - (k0 / 2) a^2 [t_s/n_s + t_i/n_i - t_i*/n_i* + t_g/n_g - t_g*/n_g*] + O(a^4),
    and inserting Eq. 17 (t_i/n_i = t_s/n_i - t_s/n_s - t_g/n_g + t_g*/n_g* + t_i*/n_i*) the bracket collapses to
    t_s / n_i for ANY design values: the paraxial curvature of a defocus by t_s in the immersion medium.  A sign slip or
    a swapped index in any glass / design term of Eq. 16 or Eq. 17 changes the bracket by ~t_g/n_g = 100 um against
    t_s/n_i = 1 um.  The coefficient is taken by Richardson-extrapolated second differences (even function of a: the
    h^2 and h^4 error terms are cancelled); the bar 1e-8 is the rounding of W ~ 1e2 rad in the differences."""
    for case in (W.small_random_case(3), replace(W.small_random_case(4), n_glass=1.47, t_glass_um=163.0,
                                                 t_immersion_design_um=140.0, n_immersion_design=1.52, particle_depth_um=3.1)):
        assert (case.n_glass, case.t_glass_um) != (case.n_glass_design, case.t_glass_design_um)
        assert case.n_immersion_design != case.n_immersion and case.t_immersion_um is None
        k0 = 2 * math.pi / case.wavelength_um
        n_i = case.n_immersion

        def w(a):
            v = O.gibson_lanni_phase(case, np.array([a / n_i]))[0]
            assert v.imag == 0.0
            return v.real

        w0 = w(0.0)
        d = lambda h: (w(h) - w0) / (h * h)
        h = 0.05
        r2a, r2b = (4 * d(h / 2) - d(h)) / 3, (4 * d(h / 4) - d(h / 2)) / 3
        c2 = (16 * r2b - r2a) / 15
        want = -0.5 * k0 * case.particle_depth_um / n_i
        assert abs(c2 / want - 1.0) < 1e-8, (c2, want)


# ---- tilt (A9) and Zernike defocus ---------------------------------------------------------------------------------

def test_tilt_is_an_exact_pixel_shift():
    px = 0.05
    base = _case(pupil_n=20, out_m=15, pixel_um=px, z_um=np.array([0.3]), pol=W.POL_CIRC_L,
                 zernike=np.array([0.2, 0.1, -0.15], dtype=np.float32), noll_first=5)
    sh = replace(base, shifts_um=np.array([[2 * px, -3 * px]], dtype=np.float32).astype(np.float32))
    # float32(2*0.05) is not exactly 2 pixels: evaluate the unshifted field at the shifted points instead
    xb, yb = (float(v) for v in sh.shifts_um[0])
    xs = O.out_coords(15, px)
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    want = O.intensity_at(base, 0, (X - xb).ravel(), (Y - yb).ravel()).reshape(15, 15)
    got = O.stack_T2(sh)[0]
    assert np.abs(got - want).max() < 1e-12 * want.max()
    # and a whole-pixel shift is an index shift (up to the fp32 rounding of the shift itself)
    I0 = O.stack_T2(base)[0]
    assert np.abs(got[:-3, 2:] - I0[3:, :-2]).max() < 1e-5 * I0.max()


def test_noll2_noll3_are_exact_lateral_shifts_of_the_combined_aberrated_field():
    """PAPER.md:176 Eq. 18 inside PAPER.md:116 Eq. 9.  Noll 2 and 3 are Z_2 = 2 rho cos(phi) = 2 s_x / s_max and
    Z_3 = 2 s_y / s_max, linear in the pupil coordinates, so c_2 Z_2 + c_3 Z_3 adds to the Fourier kernel
    k (s_x x + s_y y) exactly a lateral shift: with them the field at (x, y) is the field without them at
    (x + 2 c_2 / (k s_max), y + 2 c_3 / (k s_max)).  Checked through the whole combined path -- Gibson-Lanni with
    design != actual, circular input, two more Zernike terms, defocus -- by comparing T2 on the grid (zernike_noll ->
    plane_phase -> matmul sums) with the literal sum T1 at the shifted points without the two terms: this pins the
    non-axisymmetric aberrated combination (the class of configs 2, 4, 5) against something other than itself."""
    base = W.small_random_case(5, pupil_n=22, out_m=13, n_planes=2, pol=W.POL_CIRC_L, per_plane=False, shifts=False)
    c = np.array([0.45, -0.3, 0.25, -0.2], dtype=np.float32)            # Noll 2, 3, 4, 5
    with_tilt = replace(base, zernike=c, noll_first=2)
    c0 = c.copy()
    c0[:2] = 0.0
    without = replace(base, zernike=c0, noll_first=2)
    pup = O.Pupil(base)
    dx, dy = 2.0 * float(c[0]) / (pup.k * pup.s_max), 2.0 * float(c[1]) / (pup.k * pup.s_max)
    xs = O.out_coords(13, base.pixel_um)
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    got = O.stack_T2(with_tilt)
    for b in range(2):
        want = O.intensity_at(without, b, (X + dx).ravel(), (Y + dy).ravel()).reshape(13, 13)
        assert np.abs(got[b] - want).max() < 1e-12 * want.max()
    # the shift is real: about 0.3 and 0.2 pixels here, and the unshifted stack differs at the 10 % level
    assert abs(dx) > 0.2 * base.pixel_um and np.abs(got - O.stack_T2(without)).max() > 0.05 * got.max()
    # per-plane rows take the same route (config 4's mode): row b shifts plane b only
    rows = np.stack([c, c0]).astype(np.float32)
    per = O.stack_T2(replace(base, zernike=rows, noll_first=2))
    assert np.abs(per[0] - got[0]).max() < 1e-12 * got.max()
    assert np.abs(per[1] - O.stack_T2(without)[1]).max() < 1e-12 * got.max()


def test_in_disc_sample_counts():
    """in-disc samples of the midpoint grid (integer rim test) for the config sizes."""
    for N, count in ((64, 3228), (128, 12892), (256, 51468), (512, 205892)):
        assert int(O.disc_mask(N).sum()) == count
    # and by plain integer brute force on a small grid
    N = 10
    cnt = sum(1 for py in range(N) for px in range(N) if (2 * px + 1 - N) ** 2 + (2 * py + 1 - N) ** 2 <= N * N)
    assert int(O.disc_mask(N).sum()) == cnt


def test_single_c4_is_a_quadratic_pupil_phase():
    """A lone Noll-4 coefficient adds c4 sqrt(3) (2 rho^2 - 1) to the phase: check through the field."""
    c4 = 0.37
    case = _case(pupil_n=16, out_m=6, zernike=np.array([c4], dtype=np.float32), noll_first=4)
    pup = O.Pupil(case)
    ph = pup.plane_phase(0).real
    assert np.allclose(ph, float(np.float32(c4)) * math.sqrt(3) * (2 * pup.rho ** 2 - 1), atol=1e-13)


# ---- further correction factors --------------------------------------------------------

def test_gaussian_envelope_on_axis_dawson_closed_form_and_bessel_form():
    """PAPER.md:194 Eq. 20.  Scalar, no apodisation, at focus on axis:
    E = -i k int_c^1 exp(-(1 - u^2)/s^2) du = -i k s [D(1/s) - exp(-(1 - c^2)/s^2) D(c/s)],  D = Dawson's integral."""
    from scipy.special import dawsn
    s = 0.6
    case = _case(apodize=False, envelope_s=s)
    k = 2 * math.pi * 1.518 / 0.6
    c = math.sqrt(1 - (1.4 / 1.518) ** 2)
    closed = -1j * k * s * (dawsn(1 / s) - math.exp(-(1 - c * c) / s ** 2) * dawsn(c / s))
    Eb = O.bessel_field(case, 0.0, 0.0, 0.0, model="scalar")[0, 0]
    assert abs(Eb - closed) < 1e-10 * k
    Ec = O.field_at(replace(case, pupil_n=256), 0, 0.0, 0.0, model="scalar")[0, 0]
    assert abs(Ec - closed) < 3e-3 * abs(closed)
    # the envelope really is a factor of the amplitude: without it the focus amplitude is the plain k (1 - c)
    E0 = O.field_at(replace(case, pupil_n=256, envelope_s=0.0), 0, 0.0, 0.0, model="scalar")[0, 0]
    assert abs(abs(E0) - k * (1 - c)) < 3e-3 * k * (1 - c) and abs(Ec) < 0.5 * abs(E0)
    # vectorial, apodised, off axis and defocused: Cartesian sum against the Bessel form (Eq. 11-14 with a(theta))
    cv = _case(envelope_s=0.8, pupil_n=128, out_m=16, pixel_um=0.09, z_um=np.array([-0.4, 0.3]), pol=W.POL_CIRC_L)
    Ic, Ib = O.stack_T2(cv), O.bessel_stack(cv, n_nodes=2001)
    assert np.abs(Ic - Ib).max() / Ib.max() < 1e-2


def test_phase_mask_vortex_half_moon_and_zernike_equivalence():
    """W_0 of PAPER.md:176 Eq. 18 on the pupil grid."""
    N = 24
    a = (2 * np.arange(N) + 1 - N).astype(np.float64)
    phi = np.arctan2(a[:, None], a[None, :])                       # row = p_y
    base = _case(pupil_n=N, out_m=9, z_um=np.array([0.0, 0.35]), model="scalar")
    # vortex ramp exp(i phi): the grid maps onto itself under a 90 degree turn, which multiplies the pupil by i, so the
    # on-axis field is zero exactly (donut); the ring around it is bright
    Iv = O.stack_T2(replace(base, phase_mask=phi.astype(np.float32)))
    assert Iv[:, 4, 4].max() < 1e-9 * Iv.max() and Iv[0, 4, 6] > 0.05 * Iv.max()
    # half-moon: W_0 = pi on the half pupil s_x > 0 flips the sign of that half -> E is odd in x: zero on the line x = 0
    hm = np.where(a[None, :] > 0, np.pi, 0.0) * np.ones((N, 1))
    Ih = O.stack_T2(replace(base, phase_mask=hm.astype(np.float64)))
    assert Ih[:, :, 4].max() < 1e-24 * Ih.max()
    assert np.abs(Ih - Ih[:, :, ::-1]).max() < 1e-12 * Ih.max()
    # a mask equal to c Z_7 (coma) gives the field of the Zernike path (vectorial, every component)
    vec = _case(pupil_n=N, out_m=7, z_um=np.array([0.2]), pol=W.POL_CIRC_R)
    pup = O.Pupil(vec)
    z7 = np.zeros((N, N))
    z7[pup.py, pup.px] = O.zernike_noll(7, pup.rho, pup.cosphi, pup.sinphi)
    c7 = float(np.float32(0.41))
    Em = O.field_T2(replace(vec, phase_mask=c7 * z7))
    Ez = O.field_T2(replace(vec, zernike=np.array([c7], dtype=np.float32), noll_first=7))
    assert np.abs(Em - Ez).max() < 1e-12 * np.abs(Ez).max()
    # and it adds to the Zernike phase rather than replacing it
    Eb = O.field_T2(replace(vec, phase_mask=c7 * z7, zernike=np.array([c7], dtype=np.float32), noll_first=7))
    E2 = O.field_T2(replace(vec, zernike=np.array([2 * c7], dtype=np.float32), noll_first=7))
    assert np.abs(Eb - E2).max() < 1e-6 * np.abs(E2).max()


def test_scalar_model_is_the_case_default_and_has_one_component():
    """`case.model = "scalar"` selects PAPER.md:70 Eq. 3 in every entry point; T1 = T2; polarisation is ignored."""
    case = _case(pupil_n=12, out_m=5, z_um=np.array([0.3]), model="scalar", pol=W.POL_CIRC_L)
    E2 = O.field_T2(case)
    assert E2.shape[0] == 1
    xs = O.out_coords(5, case.pixel_um)
    E1 = O.field_at(case, 0, xs[3], xs[1])[:, 0]
    assert abs(E1[0] - E2[0, 0, 1, 3]) < 1e-12 * np.abs(E2).max()
    assert np.abs(O.stack_T2(case) - O.stack_T2(replace(case, pol=W.POL_UNPOLARIZED))).max() == 0.0
    assert np.abs(O.stack_T2(case) - O.intensity_T1(case)).max() < 1e-12 * O.stack_T2(case).max()


def test_fresnel_coefficients_textbook_values_and_energy_balance():
    """PAPER.md:102-107 Eq. 7-8 (readings G2, A2) against what the textbook fixes for a single interface: normal
    incidence, Brewster's angle, and T + R = 1 with the reflection coefficients written out independently."""
    n1, n2 = 1.518, 1.33
    one = _case(n_immersion=n1, n_glass=n1, n_sample=n2, NA=1.2)          # glass = immersion: a single interface
    qs0, qp0 = O.fresnel_q(one, np.array([0.0]))
    assert abs(qs0[0] - 2 * n1 / (n1 + n2)) < 1e-15 and abs(qp0[0] - 2 * n1 / (n1 + n2)) < 1e-15
    thB = math.atan(n2 / n1)                                               # Brewster: no p reflection, t_p = n1 / n2
    _, qpB = O.fresnel_q(one, np.array([math.sin(thB)]))
    assert abs(qpB[0] - n1 / n2) < 1e-14
    th = np.linspace(0.0, math.asin(n2 / n1) * 0.999, 50)                  # below the critical angle
    c1 = np.cos(th)
    c2 = np.sqrt(1 - (n1 * np.sin(th) / n2) ** 2)
    qs, qp = O.fresnel_q(one, np.sin(th))
    Rs = ((n1 * c1 - n2 * c2) / (n1 * c1 + n2 * c2)) ** 2
    Rp = ((n2 * c1 - n1 * c2) / (n2 * c1 + n1 * c2)) ** 2
    T = n2 * c2 / (n1 * c1)
    assert np.abs(T * np.abs(qs) ** 2 + Rs - 1).max() < 1e-13 and np.abs(T * np.abs(qp) ** 2 + Rp - 1).max() < 1e-13
    # two interfaces multiply; matched indices transmit everything
    two = _case(n_immersion=1.518, n_glass=1.46, n_sample=1.33, NA=1.2)
    s = np.array([0.3, 0.7])
    a = O.fresnel_q(_case(n_immersion=1.518, n_glass=1.518, n_sample=1.46, NA=1.2), s)
    b = O.fresnel_q(_case(n_immersion=1.46, n_glass=1.46, n_sample=1.33, NA=1.2), s * 1.518 / 1.46)
    qs2, qp2 = O.fresnel_q(two, s)
    assert np.abs(qs2 - a[0] * b[0]).max() < 1e-15 and np.abs(qp2 - a[1] * b[1]).max() < 1e-15
    m = O.fresnel_q(_case(n_glass=1.518), np.array([0.1, 0.9]))
    assert np.abs(m[0] - 1).max() == 0 and np.abs(m[1] - 1).max() == 0
    # past the critical angle the coefficients are complex with |q_s| <= 2 (total internal reflection: phase only in r)
    qs_t, _ = O.fresnel_q(one, np.array([0.95]))
    assert abs(qs_t[0].imag) > 0.1


def test_fresnel_through_the_field_cartesian_equals_bessel_form():
    """With Fresnel factors the phi integral of Eq. 6 gives (q_s + q_p cos), q_p sin, (q_p cos - q_s) in Eq. 12-14;
    the discrete Cartesian sum with the complex q_s, q_p inside Eq. 6 must agree with that Bessel form (axisymmetric
    case with index mismatch, supercritical rim included)."""
    case = replace(W.config3(), pupil_n=512, out_m=18, pixel_um=0.1, z_um=np.array([-2.6, -2.0]), fresnel=True, n_glass=1.46,
                   pol=W.POL_CIRC_R)
    Ib = O.bessel_stack(case, n_nodes=4001)
    Ic = O.stack_T2(case)
    err = np.abs(Ic - Ib).max() / Ib.max()
    coarse = np.abs(O.stack_T2(replace(case, pupil_n=128)) - Ib).max() / Ib.max()
    assert err < 2e-3 and coarse > 5 * err                  # quadrature error of the pupil grid, falling with N
    I0 = O.stack_T2(replace(case, fresnel=False))
    assert np.abs(Ic - I0).max() / I0.max() > 5e-2          # the coefficients do change the PSF


@pytest.mark.parametrize("pol", [W.POL_JONES, W.POL_UNPOLARIZED])
def test_adjoint_gradients_match_finite_differences_of_the_forward_sum(pol):
    """`grad_T2` (adjoint formula) against central differences of the pinned forward sum `stack_T2`: per-plane Zernike
    rows, shared coefficients (column sums) and the defocus of every plane; every option on (Gibson-Lanni with the
    evanescent rim, shifts, complex Jones vector / unpolarised)."""
    rng = np.random.default_rng(5)
    case = replace(W.small_random_case(101, pupil_n=14, out_m=11, n_planes=3, pol=pol), envelope_s=0.9)
    G = rng.standard_normal((3, 11, 11))
    L = lambda c: float(np.sum(G * O.stack_T2(c)))
    dz, dc = O.grad_T2(case, G)
    h = 1e-6
    for b in range(3):
        zp, zm = case.z_um.copy(), case.z_um.copy()
        zp[b] += h; zm[b] -= h
        fd = (L(replace(case, z_um=zp)) - L(replace(case, z_um=zm))) / (2 * h)
        assert abs(fd - dz[b]) < 1e-6 * np.abs(dz).max()
        for j in (0, 3, 5):
            cp, cm = case.zernike.astype(np.float64), case.zernike.astype(np.float64)
            cp[b, j] += h; cm[b, j] -= h
            fd = (L(replace(case, zernike=cp)) - L(replace(case, zernike=cm))) / (2 * h)
            assert abs(fd - dc[b, j]) < 1e-6 * np.abs(dc).max()
    # shared coefficients: the gradient is the column sum over the planes
    sh = replace(case, zernike=case.zernike[0].astype(np.float64), shifts_um=None)
    _, dcs = O.grad_T2(sh, G)
    cp, cm = sh.zernike.copy(), sh.zernike.copy()
    cp[2] += h; cm[2] -= h
    fd = (L(replace(sh, zernike=cp)) - L(replace(sh, zernike=cm))) / (2 * h)
    assert abs(fd - dcs[:, 2].sum()) < 1e-6 * np.abs(dcs.sum(0)).max()
