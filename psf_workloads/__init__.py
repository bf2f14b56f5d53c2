"""Seeded synthetic input generators for the five BASELINE.json workloads.

This module serves BOTH the fp64 CPU oracle (`oracle/`) and the CUDA path
(`paper_2502_03170_b200/`).  It holds no arithmetic of the method (no pupil, no phase,
no DFT): only plain parameter records and the seeded random draws that fill them,
following the recipe of SURVEY.md §8(d) "Synthetic inputs" (the paper evaluates on no
public dataset; its workloads are PSFs generated from parameters).

Values that cross the C-ABI as fp32 (Zernike coefficients, emitter shifts) are drawn in
fp64, rounded to fp32 here, and both sides consume exactly those fp32 values ("inputs are
shared as bytes").  z lists stay fp64; the per-emitter z of config 4 is rounded to fp32 and
widened back, so that both sides see the same double.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# polarisation states (names only; the Jones vectors are defined by each side, A8)
POL_X = "x"
POL_Y = "y"
POL_CIRC_L = "circ_l"      # (1, +i)/sqrt(2)
POL_CIRC_R = "circ_r"      # (1, -i)/sqrt(2)
POL_JONES = "jones"        # custom complex (px, py)
POL_UNPOLARIZED = "unpolarized"  # 1/2 (I_x + I_y)


@dataclass
class PsfCase:
    """Plain description of one PSF job (lengths in micrometres)."""
    name: str
    NA: float
    wavelength_um: float
    n_immersion: float
    n_sample: float
    pupil_n: int
    out_m: int
    pixel_um: float
    z_um: np.ndarray                      # float64 [Z]
    pol: str = POL_X
    jones: tuple = (1.0, 0.0, 0.0, 0.0)   # re px, im px, re py, im py (POL_JONES only)
    apodize: bool = True
    gibson_lanni: bool = False
    # Gibson-Lanni parameters (PAPER.md:154 Eq. 16, :167 Eq. 17); design = actual by default (A3c)
    particle_depth_um: float = 0.0        # t_s
    n_glass: float = 1.5
    t_glass_um: float = 170.0
    n_glass_design: float = 1.5
    t_glass_design_um: float = 170.0
    n_immersion_design: Optional[float] = None   # None -> n_immersion
    t_immersion_design_um: float = 150.0
    t_immersion_um: Optional[float] = None       # None -> Eq. 17 as printed
    # Zernike phase (radians), Noll indices noll_first .. noll_first+K-1
    noll_first: int = 4
    zernike: Optional[np.ndarray] = None  # float32 [K] (shared) or [Z, K] (per plane)
    # per-plane lateral emitter positions (config 4), float32 [Z, 2] = (x_b, y_b)
    shifts_um: Optional[np.ndarray] = None
    seed: Optional[int] = None
    # remaining correction factors of the paper; all fold into the static pupil
    model: str = "vectorial"              # "vectorial" (Eq. 9) or "scalar" (Eq. 3: e_inf = e_inc = 1)
    envelope_s: float = 0.0               # s_env of the Gaussian envelope exp(-sin^2 theta / s_env^2) (Eq. 20); 0 = off
    fresnel: bool = False                 # q_s, q_p of PAPER.md:102-107 Eq. 7-8 over immersion -> glass -> sample (reading A2)
    phase_mask: Optional[np.ndarray] = None   # W_0 of PAPER.md:176 Eq. 18: float32 [N, N] radians on the pupil grid (row = p_y)

    @property
    def n_planes(self) -> int:
        return int(len(self.z_um))

    @property
    def per_plane_zernike(self) -> bool:
        return self.zernike is not None and self.zernike.ndim == 2

    def voxels(self) -> int:
        return self.n_planes * self.out_m * self.out_m

    def with_planes(self, idx) -> "PsfCase":
        """Sub-case holding only the planes `idx` (keeps per-plane rows aligned)."""
        idx = np.asarray(idx, dtype=np.int64)
        kw = dict(z_um=np.ascontiguousarray(self.z_um[idx]))
        if self.per_plane_zernike:
            kw["zernike"] = np.ascontiguousarray(self.zernike[idx])
        if self.shifts_um is not None:
            kw["shifts_um"] = np.ascontiguousarray(self.shifts_um[idx])
        return replace(self, **kw)


def config1() -> PsfCase:
    """Smallest vectorial PSF (BASELINE.json configs[0])."""
    return PsfCase(name="cfg1_small", NA=1.4, wavelength_um=0.6, n_immersion=1.518, n_sample=1.518,
                   pupil_n=64, out_m=64, pixel_um=0.040, z_um=np.linspace(-1.0, 1.0, 16), pol=POL_X)


def config2() -> PsfCase:
    """Seeded random Zernike aberrations, circular polarisation (configs[1])."""
    rng = np.random.default_rng(1002)
    c = (0.1 * rng.standard_normal(12)).astype(np.float32)
    return PsfCase(name="cfg2_zernike", NA=1.4, wavelength_um=0.52, n_immersion=1.518, n_sample=1.518,
                   pupil_n=128, out_m=128, pixel_um=0.030, z_um=np.linspace(-2.0, 2.0, 64),
                   pol=POL_CIRC_L, noll_first=4, zernike=c, seed=1002)


def config3() -> PsfCase:
    """Gibson-Lanni index mismatch (configs[2])."""
    return PsfCase(name="cfg3_gibson_lanni", NA=1.4, wavelength_um=0.6, n_immersion=1.518, n_sample=1.33,
                   pupil_n=256, out_m=256, pixel_um=0.025, z_um=np.linspace(-3.0, 3.0, 128), pol=POL_X,
                   gibson_lanni=True, particle_depth_um=2.0, n_glass=1.5, t_glass_um=170.0,
                   n_glass_design=1.5, t_glass_design_um=170.0, t_immersion_design_um=150.0)


def config4(n_emitters: int = 4096) -> PsfCase:
    """SMLM emitter batch: independent single-plane PSFs (configs[3])."""
    rng = np.random.default_rng(1004)
    x = rng.uniform(-0.2, 0.2, 4096)
    y = rng.uniform(-0.2, 0.2, 4096)
    z = rng.uniform(-0.8, 0.8, 4096)
    c = 0.05 * rng.standard_normal((4096, 8))
    x, y, z, c = x[:n_emitters], y[:n_emitters], z[:n_emitters], c[:n_emitters]
    shifts = np.stack([x, y], axis=1).astype(np.float32)
    return PsfCase(name="cfg4_smlm_batch", NA=1.45, wavelength_um=0.67, n_immersion=1.518, n_sample=1.518,
                   pupil_n=64, out_m=32, pixel_um=0.100,
                   z_um=z.astype(np.float32).astype(np.float64), pol=POL_X,
                   noll_first=4, zernike=np.ascontiguousarray(c.astype(np.float32)),
                   shifts_um=np.ascontiguousarray(shifts), seed=1004)


def config5(n_planes: int = 256) -> PsfCase:
    """Large stack: unpolarised, Zernike + Gibson-Lanni (configs[4])."""
    rng = np.random.default_rng(1005)
    c = (0.08 * rng.standard_normal(18)).astype(np.float32)
    return PsfCase(name="cfg5_large_stack", NA=1.4, wavelength_um=0.5, n_immersion=1.518, n_sample=1.33,
                   pupil_n=512, out_m=512, pixel_um=0.020, z_um=np.linspace(-4.0, 4.0, n_planes),
                   pol=POL_UNPOLARIZED, gibson_lanni=True, particle_depth_um=5.0,
                   noll_first=4, zernike=c, seed=1005)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def get_config(i: int) -> PsfCase:
    return CONFIGS[int(i)]()


def small_random_case(seed: int, pupil_n: int = 12, out_m: int = 9, n_planes: int = 3,
                      pol: str = POL_JONES, gibson_lanni: bool = True, per_plane: bool = True,
                      shifts: bool = True) -> PsfCase:
    """A tiny seeded case with every option on (odd/even sizes, ragged tiles) for brute-force tests."""
    rng = np.random.default_rng(seed)
    z = rng.uniform(-1.0, 1.0, n_planes).astype(np.float32).astype(np.float64)
    k = 6
    zern = (0.3 * rng.standard_normal((n_planes, k) if per_plane else k)).astype(np.float32)
    sh = rng.uniform(-0.15, 0.15, (n_planes, 2)).astype(np.float32) if shifts else None
    jones = tuple(rng.standard_normal(4))
    nrm = float(np.sqrt(sum(v * v for v in jones)))
    jones = tuple(v / nrm for v in jones)
    return PsfCase(name=f"small_{seed}", NA=1.35, wavelength_um=0.55, n_immersion=1.518,
                   n_sample=1.33 if gibson_lanni else 1.518, pupil_n=pupil_n, out_m=out_m, pixel_um=0.07,
                   z_um=z, pol=pol, jones=jones, gibson_lanni=gibson_lanni, particle_depth_um=1.5,
                   n_glass=1.52, t_glass_um=171.0, n_glass_design=1.5, t_glass_design_um=170.0,
                   n_immersion_design=1.515, t_immersion_design_um=150.0,
                   noll_first=2, zernike=zern, shifts_um=sh, seed=seed)
