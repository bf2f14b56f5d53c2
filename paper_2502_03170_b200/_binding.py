"""ctypes binding of libpsf_b200.so (include/psf.h).  Argument marshalling only: every step of the hot path runs in
the library's CUDA kernels.  There is no CPU fallback: a missing library or device raises."""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import build as _build

PSF_OK, PSF_ERR_INVALID_ARG, PSF_ERR_UNSUPPORTED, PSF_ERR_ALLOC, PSF_ERR_CUDA, PSF_ERR_STATE = range(6)
STATUS_NAMES = {0: "PSF_OK", 1: "PSF_ERR_INVALID_ARG", 2: "PSF_ERR_UNSUPPORTED", 3: "PSF_ERR_ALLOC",
                4: "PSF_ERR_CUDA", 5: "PSF_ERR_STATE"}
POL = {"x": 0, "y": 1, "circ_l": 2, "circ_r": 3, "jones": 4, "unpolarized": 5}
FLAG_APODIZE, FLAG_GIBSON_LANNI, FLAG_FRESNEL, FLAG_GAUSSIAN_ENVELOPE = 1, 2, 4, 8
MODEL = {"vectorial": 0, "scalar": 1}
PREC = {"auto": 0, "3xtf32": 1, "fp32": 2, "3xf16": 3, "czt_fft": 4}

EXPORTS = ["psf_plan_create", "psf_set_zernike", "psf_set_shifts", "psf_set_phase_mask", "psf_compute", "psf_plan_destroy",
           "psf_spherical_prepare", "psf_compute_spherical", "psf_gradients",
           "psf_last_error", "psf_launches_per_compute", "psf_path_name", "psf_host_tables",
           "psf_profile_enable", "psf_profile_read", "psf_last_upload_bytes", "psf_plan_tune", "psf_grad_terms", "psf_kernel_names", "psf_grad_path_name",
           "psf_propagate_static"]
TUNE_TC_PAIR_MASK, TUNE_TC_SCRATCH_MB, TUNE_K1P_HANDOFF, TUNE_K1P_DEFER, TUNE_TC_FUSED, TUNE_SMLM, TUNE_GRAD_TENSOR, TUNE_K1P_ASPLIT, TUNE_FUSED_WINDOW, TUNE_DEVICE_REFRESH, TUNE_PDL, TUNE_K1P_WAITFIRST = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12


class PsfError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class psf_plan_desc(C.Structure):
    _fields_ = [("NA", C.c_double), ("wavelength_um", C.c_double), ("n_immersion", C.c_double),
                ("n_sample", C.c_double), ("particle_depth_um", C.c_double), ("n_glass", C.c_double),
                ("t_glass_um", C.c_double), ("n_glass_design", C.c_double), ("t_glass_design_um", C.c_double),
                ("n_immersion_design", C.c_double), ("t_immersion_design_um", C.c_double),
                ("t_immersion_um", C.c_double), ("pupil_n", C.c_int), ("out_m", C.c_int), ("pixel_um", C.c_double),
                ("n_planes", C.c_int), ("z_um", C.POINTER(C.c_double)), ("pol", C.c_int), ("jones", C.c_double * 4),
                ("flags", C.c_uint), ("precision", C.c_int), ("device", C.c_int),
                ("model", C.c_int), ("envelope_s", C.c_double)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def load_library(build_if_missing: bool = True):
    """Loads libpsf_b200.so (building it with nvcc first if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.needs_build():
        _build.build()
    if not os.path.exists(_build.LIB):
        raise ImportError(f"{_build.LIB} is missing: build it with `python -m paper_2502_03170_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(_build.LIB)
    P = C.c_void_p
    lib.psf_plan_create.argtypes = [C.POINTER(psf_plan_desc), C.POINTER(P)]
    lib.psf_plan_create.restype = C.c_int
    lib.psf_set_zernike.argtypes = [P, C.POINTER(C.c_float), C.c_int, C.c_int, C.c_int]
    lib.psf_set_zernike.restype = C.c_int
    lib.psf_set_shifts.argtypes = [P, C.POINTER(C.c_float)]
    lib.psf_set_shifts.restype = C.c_int
    lib.psf_set_phase_mask.argtypes = [P, C.POINTER(C.c_float)]
    lib.psf_set_phase_mask.restype = C.c_int
    lib.psf_compute.argtypes = [P, P, P, P]
    lib.psf_gradients.argtypes = [P, P, P, P, P]
    lib.psf_gradients.restype = C.c_int
    lib.psf_spherical_prepare.argtypes = [P, C.c_int]
    lib.psf_spherical_prepare.restype = C.c_int
    lib.psf_compute_spherical.argtypes = [P, P, P]
    lib.psf_compute_spherical.restype = C.c_int
    lib.psf_compute.restype = C.c_int
    lib.psf_plan_destroy.argtypes = [P]
    lib.psf_plan_destroy.restype = C.c_int
    lib.psf_last_error.argtypes = [P]
    lib.psf_last_error.restype = C.c_char_p
    lib.psf_launches_per_compute.argtypes = [P]
    lib.psf_launches_per_compute.restype = C.c_int
    lib.psf_path_name.argtypes = [P]
    lib.psf_path_name.restype = C.c_char_p
    lib.psf_profile_enable.argtypes = [P, C.c_int]
    lib.psf_profile_enable.restype = C.c_int
    lib.psf_profile_read.argtypes = [P, C.POINTER(C.c_float), C.POINTER(C.c_int)]
    lib.psf_profile_read.restype = C.c_int
    lib.psf_last_upload_bytes.argtypes = [P]
    lib.psf_last_upload_bytes.restype = C.c_longlong
    lib.psf_plan_tune.argtypes = [P, C.c_int, C.c_longlong]
    lib.psf_plan_tune.restype = C.c_int
    lib.psf_kernel_names.argtypes = [P]
    lib.psf_kernel_names.restype = C.c_char_p
    lib.psf_grad_path_name.argtypes = [P]
    lib.psf_grad_path_name.restype = C.c_char_p
    lib.psf_grad_terms.argtypes = [P]
    lib.psf_grad_terms.restype = C.c_int
    lib.psf_host_tables.argtypes = [C.POINTER(psf_plan_desc), C.POINTER(C.c_float), C.c_int, C.c_int,
                                    C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                    C.POINTER(C.c_double), C.POINTER(C.c_ubyte)]
    lib.psf_host_tables.restype = C.c_int
    lib.psf_propagate_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                         C.c_double, C.POINTER(C.c_float), C.c_void_p]
    lib.psf_propagate_static.restype = C.c_int
    _lib = lib
    return lib


def _nan_if_none(v):
    return float("nan") if v is None else float(v)


def make_desc(case, device: int = 0, precision: str = "auto"):
    """psf_plan_desc from any object with the attributes of psf_workloads.PsfCase.  Returns (desc, keepalive)."""
    z = np.ascontiguousarray(np.asarray(case.z_um, dtype=np.float64))
    d = psf_plan_desc()
    d.NA, d.wavelength_um = float(case.NA), float(case.wavelength_um)
    d.n_immersion, d.n_sample = float(case.n_immersion), float(case.n_sample)
    d.particle_depth_um = float(case.particle_depth_um)
    d.n_glass, d.t_glass_um = float(case.n_glass), float(case.t_glass_um)
    d.n_glass_design, d.t_glass_design_um = float(case.n_glass_design), float(case.t_glass_design_um)
    d.n_immersion_design = _nan_if_none(case.n_immersion_design)
    d.t_immersion_design_um = float(case.t_immersion_design_um)
    d.t_immersion_um = _nan_if_none(case.t_immersion_um)
    d.pupil_n, d.out_m, d.pixel_um = int(case.pupil_n), int(case.out_m), float(case.pixel_um)
    d.n_planes = int(z.shape[0])
    d.z_um = z.ctypes.data_as(C.POINTER(C.c_double))
    d.pol = POL[case.pol]
    d.jones = (C.c_double * 4)(*[float(v) for v in case.jones])
    env = float(getattr(case, "envelope_s", 0.0) or 0.0)
    d.flags = ((FLAG_APODIZE if case.apodize else 0) | (FLAG_GIBSON_LANNI if case.gibson_lanni else 0) |
               (FLAG_GAUSSIAN_ENVELOPE if env > 0 else 0) | (FLAG_FRESNEL if getattr(case, "fresnel", False) else 0))
    d.model = MODEL[getattr(case, "model", "vectorial")]
    d.envelope_s = env
    d.precision = PREC[precision]
    d.device = int(device)
    return d, z


def _fptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


class PsfPlan:
    """Owns one psf_plan.  `compute` enqueues on a CUDA stream and returns device tensors."""

    def __init__(self, case, device: int = 0, precision: str = "auto"):
        self._lib = load_library()
        self._h = C.c_void_p()
        desc, keep = make_desc(case, device, precision)
        st = self._lib.psf_plan_create(C.byref(desc), C.byref(self._h))
        if st != PSF_OK:
            raise PsfError(st, self._lib.psf_last_error(None).decode())
        self.n_planes, self.out_m, self.pupil_n = desc.n_planes, desc.out_m, desc.pupil_n
        self.device = int(device)
        self.n_components = 1 if getattr(case, "model", "vectorial") == "scalar" else 3
        self.unpolarized = case.pol == "unpolarized" and self.n_components == 3

    def _check(self, st):
        if st != PSF_OK:
            raise PsfError(st, self._lib.psf_last_error(self._h).decode())

    def set_zernike(self, coeffs, noll_first: int = 4):
        """coeffs: None, float32 [K] (shared) or [n_planes, K] (per plane)."""
        if coeffs is None:
            self._check(self._lib.psf_set_zernike(self._h, None, 1, 0, 0))
            return
        a = np.ascontiguousarray(np.asarray(coeffs, dtype=np.float32))
        if a.ndim == 2 and a.shape[0] != self.n_planes:
            raise ValueError("per-plane Zernike rows must match n_planes")
        self._check(self._lib.psf_set_zernike(self._h, _fptr(a), int(noll_first), int(a.shape[-1]), int(a.ndim == 2)))

    def set_phase_mask(self, w0_rad):
        """Free phase mask W_0: None or float32 [N, N] radians on the pupil grid (row = p_y)."""
        if w0_rad is None:
            self._check(self._lib.psf_set_phase_mask(self._h, None))
            return
        a = np.ascontiguousarray(np.asarray(w0_rad, dtype=np.float32))
        if a.shape != (self.pupil_n, self.pupil_n):
            raise ValueError("phase mask must be [pupil_n, pupil_n]")
        self._check(self._lib.psf_set_phase_mask(self._h, _fptr(a)))

    def set_shifts(self, xy_um):
        if xy_um is None:
            self._check(self._lib.psf_set_shifts(self._h, None))
            return
        a = np.ascontiguousarray(np.asarray(xy_um, dtype=np.float32))
        if a.shape != (self.n_planes, 2):
            raise ValueError("shifts must be [n_planes, 2]")
        self._check(self._lib.psf_set_shifts(self._h, _fptr(a)))

    def compute_raw(self, stream_ptr: int, intensity_ptr: int, field_ptr: int = 0):
        """psf_compute with raw pointers (device memory, 16-byte aligned)."""
        self._check(self._lib.psf_compute(self._h, C.c_void_p(stream_ptr), C.c_void_p(intensity_ptr),
                                          C.c_void_p(field_ptr) if field_ptr else None))

    def compute(self, intensity=None, field=None, want_field: bool = False, stream=None):
        import torch
        dev = torch.device("cuda", self.device)
        Z, M = self.n_planes, self.out_m
        if intensity is None:
            intensity = torch.empty((Z, M, M), dtype=torch.float32, device=dev)
        if want_field and field is None:
            field = torch.empty((self.n_components, Z, M, M), dtype=torch.complex64, device=dev)
        for t, shape, dt in ((intensity, (Z, M, M), torch.float32), (field, (self.n_components, Z, M, M), torch.complex64)):
            if t is not None and (tuple(t.shape) != shape or t.dtype != dt or not t.is_contiguous() or not t.is_cuda):
                raise ValueError(f"output must be a contiguous CUDA tensor of shape {shape} and dtype {dt}")
        s = torch.cuda.current_stream(dev) if stream is None else stream
        self.compute_raw(s.cuda_stream, intensity.data_ptr(), field.data_ptr() if field is not None else 0)
        return (intensity, field) if field is not None else intensity

    def compute_spherical(self, n_nodes: int = 2001, intensity=None, stream=None):
        """Spherical (Bessel) parametrisation, axisymmetric pupils only; prepares its tables on first use or when
        n_nodes changes."""
        import torch
        dev = torch.device("cuda", self.device)
        if getattr(self, "_sph_nodes", None) != int(n_nodes):
            self._check(self._lib.psf_spherical_prepare(self._h, int(n_nodes)))
            self._sph_nodes = int(n_nodes)
        Z, M = self.n_planes, self.out_m
        if intensity is None:
            intensity = torch.empty((Z, M, M), dtype=torch.float32, device=dev)
        s = torch.cuda.current_stream(dev) if stream is None else stream
        self._check(self._lib.psf_compute_spherical(self._h, C.c_void_p(s.cuda_stream), C.c_void_p(intensity.data_ptr())))
        return intensity

    def gradients(self, dL_dI, n_terms: int | None = None, stream=None):
        """Adjoint: dL_dI is a CUDA float32 tensor [Z, M, M]; returns (dL_dz [Z], dL_dc [Z, K] or None), float64 CUDA
        tensors.  K = the number of Zernike terms currently set (psf_grad_terms); n_terms, if given, must be 0 (defocus
        gradients only) or K: the library writes rows of K values."""
        import torch
        dev = torch.device("cuda", self.device)
        Z, M = self.n_planes, self.out_m
        K = int(self._lib.psf_grad_terms(self._h))
        if n_terms is None:
            n_terms = K
        if n_terms not in (0, K):
            raise ValueError(f"n_terms must be 0 or the number of Zernike terms set ({K})")
        if tuple(dL_dI.shape) != (Z, M, M) or dL_dI.dtype != torch.float32 or not dL_dI.is_contiguous() or not dL_dI.is_cuda:
            raise ValueError("dL_dI must be a contiguous CUDA float32 tensor [n_planes, M, M]")
        dz = torch.empty((Z,), dtype=torch.float64, device=dev)
        dc = torch.empty((Z, n_terms), dtype=torch.float64, device=dev) if n_terms > 0 else None
        s = torch.cuda.current_stream(dev) if stream is None else stream
        self._check(self._lib.psf_gradients(self._h, C.c_void_p(s.cuda_stream), C.c_void_p(dL_dI.data_ptr()),
                                            C.c_void_p(dz.data_ptr()), C.c_void_p(dc.data_ptr()) if dc is not None else None))
        return dz, dc

    def tune(self, knob: int, value: int):
        """psf_plan_tune: TUNE_TC_PAIR_MASK / TUNE_TC_SCRATCH_MB (tests and A/B runs)."""
        self._check(self._lib.psf_plan_tune(self._h, int(knob), int(value)))

    def profile_enable(self, enable: bool = True):
        self._check(self._lib.psf_profile_enable(self._h, int(bool(enable))))

    def profile_read(self):
        """(stage_ms[4], launches[4]) of the last compute; the caller must have synchronised its stream."""
        ms = (C.c_float * 4)()
        ln = (C.c_int * 4)()
        self._check(self._lib.psf_profile_read(self._h, ms, ln))
        return list(ms), list(ln)

    @property
    def last_upload_bytes(self) -> int:
        return int(self._lib.psf_last_upload_bytes(self._h))

    @property
    def launches_per_compute(self) -> int:
        return int(self._lib.psf_launches_per_compute(self._h))

    @property
    def grad_path(self) -> str:
        return self._lib.psf_grad_path_name(self._h).decode()

    @property
    def kernel_names(self) -> list:
        return [k for k in self._lib.psf_kernel_names(self._h).decode().split(",") if k]

    @property
    def path(self) -> str:
        return self._lib.psf_path_name(self._h).decode()

    def destroy(self):
        if self._h:
            self._lib.psf_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def plan_from_case(case, device: int = 0, precision: str = "auto") -> PsfPlan:
    """Plan with the case's Zernike coefficients and shifts applied."""
    plan = PsfPlan(case, device, precision)
    if case.zernike is not None:
        plan.set_zernike(case.zernike, case.noll_first)
    if case.shifts_um is not None:
        plan.set_shifts(case.shifts_um)
    if getattr(case, "phase_mask", None) is not None:
        plan.set_phase_mask(case.phase_mask)
    return plan


STATIC_SCRATCH_BYTES = 16 << 20


def propagate_static(pupil, out_m: int, NA: float, wavelength_um: float, pixel_um: float, weights, intensity, stream=None):
    """psf_propagate_static: pupil = CUDA complex64 (or float32 [..., 2]) tensor [Z, C, N, N], intensity = CUDA float32 tensor
    [Z, out_m, out_m] that the CALLER provides (the entry point allocates nothing, and neither does this wrapper)."""
    import torch
    lib = load_library()
    if pupil.dtype == torch.complex64:
        Z, Cn, N, N2 = pupil.shape
    else:
        Z, Cn, N, N2, two = pupil.shape
        if two != 2 or pupil.dtype != torch.float32:
            raise ValueError("pupil must be complex64 [Z, C, N, N] or float32 [Z, C, N, N, 2]")
    if N != N2 or not pupil.is_cuda or not pupil.is_contiguous():
        raise ValueError("pupil must be a contiguous CUDA tensor [Z, C, N, N]")
    if tuple(intensity.shape) != (Z, out_m, out_m) or intensity.dtype != torch.float32 or not intensity.is_cuda or \
            not intensity.is_contiguous() or intensity.device != pupil.device:
        raise ValueError("intensity must be a contiguous CUDA float32 tensor [Z, out_m, out_m] on the pupil's device")
    w = np.ascontiguousarray(np.asarray(weights, dtype=np.float32))
    if w.shape != (Cn,):
        raise ValueError("weights must have one entry per component")
    with torch.cuda.device(pupil.device):
        s = torch.cuda.current_stream(pupil.device) if stream is None else stream
        st = lib.psf_propagate_static(C.c_void_p(s.cuda_stream), C.c_void_p(pupil.data_ptr()), int(Z), int(Cn), int(N), int(out_m),
                                      float(NA), float(wavelength_um), float(pixel_um), _fptr(w), C.c_void_p(intensity.data_ptr()))
    if st != PSF_OK:
        raise PsfError(st, lib.psf_last_error(None).decode())
    return intensity


def host_tables(case, shared_coeffs=None, noll_first: int = 4):
    """psf_host_tables: the library's plan-time fp64 static pupil (no device needed)."""
    lib = load_library()
    desc, keep = make_desc(case)
    N = desc.pupil_n
    base = np.zeros((5, N, N, 2), dtype=np.float64)
    kappa = np.zeros((N, N), dtype=np.float64)
    mask = np.zeros((N, N), dtype=np.uint8)
    w = np.zeros(5, dtype=np.float64)
    nc = C.c_int(0)
    cp, K = None, 0
    if shared_coeffs is not None:
        a = np.ascontiguousarray(np.asarray(shared_coeffs, dtype=np.float32))
        cp, K = _fptr(a), int(a.shape[0])
    st = lib.psf_host_tables(C.byref(desc), cp, int(noll_first), K, C.byref(nc),
                             w.ctypes.data_as(C.POINTER(C.c_double)), base.ctypes.data_as(C.POINTER(C.c_double)),
                             kappa.ctypes.data_as(C.POINTER(C.c_double)), mask.ctypes.data_as(C.POINTER(C.c_ubyte)))
    if st != PSF_OK:
        raise PsfError(st, lib.psf_last_error(None).decode())
    c = nc.value
    return dict(n_components=c, weights=w[:c].copy(), base=base[:c, :, :, 0] + 1j * base[:c, :, :, 1],
                kappa=kappa, mask=mask.astype(bool))
