"""psf_propagate_static (include/psf.h, csrc/noalloc.cu): the entry point that allocates nothing - its row -> column scratch and
its DFT table live in a file-scope `static __device__` array of PSF_STATIC_SCRATCH_BYTES - against the existing plan path
(psf_plan_create + psf_compute) on the same pupils, within the bar of the other parity tests (2e-5 of each plane's peak), on
calls in a row that share the array.  Named test_zz_* so that pytest collects it last."""
from dataclasses import replace

import numpy as np
import pytest

import psf_workloads as W
from oracle import psf_oracle as O

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def psf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_03170_b200 as psf
    psf.load_library()
    return psf


def device_pupil(psf, case):
    """The complete pupil field of every plane, as a caller of the plan-free entry point has to bring it: the library's own
    fp64 static pupil (psf_host_tables: prefactor, apodisation, polarisation, Gibson-Lanni and shared Zernike phases) times
    the defocus phasor exp(i kappa z) (Eq. 9), rounded once to complex64."""
    import torch
    ht = psf.host_tables(case, shared_coeffs=case.zernike, noll_first=case.noll_first)
    z = np.asarray(case.z_um, dtype=np.float64)
    P = ht["base"][None, :, :, :] * np.exp(1j * ht["kappa"][None, None, :, :] * z[:, None, None, None])
    return torch.from_numpy(P.astype(np.complex64)).cuda().contiguous(), ht["weights"].astype(np.float32)


def existing_path(psf, case):
    plan = psf.plan_from_case(case)
    I = plan.compute().cpu().numpy().astype(np.float64)
    names = plan.kernel_names
    plan.destroy()
    return I, names


def plane_errors(I, ref):
    Z = len(ref)
    return np.abs(I - ref).reshape(Z, -1).max(1) / ref.reshape(Z, -1).max(1)


def static_case(seed, N, M, Z, pol, **kw):
    return replace(W.small_random_case(seed, pupil_n=N, out_m=M, n_planes=Z, per_plane=False, shifts=False, pol=pol), **kw)


def test_static_scratch_entry_point_matches_the_plan_path_on_calls_in_a_row(psf):
    import torch
    a = static_case(901, 96, 80, 3, W.POL_UNPOLARIZED)          # five pupils; tiles with ragged tails in every dimension
    b = static_case(902, 37, 33, 5, W.POL_CIRC_L)               # odd sizes, smaller than one tile: most of the scratch keeps a's data
    Pa, wa = device_pupil(psf, a)
    Pb, wb = device_pupil(psf, b)
    Ia = torch.empty((3, 80, 80), dtype=torch.float32, device="cuda")
    Ib = torch.empty((5, 33, 33), dtype=torch.float32, device="cuda")
    Ia2 = torch.empty_like(Ia)
    ref_a, names_a = existing_path(psf, a)
    ref_b, names_b = existing_path(psf, b)
    # warm-up: the first call on a device loads the module (its static array) and looks the array's address up
    psf.propagate_static(Pb, 33, b.NA, b.wavelength_um, b.pixel_um, wb, Ib)
    torch.cuda.synchronize()
    Ib.zero_()
    free0 = torch.cuda.mem_get_info()[0]
    # three calls in a row on one stream, no synchronisation between them: they share the static array in stream order
    psf.propagate_static(Pa, 80, a.NA, a.wavelength_um, a.pixel_um, wa, Ia)
    psf.propagate_static(Pb, 33, b.NA, b.wavelength_um, b.pixel_um, wb, Ib)
    psf.propagate_static(Pa, 80, a.NA, a.wavelength_um, a.pixel_um, wa, Ia2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                # nothing was allocated on the device
    ea = plane_errors(Ia.cpu().numpy().astype(np.float64), ref_a)
    eb = plane_errors(Ib.cpu().numpy().astype(np.float64), ref_b)
    assert ea.max() <= TOL, (ea, names_a)
    assert eb.max() <= TOL, (eb, names_b)
    assert torch.equal(Ia, Ia2)                                 # what an earlier call left in the array does not matter
    # and the oracle agrees with both
    assert plane_errors(Ia.cpu().numpy().astype(np.float64), O.stack_T2(a)).max() <= TOL
    assert plane_errors(Ib.cpu().numpy().astype(np.float64), O.stack_T2(b)).max() <= TOL


def test_static_scratch_entry_point_in_several_passes_against_the_tensor_path(psf):
    """12 planes of 256 x 256 with three components: 18.9 MB of row -> column scratch, two passes through the 16 MiB array;
    the existing path for this size is the tcgen05 3xFP16 one."""
    import torch
    c = static_case(903, 256, 256, 12, W.POL_X)
    P, w = device_pupil(psf, c)
    assert P.shape[1] * 256 * 256 * 8 * 12 > psf.STATIC_SCRATCH_BYTES
    ref, names = existing_path(psf, c)
    assert names[0].startswith("k1_pair")
    I = torch.empty((12, 256, 256), dtype=torch.float32, device="cuda")
    for _ in range(2):
        I.zero_()
        psf.propagate_static(P, 256, c.NA, c.wavelength_um, c.pixel_um, w, I)
        torch.cuda.synchronize()
        e = plane_errors(I.cpu().numpy().astype(np.float64), ref)
        assert e.max() <= TOL, e


def test_static_scratch_entry_point_refuses_what_does_not_fit_and_bad_arguments(psf):
    import torch
    big = torch.zeros((1, 2, 1024, 1024), dtype=torch.complex64, device="cuda")      # (2 + 1) * 1024 * 1024 * 8 = 24 MiB > 16 MiB
    out = torch.full((1, 1024, 1024), -1.0, dtype=torch.float32, device="cuda")
    with pytest.raises(psf.PsfError) as ei:
        psf.propagate_static(big, 1024, 1.2, 0.6, 0.05, [1.0, 1.0], out)
    assert "PSF_STATIC_SCRATCH_BYTES" in str(ei.value) and str(psf.STATIC_SCRATCH_BYTES) in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.min()) == -1.0 and float(out.max()) == -1.0                       # nothing was launched
    small = torch.zeros((1, 1, 8, 8), dtype=torch.complex64, device="cuda")
    o8 = torch.empty((1, 8, 8), dtype=torch.float32, device="cuda")
    for bad in (dict(NA=0.0), dict(wavelength_um=float("nan")), dict(pixel_um=-1.0), dict(weights=[float("inf")])):
        kw = dict(NA=1.2, wavelength_um=0.6, pixel_um=0.05, weights=[1.0])
        kw.update(bad)
        with pytest.raises(psf.PsfError):
            psf.propagate_static(small, 8, kw["NA"], kw["wavelength_um"], kw["pixel_um"], kw["weights"], o8)
    six = torch.zeros((1, 6, 8, 8), dtype=torch.complex64, device="cuda")
    with pytest.raises(psf.PsfError):
        psf.propagate_static(six, 8, 1.2, 0.6, 0.05, [1.0] * 6, o8)
    # a large size that fits still runs: (3 + 1) * 512 * 512 * 8 = 8 MiB of the 16
    ok = torch.zeros((1, 3, 512, 512), dtype=torch.complex64, device="cuda")
    ok[0, :, 255:257, 255:257] = 1.0
    o512 = torch.empty((1, 512, 512), dtype=torch.float32, device="cuda")
    psf.propagate_static(ok, 512, 1.2, 0.6, 0.05, [1.0, 1.0, 1.0], o512)
    torch.cuda.synchronize()
    # four in-phase samples around the axis: the on-axis pixels see |4 cos cos|^2 ~ 16 per component
    assert abs(float(o512.max()) - 48.0) < 0.05
