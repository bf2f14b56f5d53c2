"""Small GPU cases, one per kernel family, sized so that the whole file also finishes under compute-sanitizer
(memcheck / racecheck / synccheck on configs 1 and 4 and on the tensor-core kernels).  Each case is a
normal parity test as well.  The sanitizer runs are recorded in profiles/r2_sanitizer.md:

    compute-sanitizer --tool memcheck  python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q
    compute-sanitizer --tool synccheck python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q
"""
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
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2502_03170_b200 as lib
    return lib


def _check(psf, case, precision, kernels=None, tune=None):
    import torch
    plan = psf.plan_from_case(case, precision=precision)
    if tune:
        plan.tune(*tune)
    I = plan.compute()
    torch.cuda.synchronize()
    names = plan.kernel_names
    got = I.cpu().numpy().astype(np.float64)
    plan.destroy()
    ref = O.stack_T2(case)
    peak = ref.reshape(len(ref), -1).max(1)
    err = np.abs(got - ref).reshape(len(ref), -1).max(1) / peak
    assert err.max() <= TOL, (case.name, precision, names, err.max())
    if kernels is not None:
        assert names == kernels, names


def test_config1_fused_small_grid_kernel(psf):
    """config 1 (4 of its 16 planes): k_small, static mode."""
    c = W.config1()
    _check(psf, replace(c, z_um=c.z_um[::4]), "auto", ["k_small"])


def test_config4_fused_small_grid_kernel_per_plane_mode(psf):
    """config 4 (96 of its 4096 emitters): k_small, per-plane Zernike rows and shifts."""
    _check(psf, W.config4().with_planes(np.arange(0, 4096, 43)), "auto", ["k_smlm_tc"])
    _check(psf, W.config4().with_planes(np.arange(0, 4096, 43)), "auto", ["k_smlm"], tune=(psf.TUNE_SMLM, 2))
    _check(psf, W.config4().with_planes(np.arange(0, 4096, 43)), "auto", ["k_small"], tune=(psf.TUNE_SMLM, 0))


def test_ffma_tiles(psf):
    _check(psf, W.small_random_case(301, pupil_n=70, out_m=45, n_planes=2), "fp32", ["k1_stage1", "k2_stage2"])


def test_single_cta_tcgen05_kernels_tf32(psf):
    _check(psf, W.small_random_case(302, pupil_n=70, out_m=45, n_planes=2, per_plane=False, shifts=False), "3xtf32",
           ["k1_tc<tf32>", "k2_tc<tf32>"])


def test_single_cta_tcgen05_kernels_f16(psf):
    _check(psf, W.small_random_case(303, pupil_n=70, out_m=45, n_planes=2, per_plane=False, shifts=False), "3xf16",
           ["k1_tc<f16>", "k2_tc<f16>"], tune=(psf.TUNE_TC_PAIR_MASK, 0))


def test_group_mode_pair_kernel_and_resident_table_stage2(psf):
    _check(psf, W.small_random_case(304, pupil_n=130, out_m=67, n_planes=3, per_plane=False, shifts=False, pol=W.POL_CIRC_L),
           "auto", ["k1_pair<gm>", "k2_res"])


def test_pair_kernels(psf):
    _check(psf, W.small_random_case(305, pupil_n=150, out_m=300, n_planes=2, per_plane=False, shifts=False, pol=W.POL_UNPOLARIZED),
           "auto", ["k1_pair", "k2_pair"])


def test_chirp_z_fft_kernels(psf):
    _check(psf, W.small_random_case(306, pupil_n=60, out_m=50, n_planes=2, per_plane=False, shifts=False), "czt_fft",
           ["czt_rows", "czt_cols"])


def test_spherical_and_adjoint_kernels(psf):
    import torch
    case = replace(W.config1(), out_m=30, z_um=np.array([-0.4, 0.3]))
    plan = psf.plan_from_case(case)
    I = plan.compute_spherical(301).cpu().numpy().astype(np.float64)
    ref = O.bessel_stack(case, n_nodes=301)
    assert (np.abs(I - ref).reshape(2, -1).max(1) / ref.reshape(2, -1).max(1)).max() <= TOL
    plan.destroy()
    gc = W.small_random_case(307, pupil_n=24, out_m=20, n_planes=2)
    G = np.random.default_rng(3).standard_normal((2, 20, 20)).astype(np.float32)
    dz_ref, dc_ref = O.grad_T2(gc, G.astype(np.float64))
    plan = psf.plan_from_case(gc)
    dz, dc = plan.gradients(torch.from_numpy(G).cuda())
    torch.cuda.synchronize()
    assert np.abs(dz.cpu().numpy() - dz_ref).max() <= 2e-5 * np.abs(dz_ref).max()
    assert np.abs(dc.cpu().numpy() - dc_ref).max() <= 2e-5 * np.abs(dc_ref).max()
    plan.destroy()
