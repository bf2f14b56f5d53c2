"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/psf.h declares, validates
descriptors, and its plan-time fp64 tables (host code, independent of the oracle) agree with the oracle's."""
import ctypes as C
import os
import re
from dataclasses import replace

import numpy as np
import pytest

import paper_2502_03170_b200 as psf
import psf_workloads as W
from oracle import psf_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = psf.load_library()
    hdr = open(os.path.join(ROOT, "include", "psf.h")).read()
    declared = set(re.findall(r"\b(psf_[a-z_]+)\s*\(", hdr))
    assert declared == set(psf.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_descriptor_layout_matches_header_order():
    hdr = open(os.path.join(ROOT, "include", "psf.h")).read()
    body = hdr[hdr.index("typedef struct {"):hdr.index("} psf_plan_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        for part in decl.split(","):
            tok = re.findall(r"[A-Za-z_][A-Za-z0-9_]*", part)
            if tok:
                names.append(tok[-1] if tok[-1] != "4" else tok[-2])
    assert names == [f[0] for f in psf.psf_plan_desc._fields_]


@pytest.mark.parametrize("field,value,status", [
    ("NA", 0.0, 1), ("NA", 1.6, 1), ("wavelength_um", -1.0, 1), ("pupil_n", 1, 1), ("out_m", 0, 1),
    ("pixel_um", 0.0, 1), ("n_sample", 0.0, 1),
])
def test_invalid_descriptors_are_rejected_before_any_device_work(field, value, status):
    case = replace(W.config1(), **{field: value})
    with pytest.raises(psf.PsfError) as e:
        psf.PsfPlan(case)
    assert e.value.status == status


def test_non_finite_z_and_null_out_are_rejected():
    case = replace(W.config1(), z_um=np.array([0.0, np.nan]))
    with pytest.raises(psf.PsfError) as e:
        psf.PsfPlan(case)
    assert e.value.status == 1
    lib = psf.load_library()
    desc, keep = psf.make_desc(W.config1())
    assert lib.psf_plan_create(C.byref(desc), None) == 1
    assert b"NULL" in lib.psf_last_error(None)
    desc.flags = 64  # unknown flag bit
    h = C.c_void_p()
    assert lib.psf_plan_create(C.byref(desc), C.byref(h)) == 1 and not h.value


def _oracle_base(case, jones=None):
    pup = O.Pupil(case, jones=jones)
    N = case.pupil_n
    out = np.zeros((len(pup.g), N, N), dtype=np.complex128)
    W_static = pup.W_static.copy()
    if case.zernike is not None and not case.per_plane_zernike:
        W_static = W_static + np.asarray(case.zernike, dtype=np.float64) @ pup.zernike_basis()
    for c, g in enumerate(pup.g):
        out[c][pup.py, pup.px] = pup.prefactor * pup.amp * g * np.exp(1j * W_static)
    kap = np.zeros((N, N))
    kap[pup.py, pup.px] = pup.k * pup.costh
    return out, kap, pup.mask


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_host_tables_match_oracle_pupil(cfg):
    case = W.get_config(cfg)
    if cfg == 3:
        case = replace(case, pupil_n=96)
    t = psf.host_tables(case, case.zernike, case.noll_first)
    base, kap, mask = _oracle_base(case)
    assert t["n_components"] == 3 and np.array_equal(t["mask"], mask)
    assert np.abs(t["kappa"] - kap).max() < 1e-12 * kap.max()
    assert np.abs(t["base"] - base).max() < 1e-11 * np.abs(base).max()


def test_host_tables_unpolarised_five_pupils_reproduce_both_inputs():
    case = replace(W.config5(), pupil_n=48)
    t = psf.host_tables(case, case.zernike, case.noll_first)
    assert t["n_components"] == 5 and np.allclose(t["weights"], [0.5, 1.0, 0.5, 0.5, 0.5])
    bx, _, _ = _oracle_base(case, jones=(1.0 + 0j, 0j))
    by, _, _ = _oracle_base(case, jones=(0j, 1.0 + 0j))
    a, b, d, cx, cy = t["base"]
    scale = np.abs(bx).max()
    for got, want in ((a, bx[0]), (b, bx[1]), (cx, bx[2]), (b, by[0]), (d, by[1]), (cy, by[2])):
        assert np.abs(got - want).max() < 1e-11 * scale


def test_host_tables_odd_grid_and_jones():
    case = W.small_random_case(21, pupil_n=13, out_m=7, per_plane=False, shifts=False)
    t = psf.host_tables(case, case.zernike, case.noll_first)
    base, kap, mask = _oracle_base(case)
    assert np.array_equal(t["mask"], mask)
    assert np.abs(t["base"] - base).max() < 1e-11 * np.abs(base).max()


def test_host_tables_scalar_model_and_gaussian_envelope():
    """PSF_MODEL_SCALAR (one pupil, polarisation ignored) and PSF_FLAG_GAUSSIAN_ENVELOPE against the oracle's pupil."""
    case = replace(W.config3(), pupil_n=40, model="scalar", envelope_s=0.7, pol=W.POL_CIRC_L)
    t = psf.host_tables(case)
    base, kap, mask = _oracle_base(case)
    assert t["n_components"] == 1 and base.shape[0] == 1 and t["weights"][0] == 1.0
    assert np.abs(t["base"][:1] - base).max() < 1e-11 * np.abs(base).max()
    vec = replace(W.config2(), pupil_n=33, envelope_s=0.45)
    t = psf.host_tables(vec, vec.zernike, vec.noll_first)
    base, _, _ = _oracle_base(vec)
    assert np.abs(t["base"] - base).max() < 1e-11 * np.abs(base).max()
    # the envelope changes the pupil (rim amplitude down by exp(-s_max^2 / s_env^2))
    t0 = psf.host_tables(replace(vec, envelope_s=0.0), vec.zernike, vec.noll_first)
    assert np.abs(t["base"]).max() < np.abs(t0["base"]).max()


def test_model_and_envelope_validation():
    lib = psf.load_library()
    desc, keep = psf.make_desc(W.config1())
    h = C.c_void_p()
    desc.model = 7
    assert lib.psf_plan_create(C.byref(desc), C.byref(h)) == 1 and b"model" in lib.psf_last_error(None)
    desc.model = 0
    desc.flags |= 8          # PSF_FLAG_GAUSSIAN_ENVELOPE with envelope_s = 0
    assert lib.psf_plan_create(C.byref(desc), C.byref(h)) == 1 and b"envelope_s" in lib.psf_last_error(None)


def test_host_tables_fresnel_coefficients():
    """PSF_FLAG_FRESNEL: complex q_s, q_p inside Eq. 6 (coherent and unpolarised pupils), supercritical rim included."""
    case = replace(W.config3(), pupil_n=36, fresnel=True, n_glass=1.46, pol=W.POL_CIRC_L)
    t = psf.host_tables(case)
    base, _, _ = _oracle_base(case)
    assert np.abs(t["base"] - base).max() < 1e-11 * np.abs(base).max()
    t0 = psf.host_tables(replace(case, fresnel=False))
    assert np.abs(t["base"] - t0["base"]).max() > 1e-2 * np.abs(base).max()
    un = replace(case, pol=W.POL_UNPOLARIZED)
    t = psf.host_tables(un)
    bx, _, _ = _oracle_base(un, jones=(1.0 + 0j, 0j))
    by, _, _ = _oracle_base(un, jones=(0j, 1.0 + 0j))
    a, b, d, cx, cy = t["base"]
    for got, want in ((a, bx[0]), (b, bx[1]), (cx, bx[2]), (b, by[0]), (d, by[1]), (cy, by[2])):
        assert np.abs(got - want).max() < 1e-11 * np.abs(bx).max()


def test_create_errors_are_per_thread_and_nothing_crosses_the_abi():
    """psf.h: distinct plans are independent across threads; the message of a failed psf_plan_create belongs to the
    calling thread.  Two threads fail in different ways many times over (no device is needed for either failure)."""
    import threading
    lib = psf.load_library()
    bad = []

    def worker(kind):
        for _ in range(200):
            if kind == 0:
                desc, keep = psf.make_desc(replace(W.config1(), NA=0.0))
                h = C.c_void_p()
                st = lib.psf_plan_create(C.byref(desc), C.byref(h))
                msg = lib.psf_last_error(None)
                if st != 1 or h.value or b"NA" not in msg:
                    bad.append((kind, st, msg))
            else:
                desc, keep = psf.make_desc(W.config1())
                st = lib.psf_plan_create(C.byref(desc), None)
                msg = lib.psf_last_error(None)
                if st != 1 or b"NULL" not in msg:
                    bad.append((kind, st, msg))

    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not bad, bad[:3]


def test_library_reads_no_environment_variable_outside_the_phase_timer():
    """SURVEY section 5 / psf.h: no environment variables steer the product; the one getenv is the PSF_TIMING development
    aid of PhaseTimer (plan.hpp), which only prints wall-clock phases."""
    csrc = os.path.join(ROOT, "paper_2502_03170_b200", "csrc")
    hits = []
    for f in sorted(os.listdir(csrc)):
        if not os.path.isfile(os.path.join(csrc, f)):
            continue
        for i, line in enumerate(open(os.path.join(csrc, f)), 1):
            if "getenv" in line:
                hits.append((f, i, line.strip()))
    assert len(hits) == 1 and hits[0][0] == "plan.hpp" and "PSF_TIMING" in hits[0][2], hits
