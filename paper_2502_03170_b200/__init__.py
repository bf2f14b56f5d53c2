"""paper_2502_03170_b200: B200-native (sm_100a) Fourier-parametrised vectorial Richards-Wolf PSF stacks.

The product is the C-ABI library `libpsf_b200.so` (include/psf.h); this package is its thin Python binding."""
from ._binding import (PsfError, PsfPlan, plan_from_case, host_tables, propagate_static, STATIC_SCRATCH_BYTES, load_library, lib_path, make_desc,
                       psf_plan_desc, EXPORTS, TUNE_TC_PAIR_MASK, TUNE_TC_SCRATCH_MB, TUNE_K1P_HANDOFF, TUNE_K1P_DEFER, TUNE_TC_FUSED, TUNE_SMLM, TUNE_GRAD_TENSOR, TUNE_K1P_ASPLIT, TUNE_FUSED_WINDOW, TUNE_DEVICE_REFRESH, TUNE_PDL, TUNE_K1P_WAITFIRST)

__all__ = ["PsfError", "PsfPlan", "plan_from_case", "host_tables", "propagate_static", "STATIC_SCRATCH_BYTES", "load_library", "lib_path", "make_desc",
           "psf_plan_desc", "EXPORTS", "TUNE_TC_PAIR_MASK", "TUNE_TC_SCRATCH_MB", "TUNE_K1P_HANDOFF", "TUNE_K1P_DEFER", "TUNE_TC_FUSED", "TUNE_SMLM", "TUNE_GRAD_TENSOR", "TUNE_K1P_ASPLIT", "TUNE_FUSED_WINDOW", "TUNE_DEVICE_REFRESH", "TUNE_PDL", "TUNE_K1P_WAITFIRST"]
