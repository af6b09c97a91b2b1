"""paper_1904_01567_b200 -- B200-native gL-BFGS hot path of gMCO (arXiv 1904.01567).

The product is ``libgmco.so`` (C ABI in ``include/gmco.h``, CUDA sources in ``csrc/``).
This package is the thin Python binding: same entry-point names, argument marshalling only.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback:
importing :mod:`paper_1904_01567_b200.binding` raises if the library has not been built.
"""
from .binding import (GmcoError, Handle, Options, gmco_create, gmco_destroy, gmco_dose_rate_matrix, gmco_evaluate, gmco_get_stats,  # noqa: F401
                      gmco_optimize, gmco_pareto_front, gmco_result, gmco_sa_run, gmco_select_plan, gmco_set_profiling, gmco_tc_schedule,
                      gmco_version, lib, lib_path, DOSE_KERNEL_NAMES,
                      GMCO_PREC_TF32X3, GMCO_PREC_SIMT_FP32, GMCO_SA_FP64, GMCO_SA_FP32)
