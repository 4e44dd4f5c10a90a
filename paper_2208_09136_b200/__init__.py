"""paper_2208_09136_b200 — the data-parallel hot path of averaged RQA (arXiv 2208.09136) on one B200.

The product is librqa.so (C ABI in include/rqa.h, CUDA kernels in csrc/).  This package is the thin Python
binding with the same names, plus the seeded workload generators (workloads.py).  Importing the package
does not import torch or load the library; the first call does, and fails loudly if the library is missing.
"""
from .binding import (RQA_ERR_CUDA, RQA_ERR_INVALID_ARG, RQA_ERR_NONFINITE_INPUT, RQA_ERR_UNSUPPORTED,  # noqa: F401
                      RQA_ERR_WORKSPACE_TOO_SMALL, RQA_MAX_K, RQA_MAX_M, RQA_NORM_EUCLID, RQA_NORM_MAX, RQA_OK,
                      EXPORTS, LIB_PATH, RqaError, RqaPoints, load_library, rqa_det_avg, rqa_embed, rqa_eps_for_rr,
                      rqa_det_prefix_avg, rqa_lam_tt, rqa_vert_hist, rqa_line_hist_static, RQA_STATIC_SCRATCH_BYTES, rqa_launch_count, rqa_line_hist, rqa_line_measures, rqa_sorting_rate_host, RqaOptions, make_options, rqa_sweep_host, rqa_sweep_workspace_bytes, rqa_version,
                      rqa_workspace_bytes, rqa_workspace_status)
from .api import SweepBuffers, averaged_rqa  # noqa: F401
