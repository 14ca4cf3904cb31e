"""paper_1007_1658_b200 -- B200-native direct Lomb-Scargle periodogram (Townsend 2010, arxiv 1007.1658).

The product is the CUDA library `liblsp_b200.so` (csrc/, C ABI in include/lsp.h); this package is
its thin Python binding.  Nothing here computes on the CPU and nothing imports `oracle/`.
"""
from .binding import (Handle, LspError, load, status_string, version, plan_query, plan_query_form, SYMBOLS, periodogram_static,
                      LSP_OK, LSP_EINVAL, LSP_ECUDA, LSP_ENOMEM, LSP_ELIMIT, STATIC_SCRATCH_BYTES, STATIC_MAX_NT, STATIC_MAX_NF,
                      PARAM_K, PARAM_THREADS, PARAM_NSPLIT, PARAM_PIPE, PARAM_FLUSH, PARAM_TIMING, PARAM_TABLE_MB, PARAM_COARSE, PARAM_TRUNC, PARAM_SHARED, PARAM_PDL, PARAM_CORR, PARAM_REFINE, PARAM_ORDER,
                      PIPE_AUTO, PIPE_FP32, PIPE_TENSOR)
from .build import build

__all__ = ["Handle", "LspError", "load", "status_string", "version", "build", "SYMBOLS"]
