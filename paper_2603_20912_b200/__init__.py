"""paper_2603_20912_b200 -- B200-native CCSD particle-particle ladder (Cholesky ERIs), FP64.

    R[i,j,a,b] += sum_cd (ac|bd) t2[i,j,c,d],   (ac|bd) = sum_P L[P,a,c] L[P,b,d]

The product is the C-ABI library ``libppl.so`` (include/ppl.h; kernels in csrc/).  This package is
the thin binding over it.  It never imports ``oracle/`` and has no CPU path.
"""
from .binding import (  # noqa: F401
    PPL_ERR_ALLOC,
    PPL_ERR_CUDA,
    PPL_ERR_INVALID_ARG,
    PPL_ERR_PRECONDITION,
    PPL_ERR_SCRATCH_LIMIT,
    PPL_NOALLOC_SCRATCH_BYTES,
    PPL_ERR_UNSUPPORTED_DEVICE,
    PPL_ERR_WORKSPACE_TOO_SMALL,
    PPL_OK,
    PPL_OPT_VERIFY_INPUTS,
    PPL_SYM_NONE,
    PPL_LAYOUT_IAJB,
    PPL_LAYOUT_IJAB,
    PPL_SYM_PAIR,
    PPL_SYM_PAIR_SA,
    PPL_SYM_FULL,
    SYMBOLS,
    Plan,
    PplError,
    error_string,
    lib,
    library_path,
    ppl_apply,
    ppl_contract_pair,
    ppl_contract_pair_noalloc,
    ppl_debug_dmma_layout,
    ppl_destroy,
    ppl_last_error,
    ppl_plan,
    ppl_plan_dry,
    ppl_probe_fp64_peak,
    ppl_probe_fp64_pipe,
)
from ._build import build  # noqa: F401
