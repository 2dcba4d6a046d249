"""B200-native explicit EM time-marching + Joule-heat hot path of arxiv/paper_2603_07038.

The product is the C-ABI library ``libem.so`` (include/em.h, csrc/*.cu, hand-written sm_100a CUDA
kernels).  This package is the thin Python binding with the same call names; PyTorch is used only
for device memory and streams.  There is no CPU fallback: importing the binding without the built
library raises.
"""
from .binding import (  # noqa: F401
    EM, EMError, lib_path, load, load_fuzz,
    EM_LOSS_CD, EM_LOSS_EXP, EM_KERNEL_AUTO, EM_KERNEL_SPLIT, EM_KERNEL_TMA, EM_FORM_LEAPFROG, EM_FORM_EONLY,
    EM_ABI_VERSION,
    em_workspace_bytes, em_cfl_dt,
)
