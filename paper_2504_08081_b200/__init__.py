"""paper_2504_08081_b200 -- B200-native SALT3 batched band flux (JAX-bandflux paper, arXiv 2504.08081).

Thin Python binding of the C-ABI library `libsaltband.so` (include/saltband.h).  Argument
marshalling only: every step of the hot path runs in the CUDA kernels of csrc/.  PyTorch is used
for device memory and streams.  There is no CPU fallback: a missing library raises ImportError,
a missing GPU makes every compute call raise.
"""
from .api import (  # noqa: F401
    SB_F32,
    SB_F64,
    SB_FORM_DIRECT,
    SB_FORM_GROUPED,
    SB_FORM_TILED,
    SB_NOALLOC_MAX_SN,
    FIT_CONVERGED,
    FIT_EXHAUSTED,
    FIT_RUNNING,
    FIT_STALLED,
    Bands,
    Model,
    Pack,
    SaltbandError,
    last_form,
    last_launch_count,
    lib_path,
    sb_bandflux,
    sb_bandflux_grad,
    sb_bandflux_grad_host,
    sb_chi2,
    sb_chi2_host,
    sb_chi2_noalloc,
    sb_fit_lbfgs,
    sb_fit_lbfgs_host,
    sb_load_bandpasses,
    sb_load_model,
    sb_pack_observations,
    version,
)
