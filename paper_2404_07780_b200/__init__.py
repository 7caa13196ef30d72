"""B200-native batched galaxy-profile fitting hot path (arxiv 2404.07780).

Thin Python binding over the C-ABI library ``libgm.so`` (``include/gm.h``):
argument marshalling only -- every step of the path runs in the CUDA kernels
under ``csrc/``.  PyTorch supplies device memory and streams.
"""
from .binding import (  # noqa: F401
    GM_CONV_FFMA2,
    GM_CONV_TENSOR,
    GM_OPT_CONST_TAPS,
    GM_OPT_FUSED,
    GM_OPT_TENSOR,
    GmError,
    gm_get_option,
    gm_init,
    gm_measure_fp32_peak,
    gm_set_option,
    gm_trace_set,
    gm_bootstrap,
    gm_bootstrap_counts,
    gm_bootstrap_counts_static,
    gm_conv,
    gm_fit,
    gm_fit_host,
    gm_fit_multi,
    gm_fit_multi_host,
    gm_last_launch_count,
    gm_loglike,
    gm_loss_grad,
    gm_loss_grad_host,
    gm_profile_enable,
    gm_profile_read,
    gm_render,
    gm_render_host,
    gm_strerror,
    gm_uncertainty,
    gm_uncertainty_workspace_bytes,
    gm_version,
    gm_workspace_bytes,
    library_path,
)
