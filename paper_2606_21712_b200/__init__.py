"""paper_2606_21712_b200 -- B200-native combined MoE layer (the hot path behind BatchGen's `combine`).

Thin Python binding over the C-ABI library `libbg_moe.so` (see `include/bg_moe.h`).  Every step
of the path runs in the library's CUDA kernels; this package only marshals arguments.  PyTorch is
used for device memory and streams.  There is no CPU fallback: loading fails loudly if the
library has not been built (`python -m paper_2606_21712_b200.build`).
"""
from .binding import (BgMoeError, BgMoeFit, MoELayer, load_library, fit_roofline, workspace_bytes_for, choose_tokens, route_logits_noalloc, NOALLOC_MAX_TOKENS, BG_OK, BG_ERR_INVALID_ARG, BG_ERR_UNSUPPORTED,
                      BG_ERR_CUDA, BG_ERR_NOMEM, BG_ERR_NO_WEIGHTS)

__all__ = ["BgMoeError", "BgMoeFit", "MoELayer", "load_library", "fit_roofline", "workspace_bytes_for", "choose_tokens", "route_logits_noalloc", "NOALLOC_MAX_TOKENS", "BG_OK", "BG_ERR_INVALID_ARG", "BG_ERR_UNSUPPORTED",
           "BG_ERR_CUDA", "BG_ERR_NOMEM", "BG_ERR_NO_WEIGHTS"]
