"""paper_2512_20927_b200 -- B200-native (sm_100a) Quantile Rendering hot path behind the C ABI of include/qr.h.

``binding`` mirrors the C entry points one to one; ``pipeline`` chains them.  The CUDA library is the only
implementation: importing this package never touches ``oracle/``.
"""
from . import binding, pipeline  # noqa: F401
from .binding import (QRError, qr_backward, qr_backward_clear, qr_backward_workspace, qr_bin_count, qr_bin_sort, qr_bin_workspace_bytes, qr_dense_forward,  # noqa: F401
                      qr_forward, qr_num_tiles, qr_preprocess, qr_topk_forward, qr_version)

__all__ = ["binding", "pipeline", "QRError", "qr_preprocess", "qr_bin_count", "qr_bin_sort", "qr_bin_workspace_bytes",
           "qr_forward", "qr_backward", "qr_backward_clear", "qr_backward_workspace", "qr_dense_forward", "qr_topk_forward", "qr_num_tiles", "qr_version"]
