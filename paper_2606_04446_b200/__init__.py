"""paper_2606_04446_b200 -- B200-native verification hot path of D2SD (arXiv 2606.04446).

The product is the C-ABI library ``libd2sd.so`` (``include/d2sd.h``); this package is its thin
Python binding: same calls, argument marshalling only.  PyTorch is used for device memory
and streams.  There is no CPU fallback: every call raises if the CUDA library is missing.
"""
from .binding import (  # noqa: F401
    D2sdError, accept, accept_workspace_bytes, build_tree, cascade_verify_attn,
    cascade_workspace, cascade_workspace_bytes, last_error, lib, lib_path, select_prefixes, t_cap, version,
    build_tree3, commit_kv, confidence_workspace_bytes, draft_confidence, select_third, t_cap3,
    accept_static, accept_static_max_bytes,
)
