"""B200 (sm_100a) FP8 EAGLE tree-verification: thin Python binding over libeagle_verify.so.

The product is the C-ABI library declared in include/eagle_verify.h (hand-written CUDA kernels
in csrc/).  This package only marshals arguments; it never imports oracle/."""
from .binding import (  # noqa: F401
    Cache, EvError, Model, VerifyBuffers, ev_last_error, ev_launch_count, ev_capture_count, ev_verify, ev_verify_host, load_library,
    LIB_PATH, SIGNATURES, ev_model_share_head, ev_draft_tree, ev_draft_extend, ev_gather_accepted, Engine,
)
