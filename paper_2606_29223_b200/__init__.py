"""paper_2606_29223_b200 — B200-native expand/exit/commit/collapse step of Depth Exploration
Decoding (DEX, arxiv/paper_2606_29223).  The product is the C-ABI library
``libdex_b200.so`` (``include/dex.h``; sources in ``csrc/``); this package is the thin
ctypes binding with the same call names.  There is no CPU fallback: importing works without
a GPU (so the ABI can be checked), every compute call needs a B200.
"""
from .binding import (  # noqa: F401
    DexConfig, DexWeights, DexStepResult, Dex, lib, lib_path, exported_symbols,
    dex_workspace_bytes, dex_init, dex_prefill, dex_step, dex_collapse, dex_rewind, dex_get_tokens,
    dex_debug_read, dex_debug_gemm, dex_debug_phase_us, dex_profile, dex_destroy, dex_last_error, dex_gemm_noalloc,
    DEX_OK, DEX_EINVAL, DEX_ECAPACITY, DEX_ESTATE, DEX_ECUDA, DEX_STEP_AUTOCOLLAPSE,
    DEX_TAP_HIDDEN, DEX_TAP_LOGITS, DEX_TAP_B, DEX_TAP_FSM, DEX_MAX_DEPTHS, DexError,
)
