"""B200-native STARK decode library (arxiv/paper_2607_04068 section 3.6): Python side.

`binding` is a thin ctypes layer over the C-ABI library `libstark.so`
(include/stark.h); `decode` drives the four calls for one layer's beam search.
"""
from .binding import (  # noqa: F401
    StarkError, Shape, make_shape, lib, LIB_PATH, EXPORTS,
    stark_prefix_attn, stark_prefix_attn_plan, stark_tree_attn_step, stark_decode_attn, stark_beam_topk,
    stark_logits_row_offset, stark_beam_topk_logits,
    stark_kv_append_reorg, stark_workspace_bytes, alloc_partials, alloc_suffix,
    CALL_PREFIX_ATTN, CALL_TREE_ATTN_STEP, CALL_BEAM_TOPK, CALL_KV_APPEND_REORG, CALL_BEAM_TOPK_LOGITS,
)
