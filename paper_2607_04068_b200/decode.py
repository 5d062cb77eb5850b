"""One attention layer's STARK decode state: buffers + the order of the four calls.

SURVEY.md section 3.2 / PAPER.md:263-286: per decode step t
    stark_kv_append_reorg (t >= 1)  ->  stark_prefix_attn  ->  stark_tree_attn_step
and, after the caller turned the attention output into log-probs,
    stark_beam_topk.
Only buffer ownership and call ordering live here; all arithmetic is in the library.
"""
from __future__ import annotations

from typing import Optional, Sequence, Tuple

import torch

from . import binding as sb


class StarkLayer:
    """Prefix K/V (immutable, shared by all beams of a user), the compact
    per-level suffix buffers and the ancestor index of ONE layer."""

    def __init__(self, B: int, Hq: int, Hkv: int, D: int, d: int, Wmax: int, dtype: torch.dtype,
                 k_prefix: torch.Tensor, v_prefix: torch.Tensor, cu_seqlens: torch.Tensor,
                 max_prefix_len: int, softmax_scale: float = 0.0, n_q_per_step: Optional[Sequence[int]] = None):
        self.shape = sb.make_shape(B, Hq, Hkv, D, d, Wmax, dtype, softmax_scale)
        self.dtype, self.dev = dtype, k_prefix.device
        self.k_prefix, self.v_prefix, self.cu = k_prefix, v_prefix, cu_seqlens
        self.total_tokens = int(k_prefix.shape[0])
        self.max_len = int(max_prefix_len)
        self.k_suffix, self.v_suffix, self.anc = sb.alloc_suffix(self.shape, dtype, self.dev)
        self._parts = {}
        if n_q_per_step is not None:      # pre-allocate (CUDA-graph capture needs static buffers)
            for n_q in set(n_q_per_step):
                self._partials(n_q)

    def _partials(self, n_q: int):
        if n_q not in self._parts:
            ns = sb.stark_prefix_attn_plan(self.shape, n_q, self.total_tokens, self.max_len)
            self._parts[n_q] = (ns,) + sb.alloc_partials(self.shape, n_q, ns, self.dev)
        return self._parts[n_q]

    def append(self, level: int, k_new: torch.Tensor, v_new: torch.Tensor, parent: Optional[torch.Tensor],
               write_anc: bool = True) -> None:
        sb.stark_kv_append_reorg(self.shape, level, int(k_new.shape[1]), k_new, v_new, parent, self.k_suffix,
                                 self.v_suffix, self.anc if write_anc else None)

    def prefix(self, q: torch.Tensor) -> None:
        """A1: shared-prefix partials of q[B,n_q,Hq,D] into this layer's partial buffers."""
        n_q = int(q.shape[1])
        ns, pm, pl, po = self._partials(n_q)
        sb.stark_prefix_attn(self.shape, q, n_q, self.k_prefix, self.v_prefix, self.cu, self.total_tokens,
                             self.max_len, ns, pm, pl, po)

    def tree(self, level: int, q: torch.Tensor, out: torch.Tensor, anc: Optional[torch.Tensor] = None) -> None:
        """A2: ancestor-chain attention + log-sum-exp merge with the partials written by prefix(q)."""
        n_q = int(q.shape[1])
        ns, pm, pl, po = self._partials(n_q)
        sb.stark_tree_attn_step(self.shape, q, n_q, level, self.k_suffix, self.v_suffix,
                                self.anc if anc is None else anc, pm, pl, po, ns, out)

    def attend(self, level: int, q: torch.Tensor, out: Optional[torch.Tensor] = None,
               anc: Optional[torch.Tensor] = None, fused: Optional[bool] = None) -> torch.Tensor:
        """Attention of the level-`level` queries q[B,n_q,Hq,D] over prefix + ancestor chain.
        bf16: one fused launch (stark_decode_attn); fp32 (or fused=False): stark_prefix_attn followed by
        stark_tree_attn_step."""
        if out is None:
            out = torch.empty_like(q)
        if fused is None:
            fused = self.dtype == torch.bfloat16 and self.total_tokens > 0
        if fused:
            sb.stark_decode_attn(self.shape, q, int(q.shape[1]), level, self.k_prefix, self.v_prefix, self.cu,
                                 self.total_tokens, self.max_len, self.k_suffix, self.v_suffix,
                                 self.anc if anc is None else anc, out)
        else:
            self.prefix(q)
            self.tree(level, q, out, anc)
        return out

    def step(self, level: int, q: torch.Tensor, k_new: Optional[torch.Tensor], v_new: Optional[torch.Tensor],
             parent: Optional[torch.Tensor], out: Optional[torch.Tensor] = None,
             anc: Optional[torch.Tensor] = None, write_anc: bool = True) -> torch.Tensor:
        """append(level, k_new, v_new, parent) + attend(level, q) in ONE launch (stark_decode_step, bf16 only).
        `anc` = another layer's index buffer (the tree is shared: pass write_anc=False for layers > 0)."""
        if out is None:
            out = torch.empty_like(q)
        sb.stark_decode_step(self.shape, q, int(q.shape[1]), level, self.k_prefix, self.v_prefix, self.cu,
                             self.total_tokens, self.max_len, k_new, v_new, parent, self.k_suffix, self.v_suffix,
                             self.anc if anc is None else anc, write_anc, out)
        return out

    def n_splits(self, n_q: int) -> int:
        return self._partials(n_q)[0]


_WS_CACHE = {}


def topk_workspace(B: int, W_in: int, C: int, device, logits: bool = False) -> Optional[torch.Tensor]:
    """Workspace of stark_beam_topk (logits: stark_beam_topk_logits) for this shape, sized by the library's own
    helper.  include/stark.h: it must be ZERO before its first use and every call leaves it zero, so one cached
    buffer per (device, size) serves all calls that are ordered on one stream."""
    shape = sb.make_shape(B=B, Hq=1, Hkv=1, D=64, d=1, Wmax=W_in, dtype=torch.float32)
    n = sb.stark_workspace_bytes(shape, sb.CALL_BEAM_TOPK_LOGITS if logits else sb.CALL_BEAM_TOPK, W_in, C)
    if n == 0:
        return None
    key = (str(device), n, logits)
    if key not in _WS_CACHE:
        _WS_CACHE[key] = torch.zeros(n, dtype=torch.uint8, device=device)
    return _WS_CACHE[key]


def beam_topk(logp: torch.Tensor, score: Optional[torch.Tensor], W_out: int,
              out: Optional[Tuple[torch.Tensor, torch.Tensor, torch.Tensor]] = None,
              ws: Optional[torch.Tensor] = None):
    """logp[B,W_in,C] fp32, score[B,W_in] fp32 or None -> (score, parent, code) [B,W_out]."""
    B, W_in, C = logp.shape
    if out is None:
        out = (torch.empty((B, W_out), dtype=torch.float32, device=logp.device),
               torch.empty((B, W_out), dtype=torch.int32, device=logp.device),
               torch.empty((B, W_out), dtype=torch.int32, device=logp.device))
    if ws is None:
        ws = topk_workspace(B, W_in, C, logp.device)
    sb.stark_beam_topk(logp, score, B, W_in, C, W_out, out[0], out[1], out[2], ws)
    return out


def beam_topk_static(logp: torch.Tensor, score: Optional[torch.Tensor], W_out: int,
                     out: Tuple[torch.Tensor, torch.Tensor, torch.Tensor]):
    """beam_topk for callers that must not allocate: the outputs are the caller's, the scratch memory is the
    library's static array (include/stark.h: stark_beam_topk_static -- its size limit and the no-overlap rule)."""
    B, W_in, C = logp.shape
    sb.stark_beam_topk_static(logp, score, B, W_in, C, W_out, out[0], out[1], out[2])
    return out


def beam_topk_logits(logits: torch.Tensor, score: Optional[torch.Tensor], W_out: int,
                     out: Optional[Tuple[torch.Tensor, torch.Tensor, torch.Tensor]] = None,
                     ws: Optional[torch.Tensor] = None):
    """logits[B,W_in,C] fp32 (raw), score[B,W_in] fp32 or None -> (score, parent, code) [B,W_out]
    (include/stark.h A3': the log-softmax normaliser is folded into the beam score)."""
    B, W_in, C = logits.shape
    if out is None:
        out = (torch.empty((B, W_out), dtype=torch.float32, device=logits.device),
               torch.empty((B, W_out), dtype=torch.int32, device=logits.device),
               torch.empty((B, W_out), dtype=torch.int32, device=logits.device))
    if ws is None:
        ws = topk_workspace(B, W_in, C, logits.device, logits=True)
    sb.stark_beam_topk_logits(logits, score, B, W_in, C, W_out, out[0], out[1], out[2], ws)
    return out
