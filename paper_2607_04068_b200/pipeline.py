"""One whole pass of the STARK hot path (all rows of SURVEY.md section 8(a)) for one batch:
decode steps t = 0..d-1, each  append(t>=1) -> decode attention -> beam_topk.  bf16: append and attention are
ONE launch (stark_decode_step; `inline_append=False` keeps stark_kv_append_reorg -> stark_decode_attn); fp32:
stark_kv_append_reorg -> stark_prefix_attn -> stark_tree_attn_step.

Inputs (prefix K/V, per-step q / k_new / v_new, per-level log-probs) are device tensors;
`DecodePass.run()` only enqueues library calls on the current stream, so a pass is CUDA-graph
capturable (shapes are static per step).  The tree is data dependent: the
parents chosen by stark_beam_topk at level t feed stark_kv_append_reorg at level t+1.
"""
from __future__ import annotations

from typing import Dict, List, Optional

import torch

from . import binding as sb
from .decode import StarkLayer, beam_topk, beam_topk_logits


class DecodePass:
    def __init__(self, B: int, Hq: int, Hkv: int, D: int, d: int, C: int, widths: List[int], dtype: torch.dtype,
                 k_prefix: torch.Tensor, v_prefix: torch.Tensor, cu_seqlens: torch.Tensor, max_prefix_len: int,
                 q: List[torch.Tensor], k_new: List[torch.Tensor], v_new: List[torch.Tensor],
                 logp: List[torch.Tensor], inline_append: bool = True, from_logits: bool = False):
        self.B, self.d, self.C, self.widths = B, d, C, list(widths)
        self.n_q = [1] + self.widths                      # queries per user at step t
        self.fused = dtype == torch.bfloat16 and int(k_prefix.shape[0]) > 0
        self.inline_append = self.fused and inline_append
        self.layer = StarkLayer(B, Hq, Hkv, D, d, max(self.widths), dtype, k_prefix, v_prefix, cu_seqlens,
                                max_prefix_len, n_q_per_step=None if self.fused else self.n_q[:d])
        self.q, self.k_new, self.v_new, self.logp = q, k_new, v_new, logp
        dev = k_prefix.device
        # from_logits: `logp` holds RAW per-level logits and the selection is stark_beam_topk_logits (A3':
        # the log-softmax normaliser is folded into the beam score, two launches per level)
        self.from_logits = from_logits
        # one workspace for every level's selection (zero before its first use, left zero by every call)
        shp = sb.make_shape(B, 1, 1, 64, 1, max(self.n_q), torch.float32)
        call = sb.CALL_BEAM_TOPK_LOGITS if from_logits else sb.CALL_BEAM_TOPK
        need = max(sb.stark_workspace_bytes(shp, call, self.n_q[t], C) for t in range(d))
        self.topk_ws = torch.zeros(need, dtype=torch.uint8, device=dev) if need else None
        self.out = [torch.empty_like(q[t]) for t in range(d)]
        self.sel = [(torch.empty((B, w), dtype=torch.float32, device=dev),
                     torch.empty((B, w), dtype=torch.int32, device=dev),
                     torch.empty((B, w), dtype=torch.int32, device=dev)) for w in self.widths]

    #: library kernels launched by one run(): attention (1 fused or 2) + top-k per step, + append for t >= 1
    #: unless it rides inside the attention launch
    @property
    def launches(self) -> int:
        return ((2 if self.fused else 3) * self.d + (0 if self.inline_append else self.d - 1)
                + (sum(1 for t in range(self.d) if not (self.n_q[t] == 1 and self.C <= 512)) if self.from_logits else 0))

    def run(self) -> None:
        score = parent = None
        for t in range(self.d):
            if self.inline_append:
                self.layer.step(t, self.q[t], self.k_new[t] if t >= 1 else None, self.v_new[t] if t >= 1 else None,
                                parent, out=self.out[t])
            else:
                if t >= 1:
                    self.layer.append(t, self.k_new[t], self.v_new[t], parent)
                self.layer.attend(t, self.q[t], out=self.out[t], fused=self.fused)
            score, parent, _ = self.select(t, score)

    def select(self, t: int, score: Optional[torch.Tensor]):
        if self.from_logits:
            return beam_topk_logits(self.logp[t], score, self.widths[t], out=self.sel[t], ws=self.topk_ws)
        return beam_topk(self.logp[t], score, self.widths[t], out=self.sel[t], ws=self.topk_ws)

    def result(self) -> Dict[str, List[torch.Tensor]]:
        return {"score": [s[0] for s in self.sel], "parent": [s[1] for s in self.sel],
                "code": [s[2] for s in self.sel]}

    def paths(self) -> torch.Tensor:
        """[B, W_d, d] SID paths of the final beams in slot order (index bookkeeping for
        reporting; not part of the timed path)."""
        W = self.widths[-1]
        slot = torch.arange(W, device=self.sel[-1][1].device).expand(self.B, W).long()
        cols: List[Optional[torch.Tensor]] = [None] * self.d
        for t in range(self.d - 1, -1, -1):
            cols[t] = torch.gather(self.sel[t][2].long(), 1, slot)
            slot = torch.gather(self.sel[t][1].long(), 1, slot)
        return torch.stack(cols, dim=2)


class EncDecPass:
    """One pass of the hot path in the paper's ENCODER-DECODER form (DESIGN.md
    readings R23-R25): per decode step t two attention sub-layers instead of one --
      * cross-attention over the encoder memory M: the shared-prefix partials finalised ALONE
        (stark_decode_attn at level 0: every beam of a user attends the same M, read once per step);
      * causal self-attention over [e_click, e_atc, e_pay, <bos>] + the beam's ancestor chain (Eq. 7 and Eq. 14,
        PAPER.md:197-204, 265-268): the same library with a 4-row "prefix" per user (stark_decode_step: the
        level's K/V append rides inside the launch);
    then stark_beam_topk.  `run()` only enqueues library calls (CUDA-graph capturable)."""

    N_FIXED = 4

    def __init__(self, B: int, Hq: int, Hkv: int, D: int, d: int, C: int, widths: List[int], dtype: torch.dtype,
                 k_mem: torch.Tensor, v_mem: torch.Tensor, cu_mem: torch.Tensor, max_mem_len: int,
                 k_fix: torch.Tensor, v_fix: torch.Tensor, q_cross: List[torch.Tensor], q_self: List[torch.Tensor],
                 k_new: List[torch.Tensor], v_new: List[torch.Tensor], logp: List[torch.Tensor]):
        assert dtype == torch.bfloat16, "the fused launches are bf16 (fp32: compose stark_prefix_attn + stark_tree_attn_step)"
        self.B, self.d, self.C, self.widths = B, d, C, list(widths)
        self.n_q = [1] + self.widths
        dev = k_mem.device
        Wmax = max(self.widths)
        self.mem = StarkLayer(B, Hq, Hkv, D, d, Wmax, dtype, k_mem, v_mem, cu_mem, max_mem_len)
        cu_fix = (torch.arange(B + 1, device=dev, dtype=torch.int32) * self.N_FIXED).contiguous()
        self.dec = StarkLayer(B, Hq, Hkv, D, d, Wmax, dtype, k_fix.reshape(B * self.N_FIXED, Hkv, D).contiguous(),
                              v_fix.reshape(B * self.N_FIXED, Hkv, D).contiguous(), cu_fix, self.N_FIXED)
        self.q_cross, self.q_self, self.k_new, self.v_new, self.logp = q_cross, q_self, k_new, v_new, logp
        shp = sb.make_shape(B, 1, 1, 64, 1, max(self.n_q), torch.float32)
        need = max(sb.stark_workspace_bytes(shp, sb.CALL_BEAM_TOPK, self.n_q[t], C) for t in range(d))
        self.topk_ws = torch.zeros(need, dtype=torch.uint8, device=dev) if need else None
        self.cross = [torch.empty_like(q_cross[t]) for t in range(d)]
        self.self_out = [torch.empty_like(q_self[t]) for t in range(d)]
        self.sel = [(torch.empty((B, w), dtype=torch.float32, device=dev),
                     torch.empty((B, w), dtype=torch.int32, device=dev),
                     torch.empty((B, w), dtype=torch.int32, device=dev)) for w in self.widths]

    launches = property(lambda self: 3 * self.d)

    def run(self) -> None:
        score = parent = None
        for t in range(self.d):
            self.mem.attend(0, self.q_cross[t], out=self.cross[t], fused=True)
            self.dec.step(t, self.q_self[t], self.k_new[t] if t >= 1 else None, self.v_new[t] if t >= 1 else None,
                          parent, out=self.self_out[t])
            score, parent, _ = beam_topk(self.logp[t], score, self.widths[t], out=self.sel[t], ws=self.topk_ws)
