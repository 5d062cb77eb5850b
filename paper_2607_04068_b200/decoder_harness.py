"""Config 3 harness (BASELINE.json configs[2]; reading R17): a random-init decoder-only transformer
whose GEMMs run in torch/cuBLAS while decode attention, KV append/reorg and beam top-k go through the STARK
library.  A USER of the library, not part of its hot path (it lives in the package so that both `bench.py
--workload cfg3_decoder` and `tests/` can import it): it shows the four calls inside a real multi-layer decode loop (the tree is
shared by all layers: layer 0 writes the ancestor index, the others pass write_anc = 0) and captures per-call
inputs so that tests can compare sampled (layer, user, step) triples with the oracle.

Model (R17): token embedding + learned absolute positions for the prefix; SID embedding table [d*C, d_model]
+ level embedding for generated tokens; per layer RMSNorm -> QKV -> attention -> out-proj,
RMSNorm -> SwiGLU -> down; final RMSNorm; a separate head [d_model, C] per level; all weights N(0, 0.02),
norm gains 1, bf16.  Prefill = torch SDPA (causal), untimed, builds the packed prefix K/V of every layer."""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List

import torch
import torch.nn.functional as F

from .decode import StarkLayer, beam_topk


@dataclass
class DecoderShape:
    n_layers: int = 12
    d_model: int = 1024
    Hq: int = 16
    Hkv: int = 4
    D: int = 64
    ffn: int = 4096
    vocab: int = 65536
    prefix: int = 2048
    B: int = 64
    W: int = 128
    d: int = 4
    C: int = 256


def rmsnorm(x: torch.Tensor, eps: float = 1e-6) -> torch.Tensor:
    xf = x.float()
    return (xf * torch.rsqrt(xf.pow(2).mean(-1, keepdim=True) + eps)).to(x.dtype)


class Decoder:
    def __init__(self, sh: DecoderShape, seed: int = 0, device: str = "cuda"):
        self.sh, self.dev = sh, torch.device(device)
        g = torch.Generator(device="cpu").manual_seed(seed)
        w = lambda *s: (torch.randn(*s, generator=g) * 0.02).to(torch.bfloat16).to(self.dev)
        self.tok = w(sh.vocab, sh.d_model)
        self.pos = w(sh.prefix, sh.d_model)
        self.sid = w(sh.d * sh.C, sh.d_model)
        self.lvl = w(sh.d + 1, sh.d_model)
        nqkv = (sh.Hq + 2 * sh.Hkv) * sh.D
        self.layers = [dict(qkv=w(sh.d_model, nqkv), out=w(sh.Hq * sh.D, sh.d_model), gate=w(sh.d_model, sh.ffn),
                            up=w(sh.d_model, sh.ffn), down=w(sh.ffn, sh.d_model)) for _ in range(sh.n_layers)]
        self.heads = [w(sh.d_model, sh.C) for _ in range(sh.d)]

    def _qkv(self, lw, x):
        sh = self.sh
        y = rmsnorm(x) @ lw["qkv"]
        q, k, v = y.split([sh.Hq * sh.D, sh.Hkv * sh.D, sh.Hkv * sh.D], dim=-1)
        return (q.reshape(*x.shape[:-1], sh.Hq, sh.D), k.reshape(*x.shape[:-1], sh.Hkv, sh.D),
                v.reshape(*x.shape[:-1], sh.Hkv, sh.D))

    def _ffn(self, lw, x):
        h = rmsnorm(x)
        return x + (F.silu(h @ lw["gate"]) * (h @ lw["up"])) @ lw["down"]

    def prefill(self, tokens: torch.Tensor):
        """tokens [B, L] -> per-layer packed prefix K/V [B*L, Hkv, D], and the per-layer attention output of the
        LAST position (torch SDPA, causal) for the step-0 cross-check."""
        sh = self.sh
        B, L = tokens.shape
        x = self.tok[tokens] + self.pos[:L]
        kv, last_attn = [], []
        for lw in self.layers:
            q, k, v = self._qkv(lw, x)
            o = F.scaled_dot_product_attention(q.transpose(1, 2), k.transpose(1, 2), v.transpose(1, 2), is_causal=True,
                                               enable_gqa=True).transpose(1, 2)          # [B, L, Hq, D]
            kv.append((k.reshape(B * L, sh.Hkv, sh.D).contiguous(), v.reshape(B * L, sh.Hkv, sh.D).contiguous()))
            last_attn.append(o[:, -1].contiguous())
            x = self._ffn(lw, x + o.reshape(B, L, -1) @ lw["out"])
        return kv, last_attn

    def decode(self, tokens: torch.Tensor, capture: bool = True, state=None) -> Dict[str, list]:
        """Semantic-ID beam search over d levels through the library.  Returns the selections per level and, if
        `capture`, every layer's (q, k_new, v_new, attention out) per step plus the fp32 log-probs.
        `state` = (prefix K/V per layer, last-position attention, StarkLayer list) of an earlier call: skips the
        prefill and every allocation of library buffers, so that the decode loop is CUDA-graph capturable."""
        sh = self.sh
        B, L = tokens.shape
        if state is None:
            kv, last_attn = self.prefill(tokens)
            cu = (torch.arange(B + 1, device=self.dev, dtype=torch.int32) * L).contiguous()
            layers = [StarkLayer(B, sh.Hq, sh.Hkv, sh.D, sh.d, sh.W, torch.bfloat16, k, v, cu, L) for k, v in kv]
        else:
            kv, last_attn, layers = state
        cap = dict(q=[], k=[], v=[], out=[], logp=[], sel=[], prefix_kv=kv, last_attn=last_attn)
        widths, w_in = [], 1
        for t in range(sh.d):
            widths.append(min(sh.W, w_in * sh.C)); w_in = widths[-1]
        score = parent = code = None
        for t in range(sh.d):
            if t == 0:   # the last prefix token queries its own prefix (its K/V are already inside it, reading R2)
                x = (self.tok[tokens[:, -1]] + self.pos[L - 1]).unsqueeze(1)               # [B, 1, d_model]
            else:
                x = self.sid[(t - 1) * sh.C + code.long()] + self.lvl[t]                   # [B, W_t, d_model]
            cq, ck, cv, co = [], [], [], []
            for li, (lw, layer) in enumerate(zip(self.layers, layers)):
                q, k, v = self._qkv(lw, x)
                q, k, v = q.contiguous(), k.contiguous(), v.contiguous()
                # append + attention in one launch; the tree is shared by all layers: only layer 0 extends the index
                o = layer.step(t, q, k if t >= 1 else None, v if t >= 1 else None, parent, anc=layers[0].anc,
                               write_anc=(li == 0))
                if capture:
                    cq.append(q), ck.append(k), cv.append(v), co.append(o)
                x = self._ffn(lw, x + o.reshape(*x.shape[:-1], -1) @ lw["out"])
            logp = torch.log_softmax((rmsnorm(x) @ self.heads[t]).float(), dim=-1).contiguous()
            score, parent, code = beam_topk(logp, score, widths[t])
            if capture:
                cap["q"].append(cq), cap["k"].append(ck), cap["v"].append(cv), cap["out"].append(co)
                cap["logp"].append(logp)
            cap["sel"].append((score, parent, code))
        cap["layers"] = layers
        return cap

    def replay_library(self, cap: Dict[str, list]) -> None:
        """Re-issue exactly the library calls of one decode (captured inputs, no GEMMs): what the STARK kernels
        alone cost inside the 12-layer loop."""
        sh = self.sh
        layers: List[StarkLayer] = cap["layers"]
        score = parent = None
        for t in range(sh.d):
            for li, layer in enumerate(layers):
                layer.step(t, cap["q"][t][li], cap["k"][t][li] if t >= 1 else None, cap["v"][t][li] if t >= 1 else None,
                           parent, out=cap["out"][t][li], anc=layers[0].anc, write_anc=(li == 0))
            score, parent, _ = beam_topk(cap["logp"][t], score, cap["sel"][t][1].shape[1], out=cap["sel"][t])
