"""Config 1 FREE-RUNNING end to end on the GPU (SURVEY.md section 8(c) "End-to-end (config 1, fp32)";
north star: "End-to-end beam sets on the fp32 config must be identical"; STARK "preserves
the decoding results of standard beam search").

Nothing is teacher-forced: the library's own attention output drives the projection -> logits -> selection ->
next level's q/k/v loop.  Library calls (fp32 path): stark_kv_append_reorg -> stark_prefix_attn ->
stark_tree_attn_step -> (torch fp32: logits = P_t^T vec(out) + b_t; the token model of reading R14 is the
caller's, not the library's) -> log-softmax + stark_beam_topk, or stark_beam_topk_logits on the raw logits.
The q/k/v of a generated token are gathered ON THE DEVICE from the R14 tables by the selected codes.

The oracle side is oracle.conventional_beam_search with TableTokenModel (fp64 projection, replicated caches).
The two sides share only the seeded tables of workloads/.
"""
from __future__ import annotations

import numpy as np
import torch

import workloads as wl
from oracle.beam_search import conventional_beam_search
from oracle.token_models import TableTokenModel

from paper_2607_04068_b200.decode import StarkLayer, beam_topk, beam_topk_logits


def run_free_running(cfg, seed=0, from_logits=False):
    """Returns (gpu, oracle traces per user): gpu = dict(parent, code, score per level [B, W], attn per step,
    paths [B, W_d, d])."""
    assert cfg.logits == "projection" and cfg.dtype == "f32"
    torch.backends.cuda.matmul.allow_tf32 = False            # the projection is plain fp32
    tb = wl.config1_tables(cfg, seed)
    K, V, cu = wl.prefix_kv(cfg, seed)
    lens = np.diff(cu)
    scale = 1.0 / np.sqrt(cfg.D)
    widths = wl.beam_widths(cfg)
    oracle = [conventional_beam_search(K[cu[u]:cu[u + 1]], V[cu[u]:cu[u + 1]], TableTokenModel(tb), widths, cfg.C, scale)
              for u in range(cfg.B)]

    dev = torch.device("cuda")
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    Tq, Tk, Tv, P, b, q_root = (up(tb[k]) for k in ("Tq", "Tk", "Tv", "P", "b", "q_root"))
    layer = StarkLayer(cfg.B, cfg.Hq, cfg.Hkv, cfg.D, cfg.d, cfg.Wmax, torch.float32, up(K), up(V),
                       up(cu.astype(np.int32)), int(lens.max()))
    B = cfg.B
    gpu = dict(parent=[], code=[], score=[], attn=[])
    score = parent = code = None
    for t in range(cfg.d):
        if t == 0:
            q = q_root.expand(B, 1, cfg.Hq, cfg.D).contiguous()
        else:
            c = code.long()
            q = Tq[t - 1][c].contiguous()                    # [B, W_t, Hq, D]: token of level t sits in table row t-1
            layer.append(t, Tk[t - 1][c].contiguous(), Tv[t - 1][c].contiguous(), parent)
        out = layer.attend(t, q)                             # stark_prefix_attn -> stark_tree_attn_step
        logits = (out.reshape(B, q.shape[1], -1) @ P[t] + b[t]).contiguous()
        if from_logits:
            score, parent, code = beam_topk_logits(logits, score, widths[t])
        else:
            score, parent, code = beam_topk(torch.log_softmax(logits, dim=-1).contiguous(), score, widths[t])
        gpu["attn"].append(out.cpu().numpy())
        gpu["parent"].append(parent.cpu().numpy())
        gpu["code"].append(code.cpu().numpy())
        gpu["score"].append(score.cpu().numpy())
    # final SID paths [B, W_d, d] in slot order, by following the parent pointers upward
    W = widths[-1]
    slot = np.tile(np.arange(W), (B, 1))
    cols = [None] * cfg.d
    for t in range(cfg.d - 1, -1, -1):
        cols[t] = np.take_along_axis(gpu["code"][t], slot, axis=1)
        slot = np.take_along_axis(gpu["parent"][t], slot, axis=1)
    gpu["paths"] = np.stack(cols, axis=2)
    return gpu, oracle
