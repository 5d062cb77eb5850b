"""Conventional semantic-ID beam search (oracle; test infrastructure).

This is the "w/o STARK" baseline the paper describes: beams
are expanded along the batch dimension, each beam owns a private, physically
replicated KV cache (prefix included), attention is ordinary full-sequence
attention per beam, and after every selection the caches are duplicated and
rearranged into the new beam order.  Steps O1-O6 of SURVEY.md §8(c).

Step indexing (reading R2): decode step t = 0..d-1 produces the
logits of level t+1.  Step 0 has one query (the last prefix position, whose
K/V are already the last prefix row).  Step t >= 1 has W_t queries at tree
depth t, each attending to the whole prefix plus its own chain of t suffix
tokens, itself included (Eq. 14 "or j = i"; reading R9: a
token's K/V are appended before its attention).  An optional step t = d runs
the final-level tokens (hidden states for ranking) and selects
nothing.

The token model (where q/k/v of a generated token and the logits come from)
is supplied by the caller -- see `oracle/token_models.py`.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

from .attention import beam_attention
from .selection import log_softmax_fp32, select_beams


@dataclass
class _Hypothesis:
    path: Tuple[int, ...]
    score: np.float32
    K: np.ndarray      # [L + depth, Hkv, D] private copy
    V: np.ndarray


@dataclass
class BeamTrace:
    """Everything the comparison protocol needs, per user."""
    attn_out: List[np.ndarray] = field(default_factory=list)   # step t -> [n_q, Hq, D] fp64
    q: List[np.ndarray] = field(default_factory=list)          # step t -> [n_q, Hq, D]
    k_new: List[np.ndarray] = field(default_factory=list)      # step t>=1 -> [n_q, Hkv, D] (step 0: empty)
    v_new: List[np.ndarray] = field(default_factory=list)
    logp: List[np.ndarray] = field(default_factory=list)       # step t -> [n_q, C] fp32
    score_in: List[np.ndarray] = field(default_factory=list)   # step t -> [n_q] fp32
    parents: List[np.ndarray] = field(default_factory=list)    # level t+1 -> [W_{t+1}] int32
    codes: List[np.ndarray] = field(default_factory=list)
    scores: List[np.ndarray] = field(default_factory=list)     # fp32
    margins: List[float] = field(default_factory=list)         # key gap rank W vs W+1 (inf if none)
    paths: np.ndarray = None                                   # [W_d, d] int32, slot order


def conventional_beam_search(K_prefix: np.ndarray, V_prefix: np.ndarray, model, widths: Sequence[int],
                             C: int, scale: float, final_step: bool = False) -> BeamTrace:
    """One user.  K_prefix, V_prefix [L, Hkv, D]; `widths[t]` = beam width kept
    after level t+1's selection (per-level widths allowed);
    `model.qkv(t, slot, path)` -> (q[Hq,D], k[Hkv,D], v[Hkv,D]) (k, v ignored
    at t = 0); `model.logits(t, slot, path, o)` -> [C]."""
    d = len(widths)
    K_prefix = np.asarray(K_prefix, dtype=np.float64)
    V_prefix = np.asarray(V_prefix, dtype=np.float64)
    tr = BeamTrace()
    # O1
    hyps = [_Hypothesis((), np.float32(0.0), K_prefix.copy(), V_prefix.copy())]
    for t in range(d + (1 if final_step else 0)):
        outs, qs, ks, vs, logps = [], [], [], [], []
        for slot, h in enumerate(hyps):                              # O2, slot order
            q, k, v = model.qkv(t, slot, h.path)
            q = np.asarray(q, dtype=np.float64)
            if t >= 1:
                k = np.asarray(k, dtype=np.float64)
                v = np.asarray(v, dtype=np.float64)
                h.K = np.concatenate([h.K, k[None]], axis=0)         # append to ITS OWN cache
                h.V = np.concatenate([h.V, v[None]], axis=0)
                ks.append(k)
                vs.append(v)
            o = beam_attention(q, h.K, h.V, scale)
            outs.append(o)
            qs.append(q)
            if t < d:
                logps.append(log_softmax_fp32(model.logits(t, slot, h.path, o)))   # O3
        tr.attn_out.append(np.stack(outs))
        tr.q.append(np.stack(qs))
        tr.k_new.append(np.stack(ks) if ks else np.zeros((0,) + K_prefix.shape[1:]))
        tr.v_new.append(np.stack(vs) if vs else np.zeros((0,) + V_prefix.shape[1:]))
        if t == d:
            break
        score = np.array([h.score for h in hyps], dtype=np.float32)
        logp = np.stack(logps)
        tr.logp.append(logp)
        tr.score_in.append(score)
        W_out = min(int(widths[t]), len(hyps) * C)                   # reading R7
        new_score, parent, code = select_beams(score, logp, W_out)   # O4
        # selection margin (for the end-to-end identity argument)
        if W_out < len(hyps) * C:
            s2, _, _ = select_beams(score, logp, W_out + 1)
            tr.margins.append(float(np.float64(s2[W_out - 1]) - np.float64(s2[W_out])))
        else:
            tr.margins.append(float("inf"))
        # O5: deep copy of the parent's cache -- the duplication + rearrangement
        # the paper attributes to the conventional implementation
        hyps = [_Hypothesis(hyps[int(p)].path + (int(c),), np.float32(s),
                            hyps[int(p)].K.copy(), hyps[int(p)].V.copy())
                for s, p, c in zip(new_score, parent, code)]
        tr.parents.append(parent)
        tr.codes.append(code)
        tr.scores.append(new_score)
    # O6
    tr.paths = np.array([h.path for h in hyps], dtype=np.int32).reshape(len(hyps), -1)
    return tr
