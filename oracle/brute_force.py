"""Brute-force enumeration of every SID path (oracle; test infrastructure).

BASELINE.json north star, oracle check 3: "on tiny codebooks, beam width >= all
paths must recover brute-force enumeration of every SID path, ranked by summed
log-prob" (Eq. 1: P(v) = prod_j P(c_j | ..., c_<j)).

Each path is scored by its OWN independent full-sequence forward: the path's
tokens are appended one by one to a fresh copy of the prefix and attended with
ordinary causal attention -- no beams, no sharing, no selection.  Requires a
path-determined token model (e.g. `TableTokenModel`).
"""
from __future__ import annotations

import itertools
from typing import List, Tuple

import numpy as np

from .attention import beam_attention
from .selection import log_softmax_fp32


def enumerate_all_paths(K_prefix: np.ndarray, V_prefix: np.ndarray, model, d: int, C: int,
                        scale: float) -> Tuple[np.ndarray, np.ndarray, float]:
    """Returns (paths[C^d, d] int32 ranked by score descending, scores[C^d]
    fp32 accumulated level by level in fp32 exactly as a beam's score is,
    total_probability = sum over all paths of exp(score) in fp64)."""
    out: List[Tuple[float, Tuple[int, ...]]] = []
    for path in itertools.product(range(C), repeat=d):
        K = np.asarray(K_prefix, dtype=np.float64).copy()
        V = np.asarray(V_prefix, dtype=np.float64).copy()
        score = np.float32(0.0)
        for t in range(d):
            q, k, v = model.qkv(t, -1, path[:t])
            if t >= 1:
                K = np.concatenate([K, np.asarray(k, np.float64)[None]], axis=0)
                V = np.concatenate([V, np.asarray(v, np.float64)[None]], axis=0)
            o = beam_attention(np.asarray(q, np.float64), K, V, scale)
            logp = log_softmax_fp32(model.logits(t, -1, path[:t], o))
            score = np.float32(score + logp[path[t]])
        out.append((score, path))
    # rank by score descending; ties (not expected) by path order
    out.sort(key=lambda sp: (-float(sp[0]), sp[1]))
    paths = np.array([p for _, p in out], dtype=np.int32)
    scores = np.array([s for s, _ in out], dtype=np.float32)
    total = float(np.sum(np.exp(scores.astype(np.float64))))
    return paths, scores, total
