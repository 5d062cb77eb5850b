"""Ordinary softmax attention, written out (oracle; test infrastructure).

The paper gives no attention formula; the reading pinned in
DESIGN.md R3 is the standard one: scores s_j = scale * <q, K_j>, weights
p = softmax(s) with max subtraction, out = sum_j p_j V_j, scale = 1/sqrt(D),
GQA: query head h reads KV head h // G ("every 4 query
heads sharing one key-value head").

All arithmetic in float64.
"""
from __future__ import annotations

import numpy as np


def softmax_attention_single(q: np.ndarray, K: np.ndarray, V: np.ndarray, scale: float) -> np.ndarray:
    """One query vector q[D] over a full sequence K[L,D], V[L,D] -> out[D].

    L == 0 returns zeros (no visible key; reading R18: the merge must not
    produce NaN)."""
    q = np.asarray(q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    if K.shape[0] == 0:
        return np.zeros(V.shape[1], dtype=np.float64)
    s = scale * (K @ q)                 # [L]
    m = np.max(s)
    e = np.exp(s - m)
    p = e / np.sum(e)
    return p @ V                        # [D]


def beam_attention(q: np.ndarray, K_cache: np.ndarray, V_cache: np.ndarray, scale: float) -> np.ndarray:
    """one beam's query q[Hq,D] over ITS OWN cache
    K_cache, V_cache [L,Hkv,D] -> out[Hq,D].  Head h uses KV head h // G."""
    Hq = q.shape[0]
    Hkv = K_cache.shape[1]
    G = Hq // Hkv
    out = np.empty((Hq, V_cache.shape[2]), dtype=np.float64)
    for h in range(Hq):
        out[h] = softmax_attention_single(q[h], K_cache[:, h // G, :], V_cache[:, h // G, :], scale)
    return out


def masked_attention(Q: np.ndarray, K: np.ndarray, V: np.ndarray, mask: np.ndarray, scale: float) -> np.ndarray:
    """Dense masked attention over one expanded sequence.

    Q[n,Hq,D] are the query rows, K,V[S,Hkv,D] all positions of the sequence,
    mask[n,S] boolean (True = visible).  Masked scores are set to -inf before
    the softmax, the textbook way.  Returns [n,Hq,D]."""
    Q = np.asarray(Q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    n, Hq, D = Q.shape
    G = Hq // K.shape[1]
    out = np.empty((n, Hq, V.shape[2]), dtype=np.float64)
    for h in range(Hq):
        s = scale * (Q[:, h, :] @ K[:, h // G, :].T)        # [n,S]
        s = np.where(mask, s, -np.inf)
        m = np.max(s, axis=1, keepdims=True)
        e = np.exp(s - m)
        p = e / np.sum(e, axis=1, keepdims=True)
        out[:, h, :] = p @ V[:, h // G, :]
    return out
