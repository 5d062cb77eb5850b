"""The paper's own formulation: sequence-dimension expansion under the tree
mask of Eq. 14 (oracle; test infrastructure).

PAPER.md:263: "we concatenate candidate tokens along the sequence dimension
and use a predefined tree attention mask to control visibility.  Each token can
only attend to its ancestor nodes in the decoding tree and itself."
PAPER.md:265-268 (Eq. 14):  M_ij = 1 if j in Anc(p_i) or j = i, else 0.
Reading R8: every prefix column is visible to every
candidate token of the same user.

This second formulation must agree with the conventional per-beam one
(`oracle/beam_search.py`, `oracle/replay.py`); tests/ checks that.

Tree encoding: `parents[l-1][s]` = slot, at level l-1, of the parent of the
node in slot s of level l (l = 1..t).  Level-1 nodes hang off the root, which
is the last prefix position; `parents[0]` is therefore ignored.
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np

from .attention import masked_attention


def ancestor_chains(parents: Sequence[np.ndarray], t: int) -> np.ndarray:
    """chain[i, tau-1] = slot of the depth-tau ancestor of node i of level t,
    tau = 1..t (the last entry is i itself: Eq. 14's "or j = i")."""
    W_t = len(parents[t - 1])
    chain = np.empty((W_t, t), dtype=np.int64)
    for i in range(W_t):
        a = i
        for tau in range(t, 0, -1):
            chain[i, tau - 1] = a
            if tau > 1:
                a = int(parents[tau - 1][a])      # parent of a level-tau node lives at level tau-1
    return chain


def tree_mask(parents: Sequence[np.ndarray], t: int, L: int) -> np.ndarray:
    """Dense boolean mask [W_t, L + sum_{l<=t} W_l] for the level-t rows of the
    expanded sequence  prefix ++ level 1 ++ ... ++ level t  (slot order inside
    a level)."""
    widths = [len(parents[l]) for l in range(t)]
    offs = np.concatenate([[0], np.cumsum(widths)]).astype(np.int64)
    S = L + int(offs[-1])
    M = np.zeros((widths[t - 1], S), dtype=bool)
    M[:, :L] = True                                   # R8: the shared prefix
    chain = ancestor_chains(parents, t)
    for i in range(widths[t - 1]):
        for tau in range(1, t + 1):                   # Anc(p_i) and j = i
            M[i, L + offs[tau - 1] + chain[i, tau - 1]] = True
    return M


def sequence_expanded_attention(K_prefix: np.ndarray, V_prefix: np.ndarray,
                                k_levels: List[np.ndarray], v_levels: List[np.ndarray],
                                parents: Sequence[np.ndarray], q_t: np.ndarray, t: int,
                                scale: float) -> np.ndarray:
    """Attention outputs [W_t, Hq, D] of the level-t tokens, computed as ONE
    masked attention over the single expanded sequence (every K/V row stored
    once).  `k_levels[l-1]` is [W_l, Hkv, D]."""
    L = K_prefix.shape[0]
    if t == 0:
        mask = np.ones((q_t.shape[0], L), dtype=bool)
        return masked_attention(q_t, K_prefix, V_prefix, mask, scale)
    K = np.concatenate([np.asarray(K_prefix, np.float64)] + [np.asarray(k, np.float64) for k in k_levels[:t]], axis=0)
    V = np.concatenate([np.asarray(V_prefix, np.float64)] + [np.asarray(v, np.float64) for v in v_levels[:t]], axis=0)
    return masked_attention(q_t, K, V, tree_mask(parents, t, L), scale)
