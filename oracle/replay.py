"""Teacher-forced replay of ONE decode step in the conventional form (oracle;
test infrastructure).

Per-call attention parity (SURVEY.md §8c "comparison protocol") runs the GPU
and the oracle on the identical tree: same prefix, same per-level k_new/v_new,
same parent pointers, same queries.  The oracle side stays conventional
(PAPER.md:257-259): it rebuilds every beam's private cache by duplicating its
parent's cache and appending the beam's own token, then runs ordinary
full-sequence attention per beam.
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np

from .attention import beam_attention


def _replicated_caches(K_prefix, V_prefix, k_levels, v_levels, parents, t):
    """Caches of all level-t beams, built level by level with deep copies."""
    Kp = np.asarray(K_prefix, dtype=np.float64)
    Vp = np.asarray(V_prefix, dtype=np.float64)
    caches = [(Kp.copy(), Vp.copy())]                     # level 0: the root
    for l in range(1, t + 1):
        new = []
        for s in range(len(parents[l - 1])):
            p = 0 if l == 1 else int(parents[l - 1][s])
            Kc, Vc = caches[p]
            new.append((np.concatenate([Kc.copy(), np.asarray(k_levels[l - 1][s], np.float64)[None]], axis=0),
                        np.concatenate([Vc.copy(), np.asarray(v_levels[l - 1][s], np.float64)[None]], axis=0)))
        caches = new
    return caches


def replay_step_attention(K_prefix: np.ndarray, V_prefix: np.ndarray,
                          k_levels: List[np.ndarray], v_levels: List[np.ndarray],
                          parents: Sequence[np.ndarray], q_t: np.ndarray, t: int,
                          scale: float) -> np.ndarray:
    """All beams of one user at step t -> [n_q, Hq, D] fp64."""
    caches = _replicated_caches(K_prefix, V_prefix, k_levels, v_levels, parents, t)
    q_t = np.asarray(q_t, dtype=np.float64)
    assert len(caches) == q_t.shape[0]
    return np.stack([beam_attention(q_t[i], caches[i][0], caches[i][1], scale) for i in range(q_t.shape[0])])


def replay_beam_attention(K_prefix: np.ndarray, V_prefix: np.ndarray,
                          k_levels: List[np.ndarray], v_levels: List[np.ndarray],
                          parents: Sequence[np.ndarray], q_i: np.ndarray, slot: int, t: int,
                          scale: float) -> np.ndarray:
    """ONE sampled beam (for full-size configs where replaying every beam is
    too slow): its own full sequence = prefix ++ the K/V of its ancestors from
    depth 1 to depth t, gathered by following the parent pointers upward, then
    ordinary attention -> [Hq, D] fp64."""
    rows_k, rows_v = [], []
    a = slot
    for l in range(t, 0, -1):
        rows_k.append(np.asarray(k_levels[l - 1][a], dtype=np.float64))
        rows_v.append(np.asarray(v_levels[l - 1][a], dtype=np.float64))
        if l > 1:
            a = int(parents[l - 1][a])
    Kc = np.asarray(K_prefix, dtype=np.float64)
    Vc = np.asarray(V_prefix, dtype=np.float64)
    if rows_k:
        Kc = np.concatenate([Kc, np.stack(rows_k[::-1])], axis=0)
        Vc = np.concatenate([Vc, np.stack(rows_v[::-1])], axis=0)
    return beam_attention(np.asarray(q_i, dtype=np.float64), Kc, Vc, scale)
