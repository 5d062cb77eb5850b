"""The paper's encoder-decoder form of the decode attention, the ranking-feature step and target attention
(oracle; test infrastructure).  SURVEY.md section 8(f) item 3; readings R23-R25.

BASELINE.json's configs take ONE softmax over [prefix ++ suffix] (reading R1).  The paper's own decoder is an
encoder-decoder: a decoder position attends
  * through CROSS-attention to the encoder memory M ("conditioned on M through cross-attention")
    -- a softmax over the rows of M ALONE, the same M for every beam of a user;
  * through causal SELF-attention to the decoder sequence X_dec = [e_click, e_atc, e_pay, <bos>, s_1, s_2, ...]
    (Eq. 7): "all semantic ID tokens can attend to preceding task tokens", i.e. a level-t
    token sees the 4 fixed prefix positions plus its own ancestor chain under the tree mask of Eq. 14
     -- a SEPARATE softmax over those 4 + t keys.
After the last selection "decoder outputs at <bos>, s_1, s_2, ... serve as task-aware features" for ranking
(PAPER.md:215): the final-level tokens are run once more (step t = d) and every final beam reads the hidden
states along its own path.  The ranking module's target attention "applies cross-attention over the behavior
sequence encoder representations using candidate semantic IDs": one query per candidate over M.

All of it is ordinary softmax attention (oracle/attention.py) over differently assembled key sets, written in
the conventional form: every beam owns a replicated copy of what it attends to.  fp64 throughout.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np

from .attention import beam_attention

N_FIXED = 4      # e_click, e_atc, e_pay, <bos>  (Eq. 7)


def cross_attention(q: np.ndarray, K_M: np.ndarray, V_M: np.ndarray, scale: float) -> np.ndarray:
    """queries q[n,Hq,D] over the encoder memory K_M, V_M [L,Hkv,D]; softmax over M alone.
    Conventional form: every query (beam) gets its own copy of M.  -> [n,Hq,D]."""
    K_M = np.asarray(K_M, dtype=np.float64)
    V_M = np.asarray(V_M, dtype=np.float64)
    return np.stack([beam_attention(np.asarray(q[i], dtype=np.float64), K_M.copy(), V_M.copy(), scale)
                     for i in range(q.shape[0])])


def target_attention(q_cand: np.ndarray, K_M: np.ndarray, V_M: np.ndarray, scale: float) -> np.ndarray:
    """one query per candidate SID path over the encoder representations of the behaviour
    sequence.  The same operation as cross_attention (kept apart because it is a different call site: the
    queries are the W_d final candidates, after decoding)."""
    return cross_attention(q_cand, K_M, V_M, scale)


def self_tree_attention(q_t: np.ndarray, K_fix: np.ndarray, V_fix: np.ndarray, k_levels: List[np.ndarray],
                        v_levels: List[np.ndarray], parents: Sequence[np.ndarray], t: int,
                        scale: float) -> np.ndarray:
    """Causal self-attention of the level-t tokens over the decoder sequence (Eq. 7 + Eq. 14), conventional
    form: beam i owns a private sequence [e_click, e_atc, e_pay, <bos>] ++ (its ancestors' tokens, depth
    1..t, itself included), built level by level by copying the parent's sequence.
    q_t [W_t,Hq,D]; K_fix, V_fix [4,Hkv,D]; k_levels[l-1] [W_l,Hkv,D]; parents[l-1][s] = slot at level l-1 of
    the parent of slot s of level l (parents[0] ignored: level-1 tokens hang off <bos>).  -> [W_t,Hq,D]."""
    Kf = np.asarray(K_fix, dtype=np.float64)
    Vf = np.asarray(V_fix, dtype=np.float64)
    assert Kf.shape[0] == N_FIXED
    seqs = [(Kf.copy(), Vf.copy())]                      # level 0: the sequence that ends in <bos>
    for l in range(1, t + 1):
        new = []
        for s_ in range(len(parents[l - 1])):
            p = 0 if l == 1 else int(parents[l - 1][s_])
            Kc, Vc = seqs[p]
            new.append((np.concatenate([Kc.copy(), np.asarray(k_levels[l - 1][s_], np.float64)[None]], axis=0),
                        np.concatenate([Vc.copy(), np.asarray(v_levels[l - 1][s_], np.float64)[None]], axis=0)))
        seqs = new
    q_t = np.asarray(q_t, dtype=np.float64)
    assert len(seqs) == q_t.shape[0]
    return np.stack([beam_attention(q_t[i], seqs[i][0], seqs[i][1], scale) for i in range(q_t.shape[0])])


def cross_plus_self_attention(q_cross: np.ndarray, q_self: np.ndarray, K_M: np.ndarray, V_M: np.ndarray,
                              K_fix: np.ndarray, V_fix: np.ndarray, k_levels: List[np.ndarray],
                              v_levels: List[np.ndarray], parents: Sequence[np.ndarray], t: int,
                              scale: float) -> Tuple[np.ndarray, np.ndarray]:
    """One encoder-decoder layer's two attention sub-layers for the level-t tokens: (cross over M,
    self over [TAT, <bos>] + ancestor chain) -- two separate softmaxes (reading R23)."""
    return (cross_attention(q_cross, K_M, V_M, scale),
            self_tree_attention(q_self, K_fix, V_fix, k_levels, v_levels, parents, t, scale))


def path_hidden_states(outs: Sequence[np.ndarray], parents: Sequence[np.ndarray]) -> np.ndarray:
    """the decoder outputs at <bos>, s_1, ..., s_d of every FINAL beam (reading R24).
    outs[t] [W_t, ...] = decoder output of the level-t tokens (outs[0] has the single <bos> row; outs[d] comes
    from the extra step t = d); parents as above, len d.  Conventional form: every hypothesis carries its own
    list of outputs, and the lists are duplicated and rearranged with the beams after every selection.
    -> [W_d, d + 1, ...]."""
    d = len(parents)
    hist = [[np.asarray(outs[0][0])]]                    # level 0: one hypothesis, its <bos> output
    for l in range(1, d + 1):
        new = []
        for s_ in range(len(parents[l - 1])):
            p = 0 if l == 1 else int(parents[l - 1][s_])
            new.append([h.copy() for h in hist[p]] + [np.asarray(outs[l][s_])])
        hist = new
    return np.stack([np.stack(h) for h in hist])
