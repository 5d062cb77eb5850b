"""Per-level beam selection (oracle; test infrastructure).

Beam score = sum of per-level log-probabilities (Eq. 1:
P(v) = prod_j P(c_j | x_u, S_u, c_<j)); each level keeps the top-W candidate
paths.

Readings: R4 the key is ONE fp32 addition; R5 no length
normalisation; R6 order = key descending, flat index (i*C + c) ascending,
IEEE comparison (-0.0 == +0.0, -inf legal and last); R7 W_out = min(W, W_in*C).
"""
from __future__ import annotations

from typing import Tuple

import numpy as np


def log_softmax_fp32(logits: np.ndarray) -> np.ndarray:
    """logp = logits - logsumexp(logits) in fp64, then
    rounded ONCE to fp32 (round-to-nearest).  Last axis is the codebook."""
    x = np.asarray(logits, dtype=np.float64)
    m = np.max(x, axis=-1, keepdims=True)
    lse = m + np.log(np.sum(np.exp(x - m), axis=-1, keepdims=True))
    return (x - lse).astype(np.float32)


def select_beams(score: np.ndarray, logp: np.ndarray, W_out: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """SURVEY.md §8c step O4 for one user.

    score[W_in] fp32, logp[W_in, C] fp32.  key[i*C + c] = fl32(score[i] +
    logp[i, c]).  Returns the W_out entries first in the order (key descending,
    flat index ascending): (out_score[W_out] fp32, parent[W_out] int32,
    code[W_out] int32).
    """
    score = np.asarray(score, dtype=np.float32)
    logp = np.asarray(logp, dtype=np.float32)
    W_in, C = logp.shape
    assert score.shape == (W_in,)
    assert 0 < W_out <= W_in * C
    key = (score[:, None] + logp).astype(np.float32).reshape(-1)      # one fp32 add
    idx = np.arange(W_in * C, dtype=np.int64)
    # lexicographic sort: primary = key descending, secondary = index ascending.
    # np.lexsort sorts by the LAST key first.  (-key) maps -0.0/+0.0 to +0.0/-0.0,
    # which compare equal, so the index decides, as IEEE comparison requires.
    order = np.lexsort((idx, -key))[:W_out]
    return key[order].copy(), (order // C).astype(np.int32), (order % C).astype(np.int32)


def row_offset_fp32(score: np.ndarray, logits: np.ndarray) -> np.ndarray:
    """Selection straight from raw logits (reading R22).

    Eq. 1 needs log P(c | ...) = logit_c - logsumexp(logits);
    the normaliser is one scalar per parent beam, so it is folded into the
    beam's running score instead of being subtracted from every candidate:
        lse[i]    = fl32( logsumexp_c logits[i, c] )      (fp64, rounded once)
        offset[i] = fl32( score[i] - lse[i] )             (one fp32 subtraction)
    A row whose logits are all -inf (a beam with no legal continuation) has
    offset = -inf by definition, so that its keys are -inf and never NaN.
    score[W_in] fp32, logits[W_in, C] fp32 -> offset[W_in] fp32."""
    score = np.asarray(score, dtype=np.float32)
    x = np.asarray(logits, dtype=np.float32).astype(np.float64)
    m = np.max(x, axis=-1)
    dead = np.isneginf(m)
    msafe = np.where(dead, 0.0, m)
    with np.errstate(divide="ignore"):
        lse = msafe + np.log(np.sum(np.exp(x - msafe[:, None]), axis=-1))
    lse32 = lse.astype(np.float32)
    off = (score - lse32).astype(np.float32)
    return np.where(dead, np.float32(-np.inf), off).astype(np.float32)


def select_beams_from_logits(score: np.ndarray, logits: np.ndarray, W_out: int):
    """Reading R22: key[i*C + c] = fl32(offset[i] + logits[i, c]) with
    offset = row_offset_fp32(score, logits); then exactly step O4's selection
    (key descending, flat index ascending).  Same value as score + logp up to
    the rounding of two fp32 operations."""
    return select_beams(row_offset_fp32(score, logits), np.asarray(logits, dtype=np.float32), W_out)
