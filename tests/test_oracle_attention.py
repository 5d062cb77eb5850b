"""Pins for oracle/attention.py (CPU only).

The paper prints no worked numeric example (Fig. 2 is an image),
so the oracle's attention is pinned to: a library routine
(torch.nn.functional.scaled_dot_product_attention, float64, explicit boolean
mask), hand-computed closed forms, and invariants of softmax attention.
Each test names the mistake it would catch.
"""
import math

import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle.attention import beam_attention, masked_attention, softmax_attention_single


def _sdpa(Q, K, V, mask, scale, G):
    # Q[n,Hq,D], K/V[S,Hkv,D] -> torch layout [1,H,n,D]; GQA by repeating KV heads
    q = torch.from_numpy(Q).permute(1, 0, 2)[None]
    k = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    v = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    m = torch.from_numpy(mask)[None, None]
    o = F.scaled_dot_product_attention(q, k, v, attn_mask=m, scale=scale)
    return o[0].permute(1, 0, 2).numpy()


def test_hand_computed_two_keys():
    # scores (scale 1): 0 and ln 3  ->  weights 1/4, 3/4  ->  out = [3, 1]
    q = np.array([1.0, 0.0])
    K = np.array([[0.0, 7.0], [math.log(3.0), -2.0]])
    V = np.array([[0.0, 4.0], [4.0, 0.0]])
    out = softmax_attention_single(q, K, V, 1.0)
    np.testing.assert_allclose(out, [3.0, 1.0], rtol=0, atol=1e-14)
    # the scale multiplies the score: with scale 2 the second score is ln 9 -> 1/10, 9/10
    out2 = softmax_attention_single(q, K, V, 2.0)
    np.testing.assert_allclose(out2, [3.6, 0.4], rtol=0, atol=1e-14)


def test_masked_attention_equals_library_sdpa():
    rng = np.random.default_rng(1)
    n, S, Hq, Hkv, D = 7, 29, 6, 2, 16
    Q = rng.standard_normal((n, Hq, D))
    K = rng.standard_normal((S, Hkv, D))
    V = rng.standard_normal((S, Hkv, D))
    mask = rng.random((n, S)) < 0.6
    mask[:, 0] = True                               # no fully-masked row
    scale = 1.0 / math.sqrt(D)
    got = masked_attention(Q, K, V, mask, scale)
    ref = _sdpa(Q, K, V, mask, scale, Hq // Hkv)
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-13)


def test_beam_attention_equals_library_sdpa_full_sequence():
    rng = np.random.default_rng(2)
    L, Hq, Hkv, D = 41, 8, 2, 32
    q = rng.standard_normal((Hq, D))
    K = rng.standard_normal((L, Hkv, D))
    V = rng.standard_normal((L, Hkv, D))
    scale = 0.37
    got = beam_attention(q, K, V, scale)
    ref = _sdpa(q[None], K, V, np.ones((1, L), dtype=bool), scale, Hq // Hkv)[0]
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-13)


def test_gqa_head_mapping_is_h_div_G():
    # V constant per KV head -> out[h] must be the constant of head h // G
    # (catches h % Hkv and transposed head axes)
    rng = np.random.default_rng(3)
    L, Hq, Hkv, D = 9, 8, 2, 4
    q = rng.standard_normal((Hq, D))
    K = rng.standard_normal((L, Hkv, D))
    V = np.empty((L, Hkv, D))
    V[:, 0, :] = 10.0
    V[:, 1, :] = -5.0
    out = beam_attention(q, K, V, 0.5)
    np.testing.assert_allclose(out[:4], 10.0, atol=1e-12)
    np.testing.assert_allclose(out[4:], -5.0, atol=1e-12)


def test_zero_keys_give_mean_of_values():
    rng = np.random.default_rng(4)
    L, D = 13, 5
    V = rng.standard_normal((L, D))
    out = softmax_attention_single(rng.standard_normal(D), np.zeros((L, D)), V, 0.3)
    np.testing.assert_allclose(out, V.mean(axis=0), atol=1e-14)


def test_dominant_score_selects_that_value_row():
    rng = np.random.default_rng(5)
    L, D = 11, 6
    q = np.zeros(D)
    q[0] = 1.0
    K = rng.standard_normal((L, D)) * 0.01
    K[7, 0] = 1000.0
    V = rng.standard_normal((L, D))
    out = softmax_attention_single(q, K, V, 1.0)
    np.testing.assert_allclose(out, V[7], atol=1e-12)


def test_invariants_shift_convexity_permutation():
    rng = np.random.default_rng(6)
    L, D = 17, 8
    q = rng.standard_normal(D)
    K = rng.standard_normal((L, D))
    V = rng.standard_normal((L, D))
    out = softmax_attention_single(q, K, V, 0.25)
    # every output coordinate lies in the convex hull of the V rows
    assert np.all(out <= V.max(axis=0) + 1e-12) and np.all(out >= V.min(axis=0) - 1e-12)
    # adding the same constant to every score changes nothing: K_j += w with <q,w> = c
    w = q / np.dot(q, q) * 123.0
    np.testing.assert_allclose(softmax_attention_single(q, K + w, V, 0.25), out, atol=1e-9)
    # large scores do not overflow (max subtraction)
    big = softmax_attention_single(q * 1e4, K, V, 1.0)
    assert np.all(np.isfinite(big))
    # attention is a set function of (K_j, V_j) pairs
    perm = rng.permutation(L)
    np.testing.assert_allclose(softmax_attention_single(q, K[perm], V[perm], 0.25), out, atol=1e-13)


def test_split_invariance_of_log_sum_exp_merge():
    # The (m, l, o) partial format (R18): merging partial softmaxes over
    # any partition of the keys gives the unsplit result.  This pins the identity
    # the CUDA path relies on, using only the oracle's plain attention.
    rng = np.random.default_rng(7)
    L, D = 37, 8
    q = rng.standard_normal(D)
    K = rng.standard_normal((L, D))
    V = rng.standard_normal((L, D))
    scale = 0.4
    full = softmax_attention_single(q, K, V, scale)
    for cuts in ([0, 37], [0, 5, 37], [0, 1, 2, 30, 37], [0, 18, 18, 37]):
        ms, ls, os_ = [], [], []
        for a, b in zip(cuts[:-1], cuts[1:]):
            if a == b:                                   # empty split: (-inf, 0, 0)
                ms.append(-np.inf), ls.append(0.0), os_.append(np.zeros(D))
                continue
            s = scale * (K[a:b] @ q)
            m = s.max()
            e = np.exp(s - m)
            ms.append(m), ls.append(e.sum()), os_.append(e @ V[a:b])
        M = max(ms)
        w = [0.0 if m == -np.inf else math.exp(m - M) for m in ms]
        merged = sum(wi * oi for wi, oi in zip(w, os_)) / sum(wi * li for wi, li in zip(w, ls))
        np.testing.assert_allclose(merged, full, atol=1e-13)


def test_empty_sequence_returns_zeros_not_nan():
    out = softmax_attention_single(np.ones(4), np.zeros((0, 4)), np.zeros((0, 4)), 1.0)
    assert out.shape == (4,) and np.all(out == 0.0)
