"""Pins for oracle/selection.py (CPU only): the selection is pinned to the
textbook reductions (stable sort; repeated extraction of the maximum), to
hand-made adversarial cases (exact ties, -inf blocks, signed zeros, the fp32
key rounding) and to invariants.  The log-softmax is pinned to torch's and to a
closed form.
"""
import math

import numpy as np
import pytest
import torch

from oracle.selection import log_softmax_fp32, select_beams


def _extract_max_repeatedly(score, logp, W_out):
    """Brute force straight from the sentence "keep the W best; on equal keys
    the lower flat index wins": pick the best remaining candidate W_out times."""
    key = (score[:, None].astype(np.float32) + logp.astype(np.float32)).astype(np.float32).reshape(-1)
    remaining = list(range(key.size))
    picked = []
    for _ in range(W_out):
        best = remaining[0]
        for j in remaining[1:]:
            if key[j] > key[best]:            # strict: an equal key never displaces a lower index
                best = j
        picked.append(best)
        remaining.remove(best)
    C = logp.shape[1]
    pk = np.array(picked)
    return key[pk], (pk // C).astype(np.int32), (pk % C).astype(np.int32)


def _stable_sort(score, logp, W_out):
    key = (score[:, None].astype(np.float32) + logp.astype(np.float32)).astype(np.float32).reshape(-1)
    order = np.argsort(-key, kind="stable")[:W_out]
    C = logp.shape[1]
    return key[order], (order // C).astype(np.int32), (order % C).astype(np.int32)


def _same(a, b):
    assert a[0].dtype == np.float32 and b[0].dtype == np.float32
    assert np.array_equal(a[0].view(np.uint32), b[0].view(np.uint32))
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


@pytest.mark.parametrize("W_in,C,W_out", [(1, 5, 5), (1, 7, 3), (4, 6, 9), (6, 5, 30), (3, 11, 1)])
def test_matches_stable_sort_and_repeated_max(W_in, C, W_out):
    rng = np.random.default_rng(W_in * 100 + C)
    score = rng.standard_normal(W_in).astype(np.float32)
    logp = log_softmax_fp32(rng.standard_normal((W_in, C)) * 2.0)
    got = select_beams(score, logp, W_out)
    _same(got, _stable_sort(score, logp, W_out))
    _same(got, _extract_max_repeatedly(score, logp, W_out))


def test_exact_ties_resolved_by_lower_flat_index():
    rng = np.random.default_rng(11)
    W_in, C = 5, 16
    score = (np.round(rng.standard_normal(W_in) * 4) / 4).astype(np.float32)
    logp = (np.round(rng.standard_normal((W_in, C)) * 2) / 2).astype(np.float32)   # multiples of 1/2
    for W_out in (1, 7, 40, W_in * C):
        got = select_beams(score, logp, W_out)
        _same(got, _extract_max_repeatedly(score, logp, W_out))
    # all keys equal: the answer is the first W_out flat indices, in order
    s, p, c = select_beams(np.zeros(3, np.float32), np.zeros((3, 4), np.float32), 7)
    assert np.array_equal(p * 4 + c, np.arange(7))


def test_minus_inf_is_legal_and_sorts_last():
    score = np.array([0.0, -1.0], dtype=np.float32)
    logp = np.array([[-np.inf, -2.0, -np.inf], [-np.inf, -np.inf, -0.5]], dtype=np.float32)
    s, p, c = select_beams(score, logp, 5)
    # finite keys: idx 5 -> -1.5, idx 1 -> -2.0; then -inf by index: 0, 2, 3
    assert np.array_equal(p * 3 + c, [5, 1, 0, 2, 3])
    assert np.array_equal(s[:2], np.array([-1.5, -2.0], np.float32)) and np.all(np.isneginf(s[2:]))


def test_signed_zeros_compare_equal():
    score = np.array([0.0], dtype=np.float32)
    logp = np.array([[-0.0, 0.0, -0.0, -1.0]], dtype=np.float32)
    s, p, c = select_beams(score, logp, 3)
    assert np.array_equal(c, [0, 1, 2])           # index order, not sign-bit order


def test_key_is_a_single_fp32_addition():
    # fl32(1e8 - 1) == fl32(1e8 - 2) == 1e8 (ulp is 8 at 1e8): fp32 creates a tie
    # that fp64 would break the other way.  Reading R4 says fp32 decides.
    score = np.array([1e8], dtype=np.float32)
    logp = np.array([[-2.0, -1.0]], dtype=np.float32)
    s, p, c = select_beams(score, logp, 1)
    assert c[0] == 0 and s[0] == np.float32(1e8)
    # and the reported score is exactly that fp32 sum
    rng = np.random.default_rng(12)
    score = rng.standard_normal(4).astype(np.float32) * 10
    logp = log_softmax_fp32(rng.standard_normal((4, 9)))
    s, p, c = select_beams(score, logp, 6)
    assert np.array_equal(s, (score[p] + logp[p, c]).astype(np.float32))


def test_invariants():
    rng = np.random.default_rng(13)
    W_in, C, W_out = 12, 20, 50
    score = -np.abs(rng.standard_normal(W_in)).astype(np.float32)
    logp = log_softmax_fp32(rng.standard_normal((W_in, C)) * 2)
    s, p, c = select_beams(score, logp, W_out)
    assert np.all(np.diff(s) <= 0)                                    # non-increasing
    assert np.all((p >= 0) & (p < W_in) & (c >= 0) & (c < C))
    assert len({(int(a), int(b)) for a, b in zip(p, c)}) == W_out     # unique (parent, code)
    assert np.all(s <= score[p])                                      # log-probs are <= 0
    # everything left out is no better than the worst kept
    key = (score[:, None] + logp).astype(np.float32).reshape(-1)
    kept = set((p * C + c).tolist())
    rest = [key[j] for j in range(key.size) if j not in kept]
    assert max(rest) <= s[-1]


def test_log_softmax_pins():
    rng = np.random.default_rng(14)
    x = rng.standard_normal((5, 33)) * 3
    ref = torch.log_softmax(torch.from_numpy(x), dim=-1).to(torch.float32).numpy()
    got = log_softmax_fp32(x)
    assert got.dtype == np.float32 and np.array_equal(got, ref)
    # closed form: uniform logits -> -log C, whatever the offset
    u = log_softmax_fp32(np.full((1, 8), 1234.5))
    np.testing.assert_array_equal(u, np.full((1, 8), np.float32(-math.log(8.0))))
    # probabilities sum to one; huge logits do not overflow
    big = log_softmax_fp32(np.array([[1e4, 1e4 - 1.0, -1e4]]))
    assert np.all(np.isfinite(big)) and abs(np.exp(big.astype(np.float64)).sum() - 1) < 1e-6


# ---- selection from raw logits (reading R22) ---------------------------------------------------------------

def test_row_offset_matches_library_logsumexp_and_closed_forms():
    from scipy.special import logsumexp
    from oracle.selection import row_offset_fp32
    rng = np.random.default_rng(5)
    logits = (rng.standard_normal((37, 301)) * 2).astype(np.float32)
    score = rng.standard_normal(37).astype(np.float32)
    off = row_offset_fp32(score, logits)
    ref = (score - logsumexp(logits.astype(np.float64), axis=-1).astype(np.float32)).astype(np.float32)
    assert off.dtype == np.float32 and np.array_equal(off, ref)
    # closed form: C equal logits a  =>  lse = a + ln C
    for C in (1, 2, 8, 1000):
        a = np.float32(1.75)
        o = row_offset_fp32(np.zeros(1, np.float32), np.full((1, C), a, np.float32))
        assert o[0] == np.float32(-np.float32(float(a) + math.log(C)))
    # one dominant logit: lse -> that logit
    big = np.full((1, 64), -200.0, np.float32); big[0, 17] = 3.0
    assert row_offset_fp32(np.float32([0.5]), big)[0] == np.float32(0.5 - 3.0)
    # huge logits do not overflow (max subtraction); dead rows give -inf, not NaN
    assert row_offset_fp32(np.float32([0.0]), np.full((1, 4), 1e30, np.float32))[0] == np.float32(-1e30)
    dead = row_offset_fp32(np.float32([0.0, 1.0]), np.float32([[-np.inf] * 3, [0.0, -np.inf, -np.inf]]))
    assert np.isneginf(dead[0]) and dead[1] == np.float32(1.0)


def test_select_from_logits_agrees_with_logprob_selection():
    """The folded key differs from fl32(score + logp) by at most a few ulp, so: the keys agree to
    4 ulp-of-magnitude, probabilities of a row still sum to 1, and on inputs with wide margins
    (logits on a coarse grid of distinct values) the selected (parent, code) lists are identical."""
    from oracle.selection import select_beams_from_logits, row_offset_fp32
    rng = np.random.default_rng(11)
    W_in, C, W_out = 12, 40, 30
    logits = rng.permutation(W_in * C).reshape(W_in, C).astype(np.float32) * np.float32(0.03125) - 7
    score = -rng.random(W_in).astype(np.float32)
    s1, p1, c1 = select_beams_from_logits(score, logits, W_out)
    s0, p0, c0 = select_beams(score, log_softmax_fp32(logits), W_out)
    assert np.array_equal(p1, p0) and np.array_equal(c1, c0)
    assert np.max(np.abs(s1.astype(np.float64) - s0)) <= 4 * np.spacing(np.float32(np.max(np.abs(s0))))
    off = row_offset_fp32(np.zeros(W_in, np.float32), logits)
    total = np.exp((off[:, None] + logits).astype(np.float64)).sum(axis=-1)
    assert np.allclose(total, 1.0, atol=1e-5)


def test_select_from_logits_shift_invariance_and_ties():
    """Adding a power-of-two-exact constant to every logit of a row changes nothing that is selected
    when all quantities stay exactly representable; exact ties go to the lower flat index."""
    from oracle.selection import select_beams_from_logits
    logits = np.float32([[0.0, 0.0, -1.0, 0.0], [0.0, -1.0, 0.0, 0.0]])
    score = np.float32([0.0, 0.0])
    s, p, c = select_beams_from_logits(score, logits, 5)
    # both rows have the same multiset of logits => same lse => keys tie across rows; index order decides
    assert list(zip(p.tolist(), c.tolist())) == [(0, 0), (0, 1), (0, 3), (1, 0), (1, 2)]
    assert np.all(s == s[0])
    shifted = logits + np.float32([[8.0], [-16.0]])
    s2, p2, c2 = select_beams_from_logits(score, shifted, 5)
    assert np.array_equal(p2, p) and np.array_equal(c2, c)
    assert np.allclose(s2, s, atol=1e-6)
    # a dead row (all -inf) sorts last and yields -inf keys, never NaN
    lg = np.float32([[-np.inf, -np.inf], [0.0, 1.0]])
    s3, p3, c3 = select_beams_from_logits(np.float32([5.0, 0.0]), lg, 4)
    assert p3.tolist() == [1, 1, 0, 0] and c3.tolist() == [1, 0, 0, 1]
    assert not np.any(np.isnan(s3)) and np.all(np.isneginf(s3[2:]))
