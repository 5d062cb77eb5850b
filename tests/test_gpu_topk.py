"""GPU parity of stark_beam_topk (row A3) on adversarial inputs, bit-exact vs oracle.select_beams
("adversarial exact ties, -inf blocks, W_out = W_in*C"; reading R6: key descending,
flat index ascending, -0.0 == +0.0).  Every case exercises a different branch of the kernel: early exit after
one radix pass, all three passes, the boundary-value tie path (ordered by index, across cluster ranks), the
all-keys-equal shortcut, non-power-of-two codebooks, slices larger than the shared-memory cache."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _check(logp, score, W_out):
    import torch
    from oracle.selection import select_beams
    from paper_2607_04068_b200.decode import beam_topk
    B, W_in, C = logp.shape
    lp = torch.from_numpy(logp).cuda()
    sc = None if score is None else torch.from_numpy(score).cuda()
    s_g, p_g, c_g = [x.cpu().numpy() for x in beam_topk(lp, sc, W_out)]
    for u in range(B):
        s_r, p_r, c_r = select_beams(np.zeros(W_in, np.float32) if score is None else score[u], logp[u], W_out)
        assert np.array_equal(p_g[u], p_r), f"user {u}: parent differs"
        assert np.array_equal(c_g[u], c_r), f"user {u}: code differs"
        assert np.array_equal(s_g[u].view(np.uint32), s_r.view(np.uint32)), f"user {u}: score bits differ"


def _rng(tag):
    return np.random.default_rng([0, 77, tag])


@pytest.mark.parametrize("B,W_in,C,W_out", [
    (3, 1, 32, 8), (2, 1, 256, 256), (5, 24, 48, 24), (2, 64, 256, 64), (2, 96, 160, 96),
    (1, 512, 1024, 512), (3, 7, 33, 231), (2, 40, 97, 100), (1, 16, 8192, 512), (2, 130, 1000, 4096),
])
def test_random_logprobs(B, W_in, C, W_out):
    r = _rng(1)
    logits = r.normal(0, 2, (B, W_in, C))
    logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
    score = None if W_in == 1 else np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
    _check(logp, score, W_out)


@pytest.mark.parametrize("B,W_in,C,W_out", [(2, 64, 256, 64), (1, 512, 1024, 512), (3, 20, 50, 70)])
def test_quantised_ties(B, W_in, C, W_out):
    """Keys on a 1/8 grid: thousands of exact ties, the boundary value repeats far beyond the sort buffer."""
    r = _rng(2)
    logp = (np.round(r.normal(-6, 1.5, (B, W_in, C)) * 8) / 8).astype(np.float32)
    score = (np.round(r.normal(-4, 1, (B, W_in)) * 8) / 8).astype(np.float32)
    _check(logp, score, W_out)


def test_all_equal_and_signed_zero():
    logp = np.zeros((2, 16, 128), np.float32)
    logp[0, ::2] = -0.0                      # -0.0 == +0.0: index order decides
    _check(logp, None, 200)
    _check(np.full((1, 64, 256), -3.25, np.float32), np.zeros((1, 64), np.float32), 64)
    _check(np.full((2, 300, 512), -1.0, np.float32), None, 4096)


def test_neg_inf_blocks():
    r = _rng(3)
    logp = r.normal(-5, 1, (2, 32, 256)).astype(np.float32)
    logp[:, :, 10:] = -np.inf                # only 10 finite codes per beam: 320 finite keys
    score = r.normal(-3, 1, (2, 32)).astype(np.float32)
    _check(logp, score, 64)                  # all finite
    _check(logp, score, 512)                 # 320 finite + 192 of the -inf keys, by index
    logp[1] = -np.inf
    _check(logp, score, 33)


def test_two_values_boundary_inside_huge_tie():
    """One distinct large key + a sea of equal keys: radix range is wide, boundary falls inside the tie."""
    logp = np.full((2, 128, 512), -7.5, np.float32)
    logp[0, 5, 17] = -0.125
    logp[1, 127, 511] = -0.125
    _check(logp, None, 300)


def test_slice_larger_than_cache():
    """B = 1, 2^20 candidates: slices exceed the shared-memory cache, later passes re-read through L2."""
    r = _rng(4)
    logp = r.normal(-9, 2, (1, 128, 8192)).astype(np.float32)
    score = r.normal(-5, 1, (1, 128)).astype(np.float32)
    _check(logp, score, 1024)
    _check((np.round(logp * 4) / 4).astype(np.float32), (np.round(score * 4) / 4).astype(np.float32), 1024)


def test_streamed_tail_with_sorted_parent_scores():
    """The realistic large case: parent scores arrive sorted (best beams first), slices are larger than the
    cache, so the tail is streamed once against a bound that is re-tightened from the survivor list; also with a
    late burst (the best parent LAST), which overflows the list and takes the fallback."""
    r = _rng(5)
    logits = r.normal(0, 2, (2, 128, 8192))
    logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
    score = np.sort(r.normal(-8, 2, (2, 128)).astype(np.float32))[:, ::-1].copy()
    _check(logp, score, 512)
    _check(logp, score[:, ::-1].copy(), 512)
    score2 = score.copy(); score2[:, -1] = 5.0
    _check(logp, score2, 300)


def test_small_direct_path():
    """N <= 512 candidates per user (decode step 0 of a 256-code level) take the one-CTA rank-by-counting
    kernel (1 or 2 candidates per thread): ragged and odd N, N = 256 / 512 exactly, W_out = N, massive ties,
    signed zeros, -inf; N = 513 .. 1024 sits just above it."""
    r = _rng(6)
    for (B, W_in, C, W_out) in [(16, 1, 256, 64), (2, 2, 256, 512), (3, 15, 31, 400), (2, 1, 1, 1), (5, 1, 255, 7),
                               (2, 19, 27, 513), (2, 4, 256, 1024), (3, 3, 85, 200)]:
        logp = r.normal(-5, 2, (B, W_in, C)).astype(np.float32)
        score = None if W_in == 1 else r.normal(-3, 1, (B, W_in)).astype(np.float32)
        _check(logp, score, W_out)
        q = (np.round(logp * 2) / 2).astype(np.float32)          # ties everywhere: index order decides
        _check(q, None if score is None else (np.round(score * 2) / 2).astype(np.float32), W_out)
    z = np.zeros((2, 4, 128), np.float32); z[0, ::2] = -0.0; z[1, :, 5:] = -np.inf
    _check(z, None, 100)
    _check(z, np.zeros((2, 4), np.float32), 512)


def test_mid_single_cta_path():
    """512 < N <= 16384 candidates per user and W_out <= 256: one 1024-thread CTA per user (bound from the
    per-thread maxima, survivors ranked by counting; massive ties take the exact radix select + index-order tie
    pick).  Ragged N, W_out = 1024, ties far beyond the list (and the sizes just outside the path), all keys equal, -inf blocks, signed zeros."""
    r = _rng(7)
    for (B, W_in, C, W_out) in [(16, 64, 256, 64), (3, 33, 300, 200), (2, 1, 8192, 256), (2, 16, 1024, 1),
                               (4, 7, 77, 255), (2, 3, 171, 256), (1, 64, 256, 129), (2, 1, 16385, 5)]:
        logits = r.normal(0, 2, (B, W_in, C))
        logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
        score = None if W_in == 1 else np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
        _check(logp, score, W_out)
        q = (np.round(logp) ).astype(np.float32)                  # integer grid: ties in the thousands
        _check(q, None if score is None else np.round(score).astype(np.float32), W_out)
    _check(np.full((2, 64, 256), -2.5, np.float32), None, 200)     # all equal: index order only
    z = np.zeros((2, 32, 512), np.float32); z[0, ::2] = -0.0; z[1, :, 3:] = -np.inf
    _check(z, None, 100)
    _check(z, np.zeros((2, 32), np.float32), 256)
    w = r.normal(-4, 1, (1, 40, 400)).astype(np.float32); w[0, :, 5:] = -np.inf; w[0, 39, 399] = 3.0
    _check(w, r.normal(0, 1, (1, 40)).astype(np.float32), 256)   # 201 finite keys + 55 of the -inf ties


def test_wide_selection_over_small_candidate_sets():
    """512 < N <= 8192 candidates per user and 256 < W_out <= 1024 (decode step 0 with a wide beam: PAPER.md:306,
    512 of 8192 codes; config 4, 512 of 1024): R independent CTAs per user, bound by bisection, every CTA ranks a
    slice (topk_wide_kernel).  Ragged N and C, W_out = N, many users (fewer CTAs each), ties by the thousand (the
    second bisection, on the index), all keys equal, -inf blocks, signed zeros, the sizes just outside the path."""
    r = _rng(11)
    for (B, W_in, C, W_out) in [(8, 1, 1024, 512), (8, 1, 8192, 512), (1, 1, 8192, 1024), (3, 7, 333, 700),
                               (2, 19, 27, 513), (2, 4, 256, 1024), (2, 1, 1000, 1000), (40, 1, 2048, 300),
                               (300, 1, 600, 257), (2, 1, 8192, 1025), (2, 1, 8193, 512), (1, 3, 2731, 1024)]:
        logits = r.normal(0, 2, (B, W_in, C))
        logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
        score = None if W_in == 1 else np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
        _check(logp, score, W_out)
        if B <= 8:
            q = np.round(logp).astype(np.float32)                 # integer grid: ties in the thousands
            _check(q, None if score is None else np.round(score).astype(np.float32), W_out)
    _check(np.full((2, 4, 2048), -2.5, np.float32), None, 900)    # all equal: index order only
    _check(np.full((1, 1, 8192), 0.0, np.float32), None, 1024)
    z = np.zeros((2, 8, 512), np.float32); z[0, ::2] = -0.0; z[1, :, 3:] = -np.inf
    _check(z, None, 400)
    _check(z, np.zeros((2, 8), np.float32), 1024)
    w = r.normal(-4, 1, (1, 10, 800)).astype(np.float32); w[0, :, 30:] = -np.inf; w[0, 9, 799] = 3.0
    _check(w, r.normal(0, 1, (1, 10)).astype(np.float32), 512)   # 301 finite keys + 211 of the -inf ties
    two = np.where(r.random((2, 1, 4096)) < 0.1, np.float32(-1.0), np.float32(-2.0)).astype(np.float32)
    _check(two, None, 600)                                        # the boundary falls inside a huge tie


@pytest.mark.parametrize("W_out", [1025, 1536, 2048, 3000])
@pytest.mark.parametrize("B,W_in,C", [(2, 64, 1024), (1, 512, 1024), (1, 128, 8192), (3, 40, 1000)])
def test_wide_outputs_above_1024(B, W_in, C, W_out):
    """1024 < W_out <= 4096 at N >= 32768 (the shared-memory sizing of the pruned cluster kernel):
    random keys with sorted parent scores, and a tie-heavy 1/4 grid."""
    r = _rng(8)
    logits = r.normal(0, 2, (B, W_in, C))
    logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
    score = np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
    _check(logp, score, W_out)
    _check((np.round(logp * 4) / 4).astype(np.float32), (np.round(score * 4) / 4).astype(np.float32), W_out)


def test_cfg4_full_size_exact_tie_variant():
    """"plus an extra exact-tie variant (logits rounded to 1/8) for parity
    only" at FULL size (8 users x 512 beams x 1024 codes, W_out = 512), every level, all users, through both
    entries (log-probs and raw logits).  The tree is the oracle's (scores of level t come from its selection of
    level t-1), so every level is checked on its own."""
    import torch
    import workloads as wl
    from oracle.selection import log_softmax_fp32, select_beams, select_beams_from_logits
    from paper_2607_04068_b200.decode import beam_topk, beam_topk_logits
    cfg = wl.get_config("cfg4")
    nq, widths = wl.queries_per_step(cfg), wl.beam_widths(cfg)
    for from_logits in (False, True):
        score = None
        for t in range(cfg.d):
            lg = wl.tie_logits(wl.step_logits(cfg, t, nq[t]))
            assert np.array_equal(lg * 8, np.round(lg * 8))
            x = lg if from_logits else log_softmax_fp32(lg)
            sc = None if score is None else torch.from_numpy(score).cuda()
            fn = beam_topk_logits if from_logits else beam_topk
            s_g, p_g, c_g = [a.cpu().numpy() for a in fn(torch.from_numpy(x).cuda(), sc, widths[t])]
            nxt = []
            for u in range(cfg.B):
                s_u = np.zeros(nq[t], np.float32) if score is None else score[u]
                s_r, p_r, c_r = (select_beams_from_logits if from_logits else select_beams)(s_u, x[u], widths[t])
                assert np.array_equal(p_g[u], p_r) and np.array_equal(c_g[u], c_r), f"level {t} user {u} ({from_logits=})"
                assert np.array_equal(s_g[u].view(np.uint32), s_r.view(np.uint32)), f"level {t} user {u} score bits"
                nxt.append(s_r)
            score = np.stack(nxt)
    # the same shape with keys on an exact grid ACROSS beams (log-probs and scores both multiples of 1/8)
    r = _rng(9)
    logp = (np.round(r.normal(-7, 1.5, (cfg.B, 512, cfg.C)) * 8) / 8).astype(np.float32)
    score = np.sort((np.round(r.normal(-5, 1, (cfg.B, 512)) * 8) / 8).astype(np.float32))[:, ::-1].copy()
    _check(logp, score, 512)


def test_grid_path_shapes_and_exceptional_finishes():
    """Large candidate sets (>= 131072 per user, W_out <= 1024, C % 4 == 0) take the whole-GPU kernel
    (topk_grid.cu): non-power-of-two codebooks, chunks that span many parent beams, a ragged last chunk, several
    users; and its exceptional finishes -- every key equal / a sea of -inf (survivor lists overflow: the last CTA
    re-selects over all keys), unsorted and reversed parent scores (loose bound: more than 8192 survivors, radix
    passes + bucket ranking by the last CTA), quantised keys (ties inside and across beams)."""
    r = _rng(10)
    for (B, W_in, C, W_out) in [(2, 200, 1000, 512), (1, 4096, 64, 256), (3, 100, 1500, 700), (5, 64, 4096, 1024),
                               (1, 1024, 1024, 1), (2, 512, 512, 1000)]:
        logits = r.normal(0, 2, (B, W_in, C))
        logp = (logits - np.log(np.exp(logits).sum(-1, keepdims=True))).astype(np.float32)
        score = np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
        _check(logp, score, W_out)
        _check(logp, score[:, ::-1].copy(), W_out)                       # best parent last
        _check(logp, r.permutation(score.T).T.copy(), W_out)             # unsorted parents
        _check((np.round(logp * 4) / 4).astype(np.float32), (np.round(score * 4) / 4).astype(np.float32), W_out)
    _check(np.full((2, 512, 512), -1.0, np.float32), None, 300)          # all equal: index order only
    z = np.full((2, 256, 1024), -np.inf, np.float32)
    z[0, 3, 10:20] = -1.5; z[1, :, 7] = -2.0                             # 10 / 256 finite keys, the rest -inf
    _check(z, np.zeros((2, 256), np.float32), 512)
    z2 = np.zeros((1, 512, 512), np.float32); z2[0, ::2] = -0.0          # signed zeros, all equal
    _check(z2, None, 1024)
