"""GPU parity of stark_logits_row_offset / stark_beam_topk_logits (include/stark.h A3', reading R22) against
oracle.selection.row_offset_fp32 / select_beams_from_logits: the per-beam offsets bitwise, the selection
(parent, code) as integers and the scores bitwise.  Shapes: warp-per-row and CTA-per-row paths, rows longer
than the register cache, codebooks that are not a multiple of 4 (scalar loads), -inf masks, dead beams."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _rng(tag):
    return np.random.default_rng([0, 78, tag])


def _check(logits, score, W_out):
    import torch
    from oracle.selection import row_offset_fp32, select_beams_from_logits
    from paper_2607_04068_b200 import stark_logits_row_offset
    from paper_2607_04068_b200.decode import beam_topk_logits
    B, W_in, C = logits.shape
    lg = torch.from_numpy(logits).cuda()
    sc = None if score is None else torch.from_numpy(score).cuda()
    off = torch.empty((B, W_in), dtype=torch.float32, device="cuda")
    stark_logits_row_offset(lg, sc, B * W_in, C, off)
    s_g, p_g, c_g = [x.cpu().numpy() for x in beam_topk_logits(lg, sc, W_out)]
    off = off.cpu().numpy()
    for u in range(B):
        s_u = np.zeros(W_in, np.float32) if score is None else score[u]
        assert np.array_equal(off[u].view(np.uint32), row_offset_fp32(s_u, logits[u]).view(np.uint32)), \
            f"user {u}: offset bits differ"
        s_r, p_r, c_r = select_beams_from_logits(s_u, logits[u], W_out)
        assert np.array_equal(p_g[u], p_r), f"user {u}: parent differs"
        assert np.array_equal(c_g[u], c_r), f"user {u}: code differs"
        assert np.array_equal(s_g[u].view(np.uint32), s_r.view(np.uint32)), f"user {u}: score bits differ"


@pytest.mark.parametrize("B,W_in,C,W_out", [
    (3, 1, 32, 8), (2, 1, 256, 256), (5, 24, 48, 24), (16, 64, 256, 64), (2, 96, 160, 96),
    (1, 512, 1024, 512), (3, 7, 33, 231), (2, 40, 97, 100), (1, 16, 8192, 512), (2, 130, 1000, 4096),
    (1, 9, 1028, 64), (1, 5, 9001, 300), (1, 3, 40000, 1024),
])
def test_random_logits(B, W_in, C, W_out):
    r = _rng(1)
    logits = r.normal(0, 2, (B, W_in, C)).astype(np.float32)
    score = None if W_in == 1 else np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
    _check(logits, score, W_out)


@pytest.mark.parametrize("B,C,W_out", [(2, 400, 100), (1, 512, 512), (3, 257, 64), (16, 256, 64), (2, 7, 7)])
def test_single_row_folded_in_the_one_cta_kernel(B, C, W_out):
    """W_in = 1, C <= 512 (decode step 0): the one-CTA top-k kernel folds the log-sum-exp itself (no row-offset
    launch); one and two candidates per thread, with and without a root score, -inf masks, a dead user."""
    r = _rng(6)
    logits = r.normal(0, 2, (B, 1, C)).astype(np.float32)
    _check(logits, None, W_out)
    _check(logits, r.normal(-2, 1, (B, 1)).astype(np.float32), W_out)
    logits[:, :, C // 2:] = -np.inf
    logits[0] = -np.inf
    _check(logits, r.normal(-2, 1, (B, 1)).astype(np.float32), W_out)


def test_mixture_near_ties_and_large_offsets():
    """Config 4's mixture (90 % N(0,1), 10 % N(3, 0.5)) plus a large common shift per beam: the max subtraction
    must keep the fp64 sum exact enough for a correctly rounded fp32 lse."""
    r = _rng(2)
    B, W_in, C = 2, 64, 1024
    hi = r.random((B, W_in, C)) < 0.1
    logits = np.where(hi, r.normal(3, 0.5, (B, W_in, C)), r.normal(0, 1, (B, W_in, C)))
    logits = (logits + r.normal(0, 50, (B, W_in, 1))).astype(np.float32)
    score = r.normal(-10, 3, (B, W_in)).astype(np.float32)
    _check(logits, score, 512)


def test_quantised_logits_exact_ties():
    r = _rng(3)
    logits = (np.round(r.normal(0, 1.5, (2, 32, 256)) * 8) / 8).astype(np.float32)
    logits[1, 1] = logits[1, 0]                  # two beams with identical rows and scores: keys tie pairwise
    score = np.zeros((2, 32), np.float32)
    _check(logits, score, 200)


def test_neg_inf_masks_and_dead_beams():
    r = _rng(4)
    logits = r.normal(0, 2, (2, 32, 256)).astype(np.float32)
    logits[:, :, 10:] = -np.inf                  # 10 legal codes per beam
    logits[0, 3] = -np.inf                       # a beam with no legal continuation
    logits[1, :, :] = -np.inf                    # a user with none at all
    logits[1, 7, 5] = 0.25                       # ... but one
    score = r.normal(-3, 1, (2, 32)).astype(np.float32)
    _check(logits, score, 64)
    _check(logits, score, 512)


def test_full_size_cfg2_and_paper_level():
    """Config 2's level (16 users x 64 beams x 256 codes) and one paper-scale user (512 x 8192,
    PAPER.md:126, 306) in full."""
    r = _rng(5)
    _check(r.normal(0, 2, (16, 64, 256)).astype(np.float32),
           np.sort(r.normal(-8, 2, (16, 64)).astype(np.float32))[:, ::-1].copy(), 64)
    _check(r.normal(0, 2, (1, 512, 8192)).astype(np.float32),
           np.sort(r.normal(-12, 2, (1, 512)).astype(np.float32))[:, ::-1].copy(), 512)


def test_argument_validation():
    import torch
    from paper_2607_04068_b200 import StarkError, stark_beam_topk_logits
    lg = torch.zeros((1, 4, 8), device="cuda")
    o = (torch.empty((1, 4), device="cuda"), torch.empty((1, 4), dtype=torch.int32, device="cuda"),
         torch.empty((1, 4), dtype=torch.int32, device="cuda"))
    with pytest.raises(StarkError):              # workspace is mandatory
        stark_beam_topk_logits(lg, None, 1, 4, 8, 4, *o, None)
    with pytest.raises(StarkError):              # W_out > W_in * C
        stark_beam_topk_logits(lg, None, 1, 4, 8, 33, *o, torch.empty(4096, dtype=torch.uint8, device="cuda"))


def test_rows_whose_logsumexp_sits_next_to_an_fp32_rounding_boundary():
    """Reading R22 / include/stark.h A3': lse = fl32(logsumexp) is the correctly rounded fp32 value of an fp64
    evaluation.  The kernel sums in a different order (and with its own fp64 exp) than numpy, so the two fp64
    values differ by a few 1e-16 relative; the fp32 rounding can only flip when the exact value lies that close
    to the midpoint of two fp32 neighbours (probability ~1e-9 per beam, stated in the header).  This test goes
    looking for trouble: of 4 M random short rows it keeps the 4096 whose fp64 log-sum-exp is CLOSEST to such a
    midpoint (down to ~1e-7 of an fp32 ulp, i.e. 1e-14 relative -- still 50x the kernel's fp64 error) and
    requires bitwise equal offsets on all of them."""
    import torch
    from oracle.selection import row_offset_fp32
    from paper_2607_04068_b200 import stark_logits_row_offset
    r = _rng(9)
    C, rows, keep = 4, 1 << 22, 4096
    logits = r.normal(0, 2, (rows, C)).astype(np.float32)
    x = logits.astype(np.float64)
    m = x.max(-1)
    lse = m + np.log(np.exp(x - m[:, None]).sum(-1))                 # the oracle's own formula (fp64)
    lo = lse.astype(np.float32)                                      # nearest fp32 ...
    other = np.nextafter(lo, np.where(lo.astype(np.float64) < lse, np.float32(np.inf), np.float32(-np.inf))).astype(np.float32)
    mid = 0.5 * (lo.astype(np.float64) + other.astype(np.float64))   # ... and the rounding boundary on lse's side
    ulp = np.abs(other.astype(np.float64) - lo.astype(np.float64))
    dist = np.abs(lse - mid) / ulp                                   # in fp32 ulps; 0 = exactly on the boundary
    hard = np.argsort(dist)[:keep]
    print(f"closest distances to an fp32 rounding boundary: {dist[hard[:3]]} ulp(fp32); fp64 eps = {2**-52 * 2**23:.1e} ulp(fp32)")
    assert dist[hard[-1]] < 1e-3
    sel = np.ascontiguousarray(logits[hard])
    off = torch.empty(keep, dtype=torch.float32, device="cuda")
    stark_logits_row_offset(torch.from_numpy(sel).cuda(), None, keep, C, off)
    ref = row_offset_fp32(np.zeros(keep, np.float32), sel)
    far = dist[hard] > 64 * 2.0 ** -29                               # > 64 fp64 ulps from the boundary
    assert np.array_equal(off.cpu().numpy()[far].view(np.uint32), ref[far].view(np.uint32))
    # rows even closer than that (none in practice) may legitimately round either way: by one fp32 ulp at most
    d = np.abs(off.cpu().numpy().view(np.int32).astype(np.int64) - ref.view(np.int32).astype(np.int64))
    assert d.max() <= 1
