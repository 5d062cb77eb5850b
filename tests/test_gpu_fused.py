"""GPU parity of stark_decode_attn (A1 + A2 fused) on shapes chosen to hit every structural branch of the
kernel: cluster sizes 1/2/4/8 over the prefix splits (DSMEM exchange), splits that are EMPTY for short users
of a ragged batch, parity mode vs pair mode, a second Q tile with few live rows, head_dim 64, GQA groups of 1,
2, 4, 8, 16, 32, 64 and 128, chain lengths 0..d.  Reference: oracle.replay (conventional per-beam full-sequence attention,
fp64) -- every row of every user via the sequence-expanded Eq.-14 form, sampled beams via the per-beam
replay -- plus the two-call GPU path (A1 then A2) on every row.  Tolerance: DESIGN.md R20."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1.5e-2


def _bf16(x):
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def _case(B, Hq, Hkv, D, lens, W, d, seed):
    import torch
    from oracle.replay import replay_beam_attention
    from oracle.tree import sequence_expanded_attention
    from paper_2607_04068_b200.decode import StarkLayer
    rng = np.random.default_rng([0, 91, seed])
    lens = np.asarray(lens)
    cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    tot = int(cu[-1])
    K = _bf16(rng.normal(0, 1, (tot, Hkv, D))); V = _bf16(rng.normal(0, 1, (tot, Hkv, D)))
    dev = torch.device("cuda")
    bf = lambda a: torch.from_numpy(a).to(dev).to(torch.bfloat16).contiguous()
    layer = StarkLayer(B, Hq, Hkv, D, d, W, torch.bfloat16, bf(K), bf(V), torch.from_numpy(cu).to(dev), int(lens.max()))
    # the same steps through stark_decode_step (append inside the attention launch)
    layer_s = StarkLayer(B, Hq, Hkv, D, d, W, torch.bfloat16, layer.k_prefix, layer.v_prefix, layer.cu, int(lens.max()))
    scale = 1.0 / np.sqrt(D)
    k_lv, v_lv, parents = [], [], []
    for t in range(d + 1):
        n_q = 1 if t == 0 else W
        q = _bf16(rng.normal(0, 1, (B, n_q, Hq, D)))
        if t >= 1:
            kn = _bf16(rng.normal(0, 1, (B, W, Hkv, D))); vn = _bf16(rng.normal(0, 1, (B, W, Hkv, D)))
            par = rng.integers(0, 1 if t == 1 else W, (B, W)).astype(np.int32)
            k_lv.append(kn); v_lv.append(vn); parents.append(par)
            layer.append(t, bf(kn), bf(vn), torch.from_numpy(par).to(dev))
        qd = bf(q)
        fused_t = layer.attend(t, qd, fused=True)
        if t >= 1:
            step_t = layer_s.step(t, qd, bf(kn), bf(vn), torch.from_numpy(par).to(dev))
            assert torch.equal(layer_s.k_suffix[t - 1], layer.k_suffix[t - 1]), f"step {t}: inline append K"
            assert torch.equal(layer_s.v_suffix[t - 1], layer.v_suffix[t - 1]), f"step {t}: inline append V"
            assert torch.equal(layer_s.anc[t & 1, :, :, :t], layer.anc[t & 1, :, :, :t]), f"step {t}: inline index"
        else:
            step_t = layer_s.step(t, qd, None, None, None)
        assert torch.equal(step_t, fused_t), f"step {t}: stark_decode_step differs from append + stark_decode_attn"
        fused = fused_t.float().cpu().numpy().astype(np.float64)
        assert np.isfinite(fused).all()
        if Hq // Hkv <= 32:      # (stark_tree_attn_step serves GQA groups up to 32; the fused kernel up to 128)
            two = layer.attend(t, qd, fused=False).float().cpu().numpy().astype(np.float64)
            # every row: fused vs two-call (both bf16 outputs of the same fp32-accumulated math)
            ref_max = np.abs(two).max() + 1e-30
            assert np.abs(fused - two).max() <= TOL * ref_max, f"step {t}: fused vs two-call {np.abs(fused - two).max() / ref_max:.3e}"
        # EVERY row of EVERY user: fused vs the fp64 oracle (sequence-expanded masked attention, Eq. 14;
        # pinned equal to the conventional per-beam form in tests/test_oracle_beam_search.py)
        worst = 0.0
        for u in range(B):
            ref = sequence_expanded_attention(K[cu[u]:cu[u + 1]], V[cu[u]:cu[u + 1]], [x[u] for x in k_lv[:t]],
                                              [x[u] for x in v_lv[:t]], [p[u] for p in parents[:t]], q[u], t, scale)
            worst = max(worst, float(np.abs(fused[u] - ref).max() / (np.abs(ref).max() + 1e-30)))
        assert worst <= TOL, f"step {t}: fused vs oracle {worst:.3e}"
        # and the conventional per-beam replay (replicated caches) on sampled beams
        for _ in range(3):
            u, i = int(rng.integers(B)), int(rng.integers(n_q))
            ref = replay_beam_attention(K[cu[u]:cu[u + 1]], V[cu[u]:cu[u + 1]], [x[u] for x in k_lv[:t]],
                                        [x[u] for x in v_lv[:t]], [p[u] for p in parents[:t]], q[u, i], i, t, scale)
            assert float(np.abs(fused[u, i] - ref).max() / (np.abs(ref).max() + 1e-30)) <= TOL, f"step {t}: beam ({u},{i})"


@pytest.mark.parametrize("name,args", [
    # B, Hq, Hkv, D, prefix lengths, W, d
    ("cluster8_parity", (1, 4, 1, 128, [2048], 24, 2)),          # 1 CTA x 8 splits, one Q tile
    ("cluster8_ragged_empty_splits", (2, 8, 2, 128, [100, 1900], 20, 2)),   # user 0: 7 of 8 splits empty
    ("cluster4_two_tiles", (1, 8, 2, 128, [1000], 40, 3)),        # M = 160: second Q tile with 32 live rows
    ("cluster2_d64", (3, 8, 2, 64, [700, 129, 128], 48, 2)),      # head_dim 64, L = 128 -> empty second split
    ("pair_mode_many_ctas", (10, 16, 4, 128, [300] * 10, 70, 2)), # 2 Q tiles per CTA, no splits
    ("gqa1_and_short_prefix", (2, 4, 4, 128, [5, 260], 12, 2)),   # G = 1, a 5-row prefix
    ("gqa8", (2, 16, 2, 128, [640, 384], 16, 2)),                 # G = 8: 16 beams per Q tile
    # parity mode WITHOUT splits (128 CTAs): chain V rows staged by cp.async into idle ring tiles; 3 levels deep, so
    # levels 0-1 come from shared memory and level 2 from global memory; ragged prefixes incl. 1- and 2-tile users
    ("parity_nosplit_d64_deep", (32, 16, 4, 64, [100 + 37 * (x % 14) for x in range(32)], 24, 3)),
    ("parity_nosplit_d128_deep", (32, 8, 4, 128, [60 + 53 * (x % 11) for x in range(32)], 20, 3)),
    # wide GQA groups: the 32 rows a warp finishes (one TMA store box) are 32 / G beams x G heads, or -- G > 32 -- a
    # 32-head part of one beam; pair mode without splits (the single-split tail) with G = 16 and an odd tile count
    ("gqa32", (2, 32, 1, 128, [300, 200], 9, 2)),
    ("gqa64_d64", (1, 64, 1, 64, [257], 5, 2)),
    ("gqa128", (1, 128, 1, 128, [130], 3, 2)),
    ("gqa16_pair_single_tail", (26, 32, 2, 128, [200 + 7 * x for x in range(26)], 20, 2)),
])
def test_fused_structural_cases(name, args):
    _case(*args, seed=sum(map(ord, name)))
