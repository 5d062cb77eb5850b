"""Pins of oracle/encdec.py (the paper's encoder-decoder form, the ranking-feature step, target attention;
DESIGN.md readings R23-R25) against things other than itself: torch's scaled_dot_product_attention in fp64 with
an explicit mask taken from a HAND-WRITTEN fixture (tests/golden/tree_mask_tat.txt), closed forms, the
sequence-expanded Eq.-14 formulation of oracle/tree.py, and path-prefix matching on a conventional beam search."""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import workloads as wl
from oracle.attention import beam_attention
from oracle.beam_search import conventional_beam_search
from oracle.encdec import (N_FIXED, cross_attention, cross_plus_self_attention, path_hidden_states,
                           self_tree_attention, target_attention)
from oracle.token_models import DrawTokenModel
from oracle.tree import ancestor_chains, sequence_expanded_attention, tree_mask

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _read_fixture(name):
    parents, masks, chains, L = {}, {}, {}, None
    cur = None
    for line in open(os.path.join(GOLDEN, name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("L "):
            L = int(line.split()[1])
        elif line.startswith("parents"):
            parents[int(line.split()[1].rstrip(":"))] = np.array([int(x) for x in line.split(":")[1].split()])
        elif line.startswith("mask") or line.startswith("chains"):
            kind, lvl = line.split()[0], int(line.split()[1].rstrip(":"))
            cur = (masks if kind == "mask" else chains).setdefault(lvl, [])
        else:
            cur.append([int(x) for x in line.split()])
    return L, parents, masks, chains


def _sdpa(q, K, V, mask, scale, G):
    """torch SDPA fp64: q [n,Hq,D], K,V [S,Hkv,D], mask [n,S] bool or None -> [n,Hq,D]."""
    qt = torch.from_numpy(q).permute(1, 0, 2)[None]                           # [1,Hq,n,D]
    Kt = torch.from_numpy(np.repeat(K, G, axis=1)).permute(1, 0, 2)[None]     # head h reads KV head h // G
    Vt = torch.from_numpy(np.repeat(V, G, axis=1)).permute(1, 0, 2)[None]
    m = None if mask is None else torch.from_numpy(mask)[None, None]
    return F.scaled_dot_product_attention(qt, Kt, Vt, attn_mask=m, scale=scale)[0].permute(1, 0, 2).numpy()


def test_fixture_is_the_eq14_mask_with_four_fixed_positions():
    L, parents, masks, chains = _read_fixture("tree_mask_tat.txt")
    assert L == N_FIXED
    plist = [parents[1], parents[2], parents[3]]
    for t in (1, 2, 3):
        assert np.array_equal(tree_mask(plist, t, L).astype(int), np.array(masks[t]))
    assert np.array_equal(ancestor_chains(plist, 3), np.array(chains[3]))


def test_self_attention_equals_sdpa_under_the_hand_written_mask():
    """Every level of the fixture's tree: conventional per-beam sequences == ONE masked attention over the
    expanded decoder sequence [click atc pay bos | level 1 | level 2 | level 3] with the fixture's mask."""
    L, parents, masks, _ = _read_fixture("tree_mask_tat.txt")
    plist = [parents[1], parents[2], parents[3]]
    r = np.random.default_rng(5)
    Hq, Hkv, D = 4, 2, 8
    scale = 1.0 / math.sqrt(D)
    Kf, Vf = r.normal(size=(N_FIXED, Hkv, D)), r.normal(size=(N_FIXED, Hkv, D))
    k_lv = [r.normal(size=(len(p), Hkv, D)) for p in plist]
    v_lv = [r.normal(size=(len(p), Hkv, D)) for p in plist]
    for t in (1, 2, 3):
        q = r.normal(size=(len(plist[t - 1]), Hq, D))
        got = self_tree_attention(q, Kf, Vf, k_lv, v_lv, plist, t, scale)
        Kall = np.concatenate([Kf] + k_lv[:t]); Vall = np.concatenate([Vf] + v_lv[:t])
        ref = _sdpa(q, Kall, Vall, np.array(masks[t], dtype=bool), scale, Hq // Hkv)
        np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-12)
        np.testing.assert_allclose(got, sequence_expanded_attention(Kf, Vf, k_lv, v_lv, plist, q, t, scale),
                                   rtol=1e-11, atol=1e-12)
    # level 0 (<bos> itself): the four fixed positions only
    q0 = r.normal(size=(1, Hq, D))
    np.testing.assert_allclose(self_tree_attention(q0, Kf, Vf, [], [], [], 0, scale),
                               _sdpa(q0, Kf, Vf, None, scale, Hq // Hkv), rtol=1e-11, atol=1e-12)


def test_cross_and_target_attention_equal_sdpa_and_closed_forms():
    r = np.random.default_rng(6)
    Hq, Hkv, D, Lm, n = 8, 2, 16, 37, 5
    scale = 1.0 / math.sqrt(D)
    K, V = r.normal(size=(Lm, Hkv, D)), r.normal(size=(Lm, Hkv, D))
    q = r.normal(size=(n, Hq, D))
    ref = _sdpa(q, K, V, None, scale, Hq // Hkv)
    np.testing.assert_allclose(cross_attention(q, K, V, scale), ref, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(target_attention(q, K, V, scale), ref, rtol=1e-11, atol=1e-12)
    # closed forms: K = 0 => the arithmetic mean of the memory's V rows; one dominant key => that V row
    out = cross_attention(q, np.zeros_like(K), V, scale)
    for h in range(Hq):
        np.testing.assert_allclose(out[:, h], np.broadcast_to(V[:, h // (Hq // Hkv)].mean(0), (n, D)), atol=1e-12)
    K2 = np.zeros_like(K); K2[11] = 50.0 * q[2, 3] / np.dot(q[2, 3], q[2, 3]) / scale    # score 50 at row 11 for (2, 3)
    np.testing.assert_allclose(cross_attention(q, K2, V, scale)[2, 3], V[11, 3 // (Hq // Hkv)], atol=1e-9)


def test_cross_and_self_are_two_softmaxes_not_one():
    """Reading R23: cross-attention normalises over M alone, self-attention over the decoder sequence alone.
    With all V = 1 both outputs are exactly 1 (each softmax sums to 1 on its own); a single softmax over
    [M ++ decoder sequence] would give a DIFFERENT result for generic V."""
    r = np.random.default_rng(7)
    Hq, Hkv, D, Lm, W = 4, 2, 8, 20, 6
    scale = 1.0 / math.sqrt(D)
    K_M, V_M = r.normal(size=(Lm, Hkv, D)), r.normal(size=(Lm, Hkv, D))
    Kf, Vf = r.normal(size=(N_FIXED, Hkv, D)), r.normal(size=(N_FIXED, Hkv, D))
    k1, v1 = r.normal(size=(W, Hkv, D)), r.normal(size=(W, Hkv, D))
    parents = [np.zeros(W, dtype=np.int64)]
    qc, qs = r.normal(size=(W, Hq, D)), r.normal(size=(W, Hq, D))
    cross, self_ = cross_plus_self_attention(qc, qs, K_M, np.ones_like(V_M), Kf, np.ones_like(Vf), [k1], [np.ones_like(v1)],
                                             parents, 1, scale)
    np.testing.assert_allclose(cross, 1.0, atol=1e-12)
    np.testing.assert_allclose(self_, 1.0, atol=1e-12)
    cross, self_ = cross_plus_self_attention(qc, qs, K_M, V_M, Kf, Vf, [k1], [v1], parents, 1, scale)
    for i in range(W):       # each part on its own key set, by the plain single-sequence definition
        np.testing.assert_allclose(cross[i], beam_attention(qc[i], K_M, V_M, scale), rtol=1e-12)
        np.testing.assert_allclose(self_[i], beam_attention(qs[i], np.concatenate([Kf, k1[i:i + 1]]),
                                                            np.concatenate([Vf, v1[i:i + 1]]), scale), rtol=1e-12)
    joint = beam_attention(qs[0], np.concatenate([K_M, Kf, k1[:1]]), np.concatenate([V_M, Vf, v1[:1]]), scale)
    assert np.abs(joint - self_[0]).max() > 1e-3


def test_path_hidden_states_by_path_prefix_matching():
    """the features of a final beam are the decoder outputs at <bos>, s_1, ..., s_d along ITS path.
    Independent pin: SID paths are unique, so the depth-l ancestor of final beam r is the one level-l beam
    whose path equals the first l codes of r's path (the final paths are the beam search's own hypothesis
    paths; the level-l paths are rebuilt from (parent, code)) -- found by matching, not by walking r's chain."""
    cfg = wl.get_config("cfg2_small")
    scale = 1.0 / math.sqrt(cfg.D)
    lens = wl.prefix_lengths(cfg, 0)
    u = 1
    K, V = wl.prefix_kv_user(cfg, u, int(lens[u]), 0)
    nq = [1] + wl.beam_widths(cfg)
    q, k, v, lg = [], [], [], []
    for t in range(cfg.d + 1):
        qq, kk, vv = wl.step_qkv(cfg, t, nq[t], 0, users=[u])
        q.append(qq[0]), k.append(kk[0]), v.append(vv[0])
        if t < cfg.d:
            lg.append(wl.step_logits(cfg, t, nq[t], 0, users=[u])[0])
    tr = conventional_beam_search(K, V, DrawTokenModel(q, k, v, lg), wl.beam_widths(cfg), cfg.C, scale, final_step=True)
    feats = path_hidden_states(tr.attn_out, tr.parents)                    # [W_d, d+1, Hq, D]
    assert feats.shape == (tr.paths.shape[0], cfg.d + 1, cfg.Hq, cfg.D)
    # paths of the level-l beams, rebuilt from (parents, codes) level by level
    level_paths = [[()]]
    for l in range(1, cfg.d + 1):
        level_paths.append([level_paths[l - 1][0 if l == 1 else int(tr.parents[l - 1][s])] + (int(tr.codes[l - 1][s]),)
                            for s in range(len(tr.parents[l - 1]))])
    for r_, path in enumerate(tr.paths.tolist()):
        np.testing.assert_array_equal(feats[r_, 0], tr.attn_out[0][0])
        for l in range(1, cfg.d + 1):
            slot = level_paths[l].index(tuple(path[:l]))                   # unique
            np.testing.assert_array_equal(feats[r_, l], tr.attn_out[l][slot])
