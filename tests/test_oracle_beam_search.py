"""Pins for the oracle's beam search, tree formulation and replay (CPU only).

The three checks BASELINE.json's north star prescribes:
  1. tree attention (Eq. 14 mask over the sequence-expanded layout) must equal
     per-beam full-sequence attention;
  2. beam width 1 must equal greedy decoding;
  3. on tiny codebooks, beam width >= all paths must recover brute-force
     enumeration of every SID path ranked by summed log-prob.
Plus a hand-written Eq.-14 mask fixture, closed forms and invariants.
"""
import math
import os

import numpy as np
import pytest

import workloads as wl
from oracle.attention import beam_attention
from oracle.beam_search import conventional_beam_search
from oracle.brute_force import enumerate_all_paths
from oracle.replay import replay_beam_attention, replay_step_attention
from oracle.selection import log_softmax_fp32
from oracle.token_models import DrawTokenModel, TableTokenModel
from oracle.tree import ancestor_chains, sequence_expanded_attention, tree_mask

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _draw_user(cfg, u, seed=0, final_step=True):
    """One user's seeded inputs for a DrawTokenModel + its prefix."""
    lens = wl.prefix_lengths(cfg, seed)
    K, V = wl.prefix_kv_user(cfg, u, int(lens[u]), seed)
    nq = [1] + wl.beam_widths(cfg)
    q, k, v, lg = [], [], [], []
    for t in range(cfg.d + 1):
        qq, kk, vv = wl.step_qkv(cfg, t, nq[t], seed, users=[u])
        q.append(qq[0]), k.append(kk[0]), v.append(vv[0])
        if t < cfg.d:
            lg.append(wl.step_logits(cfg, t, nq[t], seed, users=[u])[0])
    return K, V, DrawTokenModel(q, k, v, lg)


# ---------------------------------------------------------------- fixture ----
def _read_fixture():
    parents, masks, chains, L = {}, {}, {}, None
    cur = None
    for line in open(os.path.join(GOLDEN, "tree_mask_small.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("L "):
            L = int(line.split()[1])
        elif line.startswith("parents"):
            lvl = int(line.split()[1].rstrip(":"))
            parents[lvl] = np.array([int(x) for x in line.split(":")[1].split()])
        elif line.startswith("mask") or line.startswith("chains"):
            kind, lvl = line.split()[0], int(line.split()[1].rstrip(":"))
            cur = (masks if kind == "mask" else chains).setdefault(lvl, [])
        else:
            cur.append([int(x) for x in line.split()])
    return L, parents, masks, chains


def test_tree_mask_matches_hand_written_fixture():
    L, parents, masks, chains = _read_fixture()
    plist = [parents[1], parents[2], parents[3]]
    for t in (1, 2, 3):
        got = tree_mask(plist, t, L).astype(int)
        assert np.array_equal(got, np.array(masks[t])), f"level {t}"
    assert np.array_equal(ancestor_chains(plist, 3), np.array(chains[3]))


# ------------------------------------------------ check 1: tree == per beam ----
@pytest.mark.parametrize("name", ["cfg5_small", "f32_gqa", "cfg2_small"])
def test_tree_attention_equals_per_beam_full_sequence_attention(name):
    cfg = wl.get_config(name)
    scale = 1.0 / math.sqrt(cfg.D)
    u = cfg.B - 1
    K, V, model = _draw_user(cfg, u)
    tr = conventional_beam_search(K, V, model, wl.beam_widths(cfg), cfg.C, scale, final_step=True)
    k_levels = [tr.k_new[t] for t in range(1, cfg.d + 1)]
    v_levels = [tr.v_new[t] for t in range(1, cfg.d + 1)]
    for t in range(cfg.d + 1):
        # the paper's formulation: ONE expanded sequence + dense Eq.-14 mask
        tree = sequence_expanded_attention(K, V, k_levels, v_levels, tr.parents, tr.q[t], t, scale)
        np.testing.assert_allclose(tree, tr.attn_out[t], rtol=1e-11, atol=1e-12)
        # teacher-forced conventional replay (all beams, and one sampled beam)
        rep = replay_step_attention(K, V, k_levels, v_levels, tr.parents, tr.q[t], t, scale)
        np.testing.assert_allclose(rep, tr.attn_out[t], rtol=1e-11, atol=1e-12)
        i = tr.q[t].shape[0] // 2
        one = replay_beam_attention(K, V, k_levels, v_levels, tr.parents, tr.q[t][i], i, t, scale)
        np.testing.assert_allclose(one, tr.attn_out[t][i], rtol=1e-11, atol=1e-12)


# --------------------------------------------------- check 2: W = 1 is greedy ----
def test_beam_width_one_is_greedy_decoding():
    cfg = wl.get_config("cfg1")
    scale = 1.0 / math.sqrt(cfg.D)
    K, V = wl.prefix_kv_user(cfg, 0, cfg.prefix_min)
    model = TableTokenModel(wl.config1_tables(cfg))
    tr = conventional_beam_search(K, V, model, [1] * cfg.d, cfg.C, scale)
    # independent greedy chain: one growing sequence, argmax of the logits each level
    Kc, Vc = K.astype(np.float64), V.astype(np.float64)
    path, total = (), np.float32(0.0)
    for t in range(cfg.d):
        q, k, v = model.qkv(t, 0, path)
        if t >= 1:
            Kc = np.concatenate([Kc, k[None]])
            Vc = np.concatenate([Vc, v[None]])
        o = beam_attention(q, Kc, Vc, scale)
        lg = model.logits(t, 0, path, o)
        c = int(np.argmax(lg))
        total = np.float32(total + log_softmax_fp32(lg)[c])
        path = path + (c,)
    assert tuple(tr.paths[0]) == path
    assert tr.scores[-1][0] == total
    assert all(int(p[0]) == 0 for p in tr.parents)


# ------------------------------------- check 3: full width == brute force ----
@pytest.mark.parametrize("C,d,Hq,Hkv", [(3, 3, 2, 1), (4, 2, 4, 4)])
def test_full_width_beam_recovers_brute_force_enumeration(C, d, Hq, Hkv):
    from dataclasses import replace
    cfg = replace(wl.get_config("cfg1"), name="tiny", config_id=99, Hq=Hq, Hkv=Hkv, D=8,
                  prefix_min=6, prefix_max=6, W=(C ** d,) * d, d=d, C=C, kv_std=1.0, q_std=1.0)
    scale = 1.0 / math.sqrt(cfg.D)
    K, V = wl.prefix_kv_user(cfg, 0, 6)
    model = TableTokenModel(wl.config1_tables(cfg))
    tr = conventional_beam_search(K, V, model, wl.beam_widths(cfg), C, scale)
    paths, scores, total = enumerate_all_paths(K, V, model, d, C, scale)
    assert tr.paths.shape == (C ** d, d)
    assert len({tuple(p) for p in tr.paths}) == C ** d                 # every path, once
    assert np.array_equal(tr.paths, paths)                             # same ranking
    assert np.array_equal(tr.scores[-1], scores)                       # same fp32 scores
    assert abs(total - 1.0) < 1e-5                                     # sum_paths P(path) = 1 (fp32 log-probs)
    # narrower beam: the kept set is the top-W of the exhaustive ranking at level 1
    tr2 = conventional_beam_search(K, V, model, [2] * d, C, scale)
    lvl1 = log_softmax_fp32(model.logits(0, 0, (), tr.attn_out[0][0]))
    assert set(tr2.codes[0].tolist()) == set(np.argsort(-lvl1, kind="stable")[:2].tolist())


def test_no_pruning_total_probability_is_one_fp64():
    # closed form: without pruning, sum over all paths of exp(score) = 1.  Use fp64
    # log-probs here (independent of the fp32 selection key) -> 1e-12.
    cfg = wl.get_config("cfg1")
    C, d = 3, 3
    from dataclasses import replace
    cfg = replace(cfg, name="tiny2", config_id=98, Hq=2, Hkv=2, D=4, prefix_min=5, prefix_max=5,
                  W=(27,) * 3, C=C, d=d)
    scale = 0.5
    K, V = wl.prefix_kv_user(cfg, 0, 5)
    model = TableTokenModel(wl.config1_tables(cfg))
    import itertools
    tot = 0.0
    for path in itertools.product(range(C), repeat=d):
        Kc, Vc, lp = K.astype(np.float64), V.astype(np.float64), 0.0
        for t in range(d):
            q, k, v = model.qkv(t, 0, path[:t])
            if t:
                Kc, Vc = np.concatenate([Kc, k[None]]), np.concatenate([Vc, v[None]])
            lg = model.logits(t, 0, path[:t], beam_attention(q, Kc, Vc, scale))
            lp += lg[path[t]] - (np.max(lg) + math.log(np.sum(np.exp(lg - np.max(lg)))))
        tot += math.exp(lp)
    assert abs(tot - 1.0) < 1e-12


# ----------------------------------------------------------- structure ----
def test_per_level_widths_and_trace_structure():
    from dataclasses import replace
    cfg = replace(wl.get_config("paper_small"), B=1)
    scale = 1.0 / math.sqrt(cfg.D)
    K, V, model = _draw_user(cfg, 0)
    widths = wl.beam_widths(cfg)
    assert widths == [16, 16, 40]                                      # per-level widths
    tr = conventional_beam_search(K, V, model, widths, cfg.C, scale)
    assert [len(p) for p in tr.parents] == widths
    assert tr.paths.shape == (40, 3)
    for t in range(cfg.d):
        assert np.all(np.diff(tr.scores[t]) <= 0)
        if t:
            assert np.all(tr.scores[t] <= tr.scores[t - 1][tr.parents[t]])
        assert tr.margins[t] >= 0
    # a path is its parent's path plus its own code
    chain = ancestor_chains(tr.parents, cfg.d)
    for r in range(40):
        assert [int(tr.codes[l][chain[r, l]]) for l in range(cfg.d)] == tr.paths[r].tolist()


def test_config1_seed0_selection_margins_recorded():
    """the end-to-end identity argument needs the key gap between
    rank W and rank W+1 to exceed the fp32-vs-fp64 attention noise (~1e-6)."""
    cfg = wl.get_config("cfg1")
    K, V = wl.prefix_kv_user(cfg, 0, cfg.prefix_min)
    tr = conventional_beam_search(K, V, TableTokenModel(wl.config1_tables(cfg)),
                                  wl.beam_widths(cfg), cfg.C, 1.0 / math.sqrt(cfg.D))
    assert tr.paths.shape == (8, 3)
    assert min(tr.margins) > 1e-4, tr.margins
