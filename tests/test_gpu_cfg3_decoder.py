"""Config 3 (BASELINE.json configs[2]): the library inside a 12-layer decoder (GEMMs in torch/cuBLAS).
Per-call parity on captured inputs ("Config 3: sampled (layer, user, step) triples"):
  * step 0: the library's attention of the last prefix token equals torch SDPA's causal result for that
    position in every layer (an independent library routine as reference);
  * sampled (layer, user, step, beam): attention row vs the oracle's conventional per-beam full-sequence
    attention over that layer's captured prefix + suffix K/V and the selected parents;
  * ALL beams of two whole (layer, user) pairs at every step vs the oracle's sequence-expanded Eq.-14 attention;
  * every level's selection bit-exact vs oracle.select_beams on the captured fp32 log-probs and scores."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu
TOL = 1.5e-2


def _check(sh, n_samples):
    from paper_2607_04068_b200.decoder_harness import Decoder
    from oracle.replay import replay_beam_attention
    from oracle.tree import sequence_expanded_attention
    from oracle.selection import select_beams
    torch.manual_seed(0)
    model = Decoder(sh, seed=0)
    g = torch.Generator(device="cpu").manual_seed(3)
    tokens = torch.randint(0, sh.vocab, (sh.B, sh.prefix), generator=g).cuda()
    cap = model.decode(tokens)
    scale = 1.0 / np.sqrt(sh.D)
    # (a) step 0 vs torch SDPA
    for li in range(sh.n_layers):
        ref = cap["last_attn"][li].float()
        got = cap["out"][0][li][:, 0].float()
        assert (got - ref).abs().max() <= TOL * ref.abs().max(), f"layer {li}: step-0 attention vs SDPA"
    # (c) selections, all users and levels, bit-exact
    sel = [[x.cpu().numpy() for x in s] for s in cap["sel"]]
    for t in range(sh.d):
        logp = cap["logp"][t].cpu().numpy()
        for u in range(sh.B):
            score = np.zeros(1, np.float32) if t == 0 else sel[t - 1][0][u]
            s_r, p_r, c_r = select_beams(score, logp[u], sel[t][1].shape[1])
            assert np.array_equal(sel[t][1][u], p_r) and np.array_equal(sel[t][2][u], c_r), f"level {t} user {u}"
            assert np.array_equal(sel[t][0][u].view(np.uint32), s_r.view(np.uint32))
    # (b) sampled triples vs the oracle
    rng = np.random.default_rng(11)
    worst = 0.0
    for _ in range(n_samples):
        li, u, t = int(rng.integers(sh.n_layers)), int(rng.integers(sh.B)), int(rng.integers(1, sh.d))
        i = int(rng.integers(cap["q"][t][li].shape[1]))
        Kp, Vp = cap["prefix_kv"][li]
        Kp = Kp[u * sh.prefix:(u + 1) * sh.prefix].float().cpu().numpy()
        Vp = Vp[u * sh.prefix:(u + 1) * sh.prefix].float().cpu().numpy()
        k_lv = [cap["k"][l][li][u].float().cpu().numpy() for l in range(1, t + 1)]
        v_lv = [cap["v"][l][li][u].float().cpu().numpy() for l in range(1, t + 1)]
        parents = [sel[l][1][u] for l in range(t)]      # parents[l-1] = parent slots of the level-l beams (l >= 1)
        ref = replay_beam_attention(Kp, Vp, k_lv, v_lv, parents, cap["q"][t][li][u, i].float().cpu().numpy(), i, t, scale)
        got = cap["out"][t][li][u, i].float().cpu().numpy()
        worst = max(worst, float(np.abs(got - ref).max() / (np.abs(ref).max() + 1e-30)))
    assert worst <= TOL, f"sampled attention rows vs oracle: {worst:.3e}"
    # (d) ALL beams of whole (layer, user) pairs, every step: first layer / first user and last layer / last user
    for li, u in ((0, 0), (sh.n_layers - 1, sh.B - 1)):
        Kp, Vp = cap["prefix_kv"][li]
        Kp = Kp[u * sh.prefix:(u + 1) * sh.prefix].float().cpu().numpy()
        Vp = Vp[u * sh.prefix:(u + 1) * sh.prefix].float().cpu().numpy()
        for t in range(sh.d):
            k_lv = [cap["k"][l][li][u].float().cpu().numpy() for l in range(1, t + 1)]
            v_lv = [cap["v"][l][li][u].float().cpu().numpy() for l in range(1, t + 1)]
            parents = [sel[l][1][u] for l in range(t)]
            ref = sequence_expanded_attention(Kp, Vp, k_lv, v_lv, parents, cap["q"][t][li][u].float().cpu().numpy(), t, scale)
            got = cap["out"][t][li][u].float().cpu().numpy()
            err = float(np.abs(got - ref).max() / (np.abs(ref).max() + 1e-30))
            assert err <= TOL, f"layer {li} user {u} step {t}: all beams vs oracle {err:.3e}"


def test_small_decoder():
    from paper_2607_04068_b200.decoder_harness import DecoderShape
    _check(DecoderShape(n_layers=3, d_model=256, Hq=8, Hkv=2, D=64, ffn=512, vocab=1000, prefix=300, B=3, W=24, d=3, C=40),
           n_samples=12)


def test_cfg3_full_size():
    from paper_2607_04068_b200.decoder_harness import DecoderShape
    _check(DecoderShape(), n_samples=10)
