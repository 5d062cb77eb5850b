"""GPU parity of the paper's encoder-decoder form (readings R23-R25)
through the UNCHANGED library calls, against oracle/encdec.py:
  * cross-attention over the encoder memory M = stark_decode_attn at level 0 (and the two-call
    form stark_prefix_attn + stark_tree_attn_step(level = 0)) with n_q = W_t queries per user;
  * self-attention over [e_click, e_atc, e_pay, <bos>] + ancestor chain (Eq. 7, Eq. 14) = stark_decode_step
    with a 4-row prefix per user, the level's append inside the launch;
  * the ranking-feature step t = d: the final tokens' attention, and every final beam's
    features gathered along its path through the library's ancestor index;
  * target attention by the W_d candidates over M = the cross-attention call again.
Selection bit-exact vs oracle.select_beams; attention within 1.5e-2 of max|ref| per user (bf16)."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1.5e-2


def _run(name, users=None):
    import torch
    from oracle.encdec import cross_attention, path_hidden_states, self_tree_attention, target_attention
    from oracle.selection import log_softmax_fp32, select_beams
    from paper_2607_04068_b200.pipeline import EncDecPass
    cfg = wl.get_config(name)
    dev = torch.device("cuda")
    bf = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev).to(torch.bfloat16).contiguous()
    K_M, V_M, cu = wl.prefix_kv(cfg)
    Kf, Vf = wl.fixed_prefix_kv(cfg)
    nq, widths, d = wl.queries_per_step(cfg), wl.beam_widths(cfg), cfg.d
    qs, ks, vs, qc, lp = [], [], [], [], []
    for t in range(d + 1):                                   # step d = the ranking-feature step
        q_, k_, v_ = wl.step_qkv(cfg, t, nq[t])
        qs.append(q_), ks.append(k_), vs.append(v_), qc.append(wl.step_q_cross(cfg, t, nq[t]))
        if t < d:
            lp.append(log_softmax_fp32(wl.step_logits(cfg, t, nq[t])))
    lens = np.diff(cu)
    p = EncDecPass(cfg.B, cfg.Hq, cfg.Hkv, cfg.D, d, cfg.C, widths, torch.bfloat16, bf(K_M), bf(V_M),
                   torch.from_numpy(cu.astype(np.int32)).to(dev), int(lens.max()), bf(Kf), bf(Vf),
                   [bf(x) for x in qc[:d]], [bf(x) for x in qs[:d]], [bf(x) for x in ks[:d]], [bf(x) for x in vs[:d]],
                   [torch.from_numpy(x).to(dev) for x in lp])
    p.run()
    g = torch.cuda.CUDAGraph()                               # and once more as a graph replay (static shapes)
    with torch.cuda.graph(g):
        p.run()
    for s_ in p.sel:
        s_[1].fill_(-7)
    g.replay()
    # step d (no selection): the final tokens through both sub-layers, then target attention by the candidates
    parent_d = p.sel[d - 1][1]
    self_d = p.dec.step(d, bf(qs[d]), bf(ks[d]), bf(vs[d]), parent_d)
    cross_d = p.mem.attend(0, bf(qc[d]), fused=True)
    q_cand = wl.step_q_cross(cfg, d + 1, nq[d])
    tgt_fused = p.mem.attend(0, bf(q_cand), fused=True)
    tgt_two = p.mem.attend(0, bf(q_cand), fused=False)       # stark_prefix_attn -> stark_tree_attn_step(level 0)
    torch.cuda.synchronize()
    sel = [[x.cpu().numpy() for x in s_] for s_ in p.sel]
    scale = 1.0 / np.sqrt(cfg.D)
    f64 = lambda x: x.float().cpu().numpy().astype(np.float64)
    cross = [f64(x) for x in p.cross] + [f64(cross_d)]
    self_ = [f64(x) for x in p.self_out] + [f64(self_d)]
    anc = p.dec.anc.cpu().numpy()
    users = list(range(cfg.B)) if users is None else users
    rel = lambda got, ref: float(np.abs(got - ref).max() / (np.abs(ref).max() + 1e-30))
    for u in range(cfg.B):                                   # selection: every user, bit-exact
        for t in range(d):
            score = np.zeros(1, np.float32) if t == 0 else sel[t - 1][0][u]
            s_r, p_r, c_r = select_beams(score, lp[t][u], widths[t])
            assert np.array_equal(sel[t][1][u], p_r) and np.array_equal(sel[t][2][u], c_r), f"user {u} level {t}"
            assert np.array_equal(sel[t][0][u].view(np.uint32), s_r.view(np.uint32))
    for u in users:
        Ku, Vu = K_M[cu[u]:cu[u + 1]], V_M[cu[u]:cu[u + 1]]
        parents = [sel[l][1][u] for l in range(d)]
        ref_self = []
        for t in range(d + 1):
            ref_c = cross_attention(qc[t][u], Ku, Vu, scale)
            assert rel(cross[t][u], ref_c) <= TOL, f"user {u} step {t}: cross-attention {rel(cross[t][u], ref_c):.3e}"
            ref_s = self_tree_attention(qs[t][u], Kf[u], Vf[u], [ks[l][u] for l in range(1, t + 1)],
                                        [vs[l][u] for l in range(1, t + 1)], parents, t, scale)
            assert rel(self_[t][u], ref_s) <= TOL, f"user {u} step {t}: self-attention {rel(self_[t][u], ref_s):.3e}"
            ref_self.append(ref_s)
        # ranking features: the library's ancestor index gathers every final beam's outputs along its path
        feats_ref = path_hidden_states(ref_self, parents)                     # [W_d, d + 1, Hq, D]
        W_d = widths[-1]
        feats = np.empty_like(feats_ref)
        feats[:, 0] = self_[0][u][0]
        for l in range(1, d + 1):
            feats[:, l] = self_[l][u][anc[d & 1, u, :W_d, l - 1]]
        assert rel(feats, feats_ref) <= TOL, f"user {u}: ranking features {rel(feats, feats_ref):.3e}"
        ref_t = target_attention(q_cand[u], Ku, Vu, scale)
        assert rel(f64(tgt_fused)[u], ref_t) <= TOL and rel(f64(tgt_two)[u], ref_t) <= TOL, f"user {u}: target attention"


def test_encdec_small_all_users():
    _run("encdec_small")


def test_encdec_full_size_whole_users():
    _run("encdec", users=[0, 15])
