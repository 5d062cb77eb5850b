"""Teacher-forced GPU-vs-oracle comparison protocol.

For one config: the oracle (conventional fp64 beam search, oracle/) runs per
user on the seeded draws of `workloads/`; the CUDA path (through the C ABI)
receives the identical fp32 log-probs and bf16/fp32 q/k/v.  Selection must be
bit-exact; attention within tol * max|out_ref| per call.
"""
from __future__ import annotations

import numpy as np
import torch

import workloads as wl
from oracle.beam_search import conventional_beam_search
from oracle.token_models import DrawTokenModel, TableTokenModel

from paper_2607_04068_b200.decode import StarkLayer, beam_topk

TOL = {"f32": 2e-3, "bf16": 1.5e-2}   # BASELINE.json north_star


def torch_dtype(cfg):
    return torch.float32 if cfg.dtype == "f32" else torch.bfloat16


def to_dev(x: np.ndarray, dtype=None) -> torch.Tensor:
    t = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return t.to(dtype).contiguous() if dtype is not None else t


def draws(cfg, seed=0, final_step=True):
    """All seeded inputs of a config: prefix + per-step q/k/v/logits (numpy)."""
    K, V, cu = wl.prefix_kv(cfg, seed)
    nq = wl.queries_per_step(cfg)
    steps = cfg.d + (1 if final_step else 0)
    if cfg.logits == "projection":      # config 1: q/k/v/logits come from the token tables
        return dict(K=K, V=V, cu=cu, tables=wl.config1_tables(cfg, seed), nq=nq, steps=steps)
    q, k, v, lg = [], [], [], []
    for t in range(steps):
        qq, kk, vv = wl.step_qkv(cfg, t, nq[t], seed)
        q.append(qq), k.append(kk), v.append(vv)
        if t < cfg.d:
            lg.append(wl.step_logits(cfg, t, nq[t], seed))
    return dict(K=K, V=V, cu=cu, q=q, k=k, v=v, lg=lg, nq=nq, steps=steps)


def oracle_traces(cfg, dr, users=None, final_step=True):
    scale = 1.0 / np.sqrt(cfg.D)
    cu = dr["cu"]
    out = {}
    for u in (range(cfg.B) if users is None else users):
        if "tables" in dr:
            m = TableTokenModel(dr["tables"])
        else:
            m = DrawTokenModel([x[u] for x in dr["q"]], [x[u] for x in dr["k"]], [x[u] for x in dr["v"]],
                               [x[u] for x in dr["lg"]])
        out[u] = conventional_beam_search(dr["K"][cu[u]:cu[u + 1]], dr["V"][cu[u]:cu[u + 1]], m, cfg.W, cfg.C,
                                          scale, final_step=final_step)
    return out


def make_layer(cfg, dr):
    dt = torch_dtype(cfg)
    lens = np.diff(dr["cu"])
    return StarkLayer(cfg.B, cfg.Hq, cfg.Hkv, cfg.D, cfg.d, cfg.Wmax, dt, to_dev(dr["K"], dt), to_dev(dr["V"], dt),
                      to_dev(dr["cu"].astype(np.int32)), int(lens.max()))


def run_teacher_forced(cfg, seed=0, final_step=True):
    """Returns a list of (what, step, ok, detail) and raises nothing: the test asserts."""
    dr = draws(cfg, seed, final_step)
    tr = oracle_traces(cfg, dr, final_step=final_step)
    layer = make_layer(cfg, dr)
    dt = torch_dtype(cfg)
    # a second layer takes every step through the single-launch boundary (stark_decode_step, bf16 only)
    layer_s = make_layer(cfg, dr) if cfg.dtype == "bf16" else None
    tol = TOL[cfg.dtype]
    report = []
    score = parent = None
    for t in range(dr["steps"]):
        # the oracle's trace holds the exact q / k_new / v_new it consumed (teacher forcing)
        q = to_dev(np.stack([tr[u].q[t] for u in range(cfg.B)]).astype(np.float32), dt)
        if t >= 1:
            kn = np.stack([tr[u].k_new[t] for u in range(cfg.B)]).astype(np.float32)
            vn = np.stack([tr[u].v_new[t] for u in range(cfg.B)]).astype(np.float32)
            kn, vn = to_dev(kn, dt), to_dev(vn, dt)
            layer.append(t, kn, vn, parent)
        else:
            kn = vn = None
        ref = np.stack([tr[u].attn_out[t] for u in range(cfg.B)])
        # both boundaries: A1 then A2 (partials through HBM), and the fused single launch (bf16 only)
        for what, fused in (("attn", False),) + ((("attn_fused", True),) if cfg.dtype == "bf16" else ()):
            out = layer.attend(t, q, fused=fused).float().cpu().numpy().astype(np.float64)
            err = np.abs(out - ref).max() / np.abs(ref).max()
            report.append((what, t, bool(np.isfinite(out).all() and err <= tol), f"rel_err={err:.3e} tol={tol}"))
        if layer_s is not None:
            out = layer_s.step(t, q, kn, vn, parent).float().cpu().numpy().astype(np.float64)
            err = np.abs(out - ref).max() / np.abs(ref).max()
            report.append(("attn_step", t, bool(np.isfinite(out).all() and err <= tol), f"rel_err={err:.3e} tol={tol}"))
            if t >= 1:   # the inline append left the same suffix rows and index rows as stark_kv_append_reorg
                n = q.shape[1]
                same = (torch.equal(layer_s.k_suffix[t - 1][:, :n], layer.k_suffix[t - 1][:, :n])
                        and torch.equal(layer_s.v_suffix[t - 1][:, :n], layer.v_suffix[t - 1][:, :n])
                        and torch.equal(layer_s.anc[t & 1, :, :n, :t], layer.anc[t & 1, :, :n, :t]))
                report.append(("step_append_state", t, bool(same), ""))
        if t == cfg.d:
            break
        logp = np.stack([tr[u].logp[t] for u in range(cfg.B)])            # fp32, the oracle's O3 output
        W_out = len(tr[0].parents[t])
        s_g, p_g, c_g = beam_topk(to_dev(logp), score, W_out)
        s_r = np.stack([tr[u].scores[t] for u in range(cfg.B)])
        p_r = np.stack([tr[u].parents[t] for u in range(cfg.B)])
        c_r = np.stack([tr[u].codes[t] for u in range(cfg.B)])
        ok = (np.array_equal(p_g.cpu().numpy(), p_r) and np.array_equal(c_g.cpu().numpy(), c_r)
              and np.array_equal(s_g.cpu().numpy().view(np.uint32), s_r.view(np.uint32)))
        report.append(("topk", t, bool(ok), f"W_out={W_out}"))
        score, parent = s_g, p_g
        if not ok:     # keep the tree identical to the oracle's for the later attention checks
            score, parent = to_dev(s_r), to_dev(p_r)
    return report


# ---- full-size configs: the launch configuration bench.py times, sampled oracle checks -------------
def run_full_size(cfg, n_samples=6, seed=0, use_graph=True, from_logits=False):
    """Free-running DecodePass (bench.py's own object, CUDA-graph replay) at BASELINE.json's full size.
    Checks: (a) every level's selection, ALL users, bit-exact vs oracle.select_beams on the identical fp32
    log-probs and scores; (b) the ancestor index vs oracle.ancestor_chains and the suffix K/V (bitwise copy);
    (c) ALL attention rows of whole users (first, last, shortest, longest prefix) vs
    oracle.sequence_expanded_attention (fp64) plus sampled rows of other users vs the per-beam replay; (d) the prefix buffers are bit-identical before/after."""
    import bench
    from oracle.selection import select_beams, select_beams_from_logits
    from oracle.tree import ancestor_chains, sequence_expanded_attention
    from oracle.replay import replay_beam_attention
    h = bench.host_inputs(cfg, seed)
    p = bench.make_pass(cfg, h, torch.device("cuda"), from_logits=from_logits)
    oracle_select = select_beams_from_logits if from_logits else select_beams   # p.logp holds raw logits then
    kp0, vp0 = p.layer.k_prefix.clone(), p.layer.v_prefix.clone()
    p.run()
    torch.cuda.synchronize()
    if use_graph:
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            p.run()
        for s in p.sel:                       # poison the outputs: the replay must rewrite them
            s[1].fill_(-7)
        g.replay()
        torch.cuda.synchronize()
    report = []
    tol, scale = TOL[cfg.dtype], 1.0 / np.sqrt(cfg.D)
    report.append(("prefix_untouched", -1, bool(torch.equal(kp0, p.layer.k_prefix) and torch.equal(vp0, p.layer.v_prefix)), ""))
    logp = [x.cpu().numpy() for x in p.logp]
    sel = [[x.cpu().numpy() for x in s] for s in p.sel]
    rng = np.random.default_rng(1234 + cfg.config_id)
    cu = h["cu"]
    ks = p.layer.k_suffix.float().cpu().numpy()
    vs = p.layer.v_suffix.float().cpu().numpy()
    anc = p.layer.anc.cpu().numpy()
    for t in range(cfg.d):
        # (a) selection
        ok = True
        for u in range(cfg.B):
            score = np.zeros(1, np.float32) if t == 0 else sel[t - 1][0][u]
            s_r, p_r, c_r = oracle_select(score, logp[t][u], p.widths[t])
            ok &= (np.array_equal(sel[t][1][u], p_r) and np.array_equal(sel[t][2][u], c_r)
                   and np.array_equal(sel[t][0][u].view(np.uint32), s_r.view(np.uint32)))
        report.append(("topk_all_users", t, bool(ok), f"N={logp[t].shape[1] * cfg.C} W_out={p.widths[t]}"))
        if t == 0:
            pass
        else:
            # (b) append: K/V of level t are a bitwise copy; anc rows follow the parents
            n = p.n_q[t]
            ok_kv = np.array_equal(ks[t - 1][:, :n], h["k"][t]) and np.array_equal(vs[t - 1][:, :n], h["v"][t])
            ok_anc = True
            for u in range(cfg.B):
                parents = [sel[l][1][u] for l in range(t)]
                ok_anc &= np.array_equal(anc[t & 1, u, :n, :t], ancestor_chains(parents, t))
            report.append(("append_kv_bitwise", t, bool(ok_kv), ""))
            if t + 2 > cfg.d - 1:      # anc ping-pongs by level parity: level t's half is reused by level t+2
                report.append(("anc_vs_oracle_chains", t, bool(ok_anc), ""))
        # (c) attention, ALL rows of whole users (first, last, shortest and longest prefix) vs the oracle's
        # sequence-expanded masked attention (Eq. 14, oracle/tree.py; pinned equal to the conventional per-beam
        # form), plus a few sampled (user, beam) rows of the other users vs the conventional per-beam replay.
        # NOTE: after the whole pass anc/suffix hold the final state; level-t rows are never overwritten by
        # later levels, so every step can be checked afterwards.
        out = p.out[t].float().cpu().numpy().astype(np.float64)
        worst, ref_max = 0.0, 0.0
        lens = np.diff(cu)
        whole = sorted({0, cfg.B - 1, int(np.argmin(lens)), int(np.argmax(lens))})
        for u in whole:
            parents = [sel[l][1][u] for l in range(t)]
            ref = sequence_expanded_attention(h["K"][cu[u]:cu[u + 1]], h["V"][cu[u]:cu[u + 1]],
                                              [h["k"][l][u] for l in range(1, t + 1)],
                                              [h["v"][l][u] for l in range(1, t + 1)], parents, h["q"][t][u], t, scale)
            worst = max(worst, float(np.abs(out[u] - ref).max()))
            ref_max = max(ref_max, float(np.abs(ref).max()))
        for _ in range(n_samples):
            u, i = int(rng.integers(cfg.B)), int(rng.integers(p.n_q[t]))
            parents = [sel[l][1][u] for l in range(t)]
            ref = replay_beam_attention(h["K"][cu[u]:cu[u + 1]], h["V"][cu[u]:cu[u + 1]],
                                        [h["k"][l][u] for l in range(1, t + 1)], [h["v"][l][u] for l in range(1, t + 1)],
                                        parents, h["q"][t][u, i], i, t, scale)
            worst = max(worst, float(np.abs(out[u, i] - ref).max()))
            ref_max = max(ref_max, float(np.abs(ref).max()))
        report.append(("attn_whole_users", t, bool(np.isfinite(out).all() and worst <= tol * ref_max),
                       f"users={whole} (+{n_samples} sampled rows) max_abs_err={worst:.3e} max|ref|={ref_max:.3e} tol={tol}"))
    return report
