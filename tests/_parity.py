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
    tol = TOL[cfg.dtype]
    report = []
    score = parent = None
    for t in range(dr["steps"]):
        # the oracle's trace holds the exact q / k_new / v_new it consumed (teacher forcing)
        q = to_dev(np.stack([tr[u].q[t] for u in range(cfg.B)]).astype(np.float32), dt)
        if t >= 1:
            kn = np.stack([tr[u].k_new[t] for u in range(cfg.B)]).astype(np.float32)
            vn = np.stack([tr[u].v_new[t] for u in range(cfg.B)]).astype(np.float32)
            layer.append(t, to_dev(kn, dt), to_dev(vn, dt), parent)
        out = layer.attend(t, q).float().cpu().numpy().astype(np.float64)
        ref = np.stack([tr[u].attn_out[t] for u in range(cfg.B)])
        err = np.abs(out - ref).max() / np.abs(ref).max()
        report.append(("attn", t, bool(np.isfinite(out).all() and err <= tol), f"rel_err={err:.3e} tol={tol}"))
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
