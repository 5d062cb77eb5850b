"""Token models for the oracle's beam search (oracle; test infrastructure).

The paper's decoder is out of scope; BASELINE.json's configs
replace it by synthetic sources of q/k/v and logits (readings R14,
R15).  These adapters only index the seeded arrays of `workloads/` and, for
config 1, apply the fixed projection that turns an attention output into
logits -- in fp64, independent of the GPU harness (which does the same
projection in torch fp32 on the device).
"""
from __future__ import annotations

import numpy as np


class TableTokenModel:
    """Config 1 (reading R14): q/k/v of a generated token depend only on its
    (level, code): Tq[l][c], Tk[l][c], Tv[l][c]; the root query is q_root;
    logits_t = P[t]^T vec(out) + b[t].  Path-determined, hence usable by the
    brute-force enumerator."""

    def __init__(self, tables):
        self.t = {k: np.asarray(v, dtype=np.float64) for k, v in tables.items()}

    def qkv(self, t, slot, path):
        if t == 0:
            return self.t["q_root"], None, None
        lvl, code = t - 1, path[-1]          # token of level t sits in table row t-1
        return self.t["Tq"][lvl, code], self.t["Tk"][lvl, code], self.t["Tv"][lvl, code]

    def logits(self, t, slot, path, o):
        return o.reshape(-1) @ self.t["P"][t] + self.t["b"][t]


class DrawTokenModel:
    """Configs 2/4/5 (reading R15): fresh draws per (step, user, slot); logits
    given directly.  `q[t]`, `k[t]`, `v[t]` are [n_q, H, D] for ONE user and
    `lg[t]` is [n_q, C]."""

    def __init__(self, q, k, v, lg):
        self.q, self.k, self.v, self.lg = q, k, v, lg

    def qkv(self, t, slot, path):
        return self.q[t][slot], self.k[t][slot], self.v[t][slot]

    def logits(self, t, slot, path, o):
        return self.lg[t][slot]
