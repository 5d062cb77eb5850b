"""Seeded draws (reading S19: numpy.random.default_rng([seed, config_id, tag,
...]) on the host; identical arrays go to the oracle and to the GPU).

Every function returns plain numpy arrays.  For bf16 configs the draws are
rounded to bf16 here (stored as float32 with the low 16 bits clear), *before*
either side sees them (SURVEY.md §8c comparison protocol), so that the oracle
upcasts exactly the values the GPU reads.

No arithmetic of the method (attention, softmax, selection, tree indexing)
lives in this file.
"""
from __future__ import annotations

from typing import Dict, Iterable, Optional, Tuple

import numpy as np

from .configs import StarkConfig

# RNG stream tags
_T_LEN, _T_PREFIX, _T_SCALE, _T_STEP, _T_LOGITS, _T_TABLES, _T_FIXED, _T_QCROSS = 1, 2, 3, 4, 5, 6, 7, 8


def rng_for(seed: int, cfg: StarkConfig, tag: int, *idx: int) -> np.random.Generator:
    return np.random.default_rng([int(seed), int(cfg.config_id), int(tag), *[int(i) for i in idx]])


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest bfloat16 (ties to even); the result is
    float32 whose low 16 bits are zero (so a later cast to bf16 is exact)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    bias = np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
    r = (u + bias) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def _finish(x: np.ndarray, cfg: StarkConfig) -> np.ndarray:
    x = x.astype(np.float32, copy=False)
    return round_to_bf16(x) if cfg.dtype == "bf16" else x


def prefix_lengths(cfg: StarkConfig, seed: int = 0) -> np.ndarray:
    """L_u per user; config 5: rng.integers(prefix_min, prefix_max + 1)."""
    if cfg.prefix_min == cfg.prefix_max:
        return np.full(cfg.B, cfg.prefix_min, dtype=np.int64)
    g = rng_for(seed, cfg, _T_LEN)
    return g.integers(cfg.prefix_min, cfg.prefix_max + 1, size=cfg.B).astype(np.int64)


def head_scales(cfg: StarkConfig, seed: int = 0) -> Tuple[np.ndarray, np.ndarray]:
    """Per-KV-head scales sK[h], sV[h] (reading S16); ones unless config 5."""
    if not cfg.per_head_scale:
        one = np.ones(cfg.Hkv, dtype=np.float32)
        return one, one
    g = rng_for(seed, cfg, _T_SCALE)
    sk = g.uniform(0.5, 2.0, size=cfg.Hkv).astype(np.float32)
    sv = g.uniform(0.5, 2.0, size=cfg.Hkv).astype(np.float32)
    return sk, sv


def prefix_kv_user(cfg: StarkConfig, u: int, L: int, seed: int = 0) -> Tuple[np.ndarray, np.ndarray]:
    """K, V of one user's history: [L, Hkv, D], one RNG stream per user so
    that a subset of users can be generated on its own."""
    sk, sv = head_scales(cfg, seed)
    g = rng_for(seed, cfg, _T_PREFIX, u)
    k = g.standard_normal((L, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
    v = g.standard_normal((L, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
    k *= sk[None, :, None]
    v *= sv[None, :, None]
    return _finish(k, cfg), _finish(v, cfg)


def prefix_kv(cfg: StarkConfig, seed: int = 0) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Packed prefix K/V [total_tokens, Hkv, D] and cu_seqlens[B+1] (int32)."""
    lens = prefix_lengths(cfg, seed)
    cu = np.zeros(cfg.B + 1, dtype=np.int32)
    cu[1:] = np.cumsum(lens)
    total = int(cu[-1])
    K = np.empty((total, cfg.Hkv, cfg.D), dtype=np.float32)
    V = np.empty((total, cfg.Hkv, cfg.D), dtype=np.float32)
    for u in range(cfg.B):
        K[cu[u]:cu[u + 1]], V[cu[u]:cu[u + 1]] = prefix_kv_user(cfg, u, int(lens[u]), seed)
    return K, V, cu


def step_qkv(cfg: StarkConfig, t: int, n_q: int, seed: int = 0,
             users: Optional[Iterable[int]] = None) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Fresh draws per (step, user, slot) (reading S15): q [U, n_q, Hq, D],
    k_new, v_new [U, n_q, Hkv, D].  At step 0 k_new/v_new are drawn but unused
    (the root query's K/V are the last prefix row)."""
    users = list(range(cfg.B)) if users is None else list(users)
    sk, sv = head_scales(cfg, seed)
    q = np.empty((len(users), n_q, cfg.Hq, cfg.D), dtype=np.float32)
    k = np.empty((len(users), n_q, cfg.Hkv, cfg.D), dtype=np.float32)
    v = np.empty((len(users), n_q, cfg.Hkv, cfg.D), dtype=np.float32)
    for j, u in enumerate(users):
        g = rng_for(seed, cfg, _T_STEP, t, u)
        q[j] = g.standard_normal((n_q, cfg.Hq, cfg.D), dtype=np.float32) * np.float32(cfg.q_std)
        k[j] = g.standard_normal((n_q, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
        v[j] = g.standard_normal((n_q, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
    k *= sk[None, None, :, None]
    v *= sv[None, None, :, None]
    return _finish(q, cfg), _finish(k, cfg), _finish(v, cfg)


def step_logits(cfg: StarkConfig, t: int, n_q: int, seed: int = 0,
                users: Optional[Iterable[int]] = None) -> np.ndarray:
    """Raw logits [U, n_q, C] float32 for the level selected after step t.
    "normal": N(0, logits_std);  "mixture" (config 4): each entry N(0,1) with
    probability 0.9, else N(3, std 0.5), to create near-ties."""
    users = list(range(cfg.B)) if users is None else list(users)
    out = np.empty((len(users), n_q, cfg.C), dtype=np.float32)
    for j, u in enumerate(users):
        g = rng_for(seed, cfg, _T_LOGITS, t, u)
        if cfg.logits == "mixture":
            a = g.standard_normal((n_q, cfg.C), dtype=np.float32)
            b = g.standard_normal((n_q, cfg.C), dtype=np.float32) * np.float32(0.5) + np.float32(3.0)
            pick = g.random((n_q, cfg.C), dtype=np.float32) < np.float32(0.9)
            out[j] = np.where(pick, a, b)
        else:
            out[j] = g.standard_normal((n_q, cfg.C), dtype=np.float32) * np.float32(cfg.logits_std)
    return out


def fixed_prefix_kv(cfg: StarkConfig, seed: int = 0, n_fixed: int = 4) -> Tuple[np.ndarray, np.ndarray]:
    """Encoder-decoder form: self-attention K, V of the decoder's fixed prefix positions
    [e_click, e_atc, e_pay, <bos>] (Eq. 7), per user: [B, n_fixed, Hkv, D] ~ N(0, kv_std)."""
    g = rng_for(seed, cfg, _T_FIXED)
    k = g.standard_normal((cfg.B, n_fixed, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
    v = g.standard_normal((cfg.B, n_fixed, cfg.Hkv, cfg.D), dtype=np.float32) * np.float32(cfg.kv_std)
    return _finish(k, cfg), _finish(v, cfg)


def step_q_cross(cfg: StarkConfig, t: int, n_q: int, seed: int = 0) -> np.ndarray:
    """Encoder-decoder form: the cross-attention queries of step t (a projection of their own):
    [B, n_q, Hq, D] ~ N(0, q_std), fresh draws per (step, user, slot) like step_qkv."""
    out = np.empty((cfg.B, n_q, cfg.Hq, cfg.D), dtype=np.float32)
    for u in range(cfg.B):
        g = rng_for(seed, cfg, _T_QCROSS, t, u)
        out[u] = g.standard_normal((n_q, cfg.Hq, cfg.D), dtype=np.float32) * np.float32(cfg.q_std)
    return _finish(out, cfg)


def tie_logits(logits: np.ndarray) -> np.ndarray:
    """Exact-tie variant for parity only: logits
    quantised to multiples of 1/8 so that many candidates share a key."""
    return (np.round(logits.astype(np.float32) * np.float32(8.0)) / np.float32(8.0)).astype(np.float32)


def config1_tables(cfg: StarkConfig, seed: int = 0) -> Dict[str, np.ndarray]:
    """Config 1's token model (reading S14): per-level tables indexed by code,
    a root query, and a fixed projection + bias per level, shared by beams.

      Tq[l][c] in R^{Hq x D}, Tk[l][c], Tv[l][c] in R^{Hkv x D}  ~ N(0,1)*q_std / kv_std
      q_root in R^{Hq x D}                                        ~ N(0,1)*q_std
      P[l] in R^{(Hq*D) x C}  ~ N(0, std 1/sqrt(64) = 0.125);  b[l] in R^C ~ N(0,1)
    """
    g = rng_for(seed, cfg, _T_TABLES)
    d, C, Hq, Hkv, D = cfg.d, cfg.C, cfg.Hq, cfg.Hkv, cfg.D
    t = {
        "Tq": g.standard_normal((d, C, Hq, D), dtype=np.float32) * np.float32(cfg.q_std),
        "Tk": g.standard_normal((d, C, Hkv, D), dtype=np.float32) * np.float32(cfg.kv_std),
        "Tv": g.standard_normal((d, C, Hkv, D), dtype=np.float32) * np.float32(cfg.kv_std),
        "q_root": g.standard_normal((Hq, D), dtype=np.float32) * np.float32(cfg.q_std),
        "P": g.standard_normal((d, Hq * D, C), dtype=np.float32) * np.float32(0.125),
        "b": g.standard_normal((d, C), dtype=np.float32),
    }
    return {k: _finish(v, cfg) if k in ("Tq", "Tk", "Tv", "q_root") else v.astype(np.float32)
            for k, v in t.items()}
