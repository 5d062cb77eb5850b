"""Shapes of the five BASELINE.json configs, scaled-down parity variants, and
the paper-scale workload (PAPER.md:126 codebook 8192, PAPER.md:306 beam widths
(512, 512, 1024), PAPER.md:304 GQA 4:1, PAPER.md:278-280 batch sizes 1 and 8).

Shapes only.  No arithmetic of the method lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Dict, List, Tuple


@dataclass(frozen=True)
class StarkConfig:
    name: str
    config_id: int            # enters the RNG key (reading S19)
    dtype: str                # "f32" | "bf16": element type of q/k/v/out
    B: int                    # users
    Hq: int                   # query heads
    Hkv: int                  # KV heads (GQA group G = Hq // Hkv)
    D: int                    # head_dim
    prefix_min: int           # prefix length range, inclusive (equal => fixed)
    prefix_max: int
    W: Tuple[int, ...]        # beam width after each level's selection (len d)
    d: int                    # SID levels
    C: int                    # codebook size per level
    kv_std: float = 1.0       # std of K/V draws (reading S13: N(a,b) => b is std)
    q_std: float = 1.0
    logits: str = "normal"    # "normal" | "mixture" | "projection"
    logits_std: float = 2.0
    per_head_scale: bool = False   # config 5 (reading S16)

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def Wmax(self) -> int:
        return max(beam_widths(self))

    @property
    def elem_bytes(self) -> int:
        return 4 if self.dtype == "f32" else 2


def beam_widths(cfg: StarkConfig) -> List[int]:
    """Live beams after the selection of level t+1, t = 0..d-1 (reading S7):
    W_out = min(W_level, W_in * C), with W_in = 1 at step 0."""
    out, w_in = [], 1
    for t in range(cfg.d):
        w = min(cfg.W[t], w_in * cfg.C)
        out.append(w)
        w_in = w
    return out


def queries_per_step(cfg: StarkConfig) -> List[int]:
    """n_q at decode step t = 0..d (step d is the optional ranking-feature
    step, reading S2)."""
    return [1] + beam_widths(cfg)


CONFIGS: Dict[str, StarkConfig] = {}


def _add(c: StarkConfig) -> StarkConfig:
    CONFIGS[c.name] = c
    return c


# --- BASELINE.json configs[0..4] -------------------------------------------
CFG1 = _add(StarkConfig("cfg1", 1, "f32", B=1, Hq=4, Hkv=4, D=64,
                        prefix_min=128, prefix_max=128, W=(8, 8, 8), d=3, C=32,
                        kv_std=0.125, q_std=0.125, logits="projection"))
CFG2 = _add(StarkConfig("cfg2", 2, "bf16", B=16, Hq=16, Hkv=4, D=128,
                        prefix_min=1024, prefix_max=1024, W=(64, 64, 64), d=3, C=256))
# cfg3's attention-side shape (the 12-layer decoder around it lives in the
# harness; its q/k/v come from the model, not from these draws).
CFG3 = _add(StarkConfig("cfg3", 3, "bf16", B=64, Hq=16, Hkv=4, D=64,
                        prefix_min=2048, prefix_max=2048, W=(128,) * 4, d=4, C=256))
CFG4 = _add(StarkConfig("cfg4", 4, "bf16", B=8, Hq=16, Hkv=4, D=128,
                        prefix_min=512, prefix_max=512, W=(512,) * 3, d=3, C=1024,
                        logits="mixture"))
CFG5 = _add(StarkConfig("cfg5", 5, "bf16", B=32, Hq=32, Hkv=8, D=128,
                        prefix_min=1024, prefix_max=8192, W=(256,) * 4, d=4, C=256,
                        per_head_scale=True))

# --- paper-scale workload ---------------------------------
PAPER_B1 = _add(replace(CFG2, name="paper_b1", config_id=11, B=1,
                        W=(512, 512, 1024), C=8192))
PAPER_B8 = _add(replace(CFG2, name="paper_b8", config_id=12, B=8,
                        W=(512, 512, 1024), C=8192))

# --- scaled-down parity variants: same structure, sizes the fp64 oracle
# finishes in seconds, still spanning several tiles and a ragged tail --------
CFG2_S = _add(replace(CFG2, name="cfg2_small", config_id=22, B=3,
                      prefix_min=333, prefix_max=333, W=(24, 24, 24), C=48))
CFG3_S = _add(replace(CFG3, name="cfg3_small", config_id=23, B=2,
                      prefix_min=257, prefix_max=257, W=(40,) * 4, C=64))
CFG4_S = _add(replace(CFG4, name="cfg4_small", config_id=24, B=2,
                      prefix_min=200, prefix_max=200, W=(96,) * 3, C=160))
CFG5_S = _add(replace(CFG5, name="cfg5_small", config_id=25, B=4,
                      prefix_min=70, prefix_max=420, W=(36,) * 4, C=40))
PAPER_S = _add(replace(PAPER_B1, name="paper_small", config_id=26, B=2,
                       prefix_min=150, prefix_max=150, W=(16, 16, 40), C=96))
# fp32 with GQA and a non-trivial batch (cfg1 itself has G = 1, B = 1)
F32_GQA = _add(replace(CFG1, name="f32_gqa", config_id=27, B=3, Hq=8, Hkv=2,
                       prefix_min=50, prefix_max=190, W=(12, 12, 12), C=20,
                       kv_std=1.0, q_std=1.0, logits="normal"))


# --- the paper's encoder-decoder form (readings R23-R25): `prefix_*` is the length of
# the encoder memory M; the decoder's own fixed prefix [e_click, e_atc, e_pay, <bos>]
# (Eq. 7) has 4 rows per user.  cfg2's heads / memory length / beam / codebook.
ENCDEC = _add(replace(CFG2, name="encdec", config_id=31))
ENCDEC_S = _add(replace(CFG2, name="encdec_small", config_id=32, B=3, prefix_min=150, prefix_max=333,
                        W=(24, 24, 24), C=48))
N_FIXED = 4   # e_click, e_atc, e_pay, <bos>


def get_config(name: str) -> StarkConfig:
    return CONFIGS[name]
