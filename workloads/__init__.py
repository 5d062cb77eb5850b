"""Seeded synthetic inputs for the STARK decode path.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2607_04068_b200/`).  It holds shapes and random-number draws and
nothing else: no attention, no softmax, no selection, no tree bookkeeping.

The recipes follow BASELINE.json `configs[0..4]` as read in SURVEY.md §8(d) and
DESIGN.md §4 (readings S13-S16, S19).  Stand-ins: the paper's Lazada logs and
trained weights are confidential (§4.1.1), so every tensor
here is a seeded draw with the shape and structure of the paper's workload
(one long shared user history, d = 3-4 SID levels, per-level codebook, wide
beam, GQA 4:1 — PAPER.md:126, 138, 304, 306).
"""
from .configs import StarkConfig, CONFIGS, N_FIXED, get_config, beam_widths, queries_per_step  # noqa: F401
from .generate import (  # noqa: F401
    rng_for,
    round_to_bf16,
    prefix_lengths,
    prefix_kv,
    prefix_kv_user,
    head_scales,
    step_qkv,
    step_logits,
    config1_tables,
    tie_logits,
    fixed_prefix_kv,
    step_q_cross,
)
