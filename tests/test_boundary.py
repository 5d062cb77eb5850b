"""The C-ABI library loads, exports every symbol include/stark.h declares, and validates
arguments before any CUDA call (no GPU needed)."""
import ctypes
import os
import re

import pytest
import torch

from paper_2607_04068_b200 import binding as sb
from paper_2607_04068_b200.build import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build()
    return sb.lib()


def test_exports_match_header(L):
    hdr = open(os.path.join(ROOT, "include", "stark.h")).read()
    declared = set(re.findall(r"\b(stark_[a-z_]+)\s*\(", hdr))
    assert declared == set(sb.EXPORTS), declared ^ set(sb.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    assert L.stark_version() == 100


def test_status_strings(L):
    for code in (0, -1, -2, -3, -4):
        assert L.stark_status_string(code).decode().startswith("STARK_")
    assert b"unknown" in L.stark_status_string(-99)


def test_sizes(L):
    sh = sb.make_shape(3, 8, 2, 64, 4, 10, torch.bfloat16)
    assert L.stark_suffix_bytes(ctypes.byref(sh)) == 4 * 3 * 10 * 2 * 64 * 2
    assert L.stark_anc_bytes(ctypes.byref(sh)) == 2 * 3 * 10 * 4 * 4
    bad = sb.make_shape(3, 8, 3, 64, 4, 10, torch.bfloat16)     # Hq % Hkv != 0
    assert L.stark_suffix_bytes(ctypes.byref(bad)) == 0


def test_plan_is_deterministic_and_positive(L):
    sh = sb.make_shape(16, 16, 4, 128, 3, 64, torch.bfloat16)
    a = sb.stark_prefix_attn_plan(sh, 1, 16 * 1024, 1024)
    b = sb.stark_prefix_attn_plan(sh, 1, 16 * 1024, 1024)
    assert a == b and 1 <= a <= 64
    assert 1 <= sb.stark_prefix_attn_plan(sh, 64, 16 * 1024, 1024) <= 64


def test_validation_before_cuda(L):
    sh = sb.make_shape(1, 4, 4, 64, 3, 8, torch.float32)
    p = ctypes.c_void_p(16)     # non-null dummy, never dereferenced: validation fails first
    assert L.stark_prefix_attn(ctypes.byref(sh), None, 1, p, p, p, 1, 1, 1, p, p, p, None, 0, None) == -1
    assert L.stark_prefix_attn(ctypes.byref(sh), p, 0, p, p, p, 1, 1, 1, p, p, p, None, 0, None) == -1
    assert L.stark_prefix_attn(ctypes.byref(sh), p, 1, p, p, p, 1, 1, 65, p, p, p, None, 0, None) == -1
    bad_d = sb.make_shape(1, 4, 4, 96, 3, 8, torch.float32)
    assert L.stark_prefix_attn(ctypes.byref(bad_d), p, 1, p, p, p, 1, 1, 1, p, p, p, None, 0, None) == -2
    assert L.stark_tree_attn_step(ctypes.byref(sh), p, 1, 4, p, p, p, p, p, p, 1, p, None) == -1   # level > d
    assert L.stark_tree_attn_step(ctypes.byref(sh), p, 9, 1, p, p, p, p, p, p, 1, p, None) == -1   # n_q > Wmax
    assert L.stark_beam_topk(p, None, 1, 2, 4, 9, p, p, p, None, 0, None) == -1                    # W_out > W_in*C
    assert L.stark_beam_topk(p, None, 1, 1 << 16, 1 << 16, 4, p, p, p, None, 0, None) == -1        # >= 2^31
    # selection from raw logits: same argument rules; the workspace (per-beam offsets) is mandatory
    assert L.stark_beam_topk_logits(None, None, 1, 2, 4, 2, p, p, p, p, 1 << 20, None) == -1        # logits missing
    assert L.stark_beam_topk_logits(p, None, 1, 2, 4, 9, p, p, p, p, 1 << 20, None) == -1          # W_out > W_in*C
    assert L.stark_beam_topk_logits(p, None, 1, 2, 4, 2, p, p, p, None, 0, None) == -3             # no workspace
    assert L.stark_beam_topk_logits(p, None, 1, 2, 4, 2, p, p, p, p, 8, None) == -3                # too small
    assert L.stark_logits_row_offset(p, None, 0, 4, p, None) == -1                                 # rows < 1
    assert L.stark_logits_row_offset(p, None, 4, 4, None, None) == -1                              # offset missing
    need = L.stark_workspace_bytes(ctypes.byref(sh), sb.CALL_BEAM_TOPK_LOGITS, 8, 32)
    assert need >= 1 * 8 * 4 and need % 256 == L.stark_workspace_bytes(ctypes.byref(sh), sb.CALL_BEAM_TOPK, 8, 32) % 256
    assert L.stark_kv_append_reorg(ctypes.byref(sh), 0, 1, p, p, p, p, p, p, None) == -1           # level < 1
    assert L.stark_kv_append_reorg(ctypes.byref(sh), 2, 1, p, p, None, p, p, p, None) == -1        # parent missing
    # fused decode attention: argument errors first, then "bf16 only" (fp32 shapes compose A1 + A2)
    bf = sb.make_shape(2, 8, 2, 128, 3, 8, torch.bfloat16)
    assert L.stark_decode_attn(ctypes.byref(bf), None, 1, 0, p, p, p, 4, 4, p, p, p, p, None) == -1   # q missing
    assert L.stark_decode_attn(ctypes.byref(bf), p, 1, 4, p, p, p, 4, 4, p, p, p, p, None) == -1      # level > d
    assert L.stark_decode_attn(ctypes.byref(bf), p, 9, 1, p, p, p, 4, 4, p, p, p, p, None) == -1      # n_q > Wmax
    assert L.stark_decode_attn(ctypes.byref(bf), p, 1, 1, p, p, p, 4, 4, p, p, None, p, None) == -1   # anc missing
    assert L.stark_decode_attn(ctypes.byref(sh), p, 1, 0, p, p, p, 4, 4, p, p, p, p, None) == -2      # fp32
    # single-launch step: (shape, q, n_q, level, kp, vp, cu, total, max_len, k_new, v_new, parent, ks, vs, anc, w, out, st)
    step = lambda s, *a: L.stark_decode_step(ctypes.byref(s), *a)
    assert step(bf, None, 1, 0, p, p, p, 4, 4, None, None, None, None, None, None, 1, p, None) == -1  # q missing
    assert step(bf, p, 1, 4, p, p, p, 4, 4, p, p, p, p, p, p, 1, p, None) == -1                      # level > d
    assert step(bf, p, 9, 1, p, p, p, 4, 4, p, p, None, p, p, p, 1, p, None) == -1                   # n_q > Wmax
    assert step(bf, p, 1, 1, p, p, p, 4, 4, None, p, None, p, p, p, 1, p, None) == -1                # k_new missing
    assert step(bf, p, 1, 2, p, p, p, 4, 4, p, p, None, p, p, p, 0, p, None) == -1                   # parent missing
    assert step(sh, p, 1, 0, p, p, p, 4, 4, None, None, None, None, None, None, 1, p, None) == -2    # fp32


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful without a GPU")
def test_no_cpu_fallback(L):
    """Without a device a well-formed call fails loudly (never computes on the CPU)."""
    sh = sb.make_shape(1, 4, 4, 64, 3, 8, torch.float32)
    p = ctypes.c_void_p(16)
    rc = L.stark_beam_topk(p, None, 1, 2, 4, 2, p, p, p, None, 0, None)
    assert rc in (-2, -4)


def test_topk_workspace_rule(L):
    """Large candidate sets need the (zero-filled) workspace stark_workspace_bytes reports; small ones need none."""
    p = ctypes.c_void_p(16)
    sh = sb.make_shape(2, 1, 1, 64, 1, 512, torch.float32)
    assert sb.stark_workspace_bytes(sh, sb.CALL_BEAM_TOPK, 1, 256) == 0
    need = sb.stark_workspace_bytes(sh, sb.CALL_BEAM_TOPK, 512, 8192)
    assert need > 0 and need == sb.stark_workspace_bytes(sh, sb.CALL_BEAM_TOPK, 512, 8192)
    assert L.stark_beam_topk(p, None, 2, 512, 8192, 512, p, p, p, None, 0, None) == -3        # no workspace
    assert L.stark_beam_topk(p, None, 2, 512, 8192, 512, p, p, p, p, need - 1, None) == -3    # too small
    assert sb.stark_workspace_bytes(sh, sb.CALL_BEAM_TOPK_LOGITS, 512, 8192) > need           # + the per-beam offsets
