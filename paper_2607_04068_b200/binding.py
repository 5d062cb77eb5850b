"""Thin ctypes binding of libstark.so (C ABI declared in include/stark.h).

Argument marshalling only: every step of the hot path runs inside the CUDA
kernels of the library.  PyTorch supplies device memory and the stream.  There
is no CPU fallback: a missing library or a non-zero status raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_float, c_int, c_int32, c_int64, c_size_t, c_void_p
from typing import Optional, Tuple

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libstark.so")

STARK_F32, STARK_BF16 = 0, 1
CALL_PREFIX_ATTN, CALL_TREE_ATTN_STEP, CALL_BEAM_TOPK, CALL_KV_APPEND_REORG, CALL_BEAM_TOPK_LOGITS = 0, 1, 2, 3, 4
EXPORTS = (
    "stark_prefix_attn", "stark_prefix_attn_plan", "stark_tree_attn_step", "stark_decode_attn", "stark_decode_step",
    "stark_beam_topk", "stark_beam_topk_static", "stark_logits_row_offset", "stark_beam_topk_logits",
    "stark_kv_append_reorg", "stark_workspace_bytes", "stark_suffix_bytes",
    "stark_anc_bytes", "stark_version", "stark_status_string", "stark_last_cuda_error",
)


class StarkError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().stark_status_string(status).decode()
        if status == -4:
            msg += f" [cudaError {lib().stark_last_cuda_error()}]"
        super().__init__(f"{where}: {msg}")


class Shape(Structure):
    """Mirror of stark_shape_t."""
    _fields_ = [("B", c_int32), ("Hq", c_int32), ("Hkv", c_int32), ("D", c_int32), ("d", c_int32),
                ("Wmax", c_int32), ("dtype", c_int32), ("softmax_scale", c_float)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libstark.so (built in-tree by paper_2607_04068_b200.build); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2607_04068_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    P = POINTER(Shape)
    L.stark_prefix_attn.restype = c_int
    L.stark_prefix_attn.argtypes = [P, c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int, c_int,
                                    c_void_p, c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
    L.stark_prefix_attn_plan.restype = c_int
    L.stark_prefix_attn_plan.argtypes = [P, c_int, c_int, c_int, POINTER(c_int)]
    L.stark_tree_attn_step.restype = c_int
    L.stark_tree_attn_step.argtypes = [P, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p,
                                       c_void_p, c_void_p, c_int, c_void_p, c_void_p]
    L.stark_decode_attn.restype = c_int
    L.stark_decode_attn.argtypes = [P, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p,
                                    c_void_p, c_void_p, c_void_p, c_void_p]
    L.stark_decode_step.restype = c_int
    L.stark_decode_step.argtypes = [P, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p,
                                    c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p]
    L.stark_beam_topk.restype = c_int
    L.stark_beam_topk.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p,
                                  c_void_p, c_size_t, c_void_p]
    L.stark_beam_topk_static.restype = c_int
    L.stark_beam_topk_static.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p,
                                         c_void_p]
    L.stark_logits_row_offset.restype = c_int
    L.stark_logits_row_offset.argtypes = [c_void_p, c_void_p, c_int64, c_int, c_void_p, c_void_p]
    L.stark_beam_topk_logits.restype = c_int
    L.stark_beam_topk_logits.argtypes = L.stark_beam_topk.argtypes
    L.stark_kv_append_reorg.restype = c_int
    L.stark_kv_append_reorg.argtypes = [P, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                        c_void_p, c_void_p]
    L.stark_workspace_bytes.restype = c_size_t
    L.stark_workspace_bytes.argtypes = [P, c_int, c_int, c_int]
    L.stark_suffix_bytes.restype = c_size_t
    L.stark_suffix_bytes.argtypes = [P]
    L.stark_anc_bytes.restype = c_size_t
    L.stark_anc_bytes.argtypes = [P]
    L.stark_version.restype = c_int
    L.stark_status_string.restype = ctypes.c_char_p
    L.stark_status_string.argtypes = [c_int]
    L.stark_last_cuda_error.restype = c_int
    _lib = L
    return L


def make_shape(B: int, Hq: int, Hkv: int, D: int, d: int, Wmax: int, dtype: torch.dtype,
               softmax_scale: float = 0.0) -> Shape:
    code = {torch.float32: STARK_F32, torch.bfloat16: STARK_BF16}[dtype]
    return Shape(B, Hq, Hkv, D, d, Wmax, code, softmax_scale)


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_contiguous(), "stark: tensors must be contiguous"
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _check(rc: int, where: str) -> None:
    if rc != 0:
        raise StarkError(rc, where)


# ---- the four calls (same names as the C ABI) ----------------------------------
def stark_prefix_attn_plan(shape: Shape, n_q: int, total_tokens: int, max_prefix_len: int) -> int:
    n = c_int(0)
    _check(lib().stark_prefix_attn_plan(byref(shape), n_q, total_tokens, max_prefix_len, byref(n)),
           "stark_prefix_attn_plan")
    return n.value


def alloc_partials(shape: Shape, n_q: int, n_splits: int, device) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    pm = torch.empty((n_splits, shape.B, n_q, shape.Hq), dtype=torch.float32, device=device)
    pl = torch.empty_like(pm)
    po = torch.empty((n_splits, shape.B, n_q, shape.Hq, shape.D), dtype=torch.float32, device=device)
    return pm, pl, po


def stark_prefix_attn(shape: Shape, q: torch.Tensor, n_q: int, k_prefix: torch.Tensor, v_prefix: torch.Tensor,
                      cu_seqlens: torch.Tensor, total_tokens: int, max_prefix_len: int, n_splits: int,
                      part_m: torch.Tensor, part_l: torch.Tensor, part_o: torch.Tensor,
                      ws: Optional[torch.Tensor] = None) -> None:
    _check(lib().stark_prefix_attn(byref(shape), _ptr(q), n_q, _ptr(k_prefix), _ptr(v_prefix), _ptr(cu_seqlens),
                                   total_tokens, max_prefix_len, n_splits, _ptr(part_m), _ptr(part_l),
                                   _ptr(part_o), _ptr(ws), ws.numel() * ws.element_size() if ws is not None else 0,
                                   _stream()), "stark_prefix_attn")


def stark_tree_attn_step(shape: Shape, q: torch.Tensor, n_q: int, level: int, k_suffix: Optional[torch.Tensor],
                         v_suffix: Optional[torch.Tensor], anc: Optional[torch.Tensor], part_m: torch.Tensor,
                         part_l: torch.Tensor, part_o: torch.Tensor, n_splits: int, out: torch.Tensor) -> None:
    _check(lib().stark_tree_attn_step(byref(shape), _ptr(q), n_q, level, _ptr(k_suffix), _ptr(v_suffix), _ptr(anc),
                                      _ptr(part_m), _ptr(part_l), _ptr(part_o), n_splits, _ptr(out), _stream()),
           "stark_tree_attn_step")


def stark_decode_attn(shape: Shape, q: torch.Tensor, n_q: int, level: int, k_prefix: torch.Tensor,
                      v_prefix: torch.Tensor, cu_seqlens: torch.Tensor, total_tokens: int, max_prefix_len: int,
                      k_suffix: Optional[torch.Tensor], v_suffix: Optional[torch.Tensor],
                      anc: Optional[torch.Tensor], out: torch.Tensor) -> None:
    """A1 + A2 fused (bf16): prefix attention, suffix chain, merge and normalise in one launch."""
    _check(lib().stark_decode_attn(byref(shape), _ptr(q), n_q, level, _ptr(k_prefix), _ptr(v_prefix),
                                   _ptr(cu_seqlens), total_tokens, max_prefix_len, _ptr(k_suffix), _ptr(v_suffix),
                                   _ptr(anc), _ptr(out), _stream()), "stark_decode_attn")


def stark_decode_step(shape: Shape, q: torch.Tensor, n_q: int, level: int, k_prefix: torch.Tensor,
                      v_prefix: torch.Tensor, cu_seqlens: torch.Tensor, total_tokens: int, max_prefix_len: int,
                      k_new: Optional[torch.Tensor], v_new: Optional[torch.Tensor], parent: Optional[torch.Tensor],
                      k_suffix: Optional[torch.Tensor], v_suffix: Optional[torch.Tensor],
                      anc: Optional[torch.Tensor], write_anc: bool, out: torch.Tensor) -> None:
    """A4 + A1 + A2 fused (bf16): append of the level's K/V and index rows inside the attention launch."""
    _check(lib().stark_decode_step(byref(shape), _ptr(q), n_q, level, _ptr(k_prefix), _ptr(v_prefix),
                                   _ptr(cu_seqlens), total_tokens, max_prefix_len, _ptr(k_new), _ptr(v_new),
                                   _ptr(parent), _ptr(k_suffix), _ptr(v_suffix), _ptr(anc), int(bool(write_anc)),
                                   _ptr(out), _stream()), "stark_decode_step")


def stark_beam_topk(logp: torch.Tensor, score: Optional[torch.Tensor], B: int, W_in: int, C: int, W_out: int,
                    out_score: torch.Tensor, out_parent: torch.Tensor, out_code: torch.Tensor,
                    ws: Optional[torch.Tensor] = None) -> None:
    _check(lib().stark_beam_topk(_ptr(logp), _ptr(score), B, W_in, C, W_out, _ptr(out_score), _ptr(out_parent),
                                 _ptr(out_code), _ptr(ws), ws.numel() * ws.element_size() if ws is not None else 0,
                                 _stream()), "stark_beam_topk")


#: size of the library's static top-k scratch array (include/stark.h: STARK_TOPK_STATIC_SCRATCH_BYTES)
TOPK_STATIC_SCRATCH_BYTES = 9 << 20


def stark_beam_topk_static(logp: torch.Tensor, score: Optional[torch.Tensor], B: int, W_in: int, C: int, W_out: int,
                           out_score: torch.Tensor, out_parent: torch.Tensor, out_code: torch.Tensor) -> None:
    """stark_beam_topk on the library's own static scratch array: allocates nothing, not safe for calls that
    overlap on the GPU, limited to problems whose workspace fits TOPK_STATIC_SCRATCH_BYTES."""
    rc = lib().stark_beam_topk_static(_ptr(logp), _ptr(score), B, W_in, C, W_out, _ptr(out_score), _ptr(out_parent),
                                      _ptr(out_code), _stream())
    if rc == -3:
        need = stark_workspace_bytes(make_shape(B, 1, 1, 64, 1, max(W_in, 1), torch.float32), CALL_BEAM_TOPK, W_in, C)
        raise StarkError(rc, f"stark_beam_topk_static (B={B}, W_in={W_in}, C={C} needs {need} bytes of scratch, the "
                             f"static array holds {TOPK_STATIC_SCRATCH_BYTES}: use stark_beam_topk with a workspace)")
    _check(rc, "stark_beam_topk_static")


def stark_logits_row_offset(logits: torch.Tensor, score: Optional[torch.Tensor], rows: int, C: int,
                            offset: torch.Tensor) -> None:
    """A3' first half: offset = fl32(score - fl32(logsumexp(logits))) per beam (reading R22)."""
    _check(lib().stark_logits_row_offset(_ptr(logits), _ptr(score), rows, C, _ptr(offset), _stream()),
           "stark_logits_row_offset")


def stark_beam_topk_logits(logits: torch.Tensor, score: Optional[torch.Tensor], B: int, W_in: int, C: int,
                           W_out: int, out_score: torch.Tensor, out_parent: torch.Tensor, out_code: torch.Tensor,
                           ws: Optional[torch.Tensor] = None) -> None:
    """A3': beam selection straight from raw logits (log-softmax normaliser folded into the beam score)."""
    _check(lib().stark_beam_topk_logits(_ptr(logits), _ptr(score), B, W_in, C, W_out, _ptr(out_score),
                                        _ptr(out_parent), _ptr(out_code), _ptr(ws),
                                        ws.numel() * ws.element_size() if ws is not None else 0, _stream()),
           "stark_beam_topk_logits")


def stark_kv_append_reorg(shape: Shape, level: int, n_new: int, k_new: torch.Tensor, v_new: torch.Tensor,
                          parent: Optional[torch.Tensor], k_suffix: torch.Tensor, v_suffix: torch.Tensor,
                          anc: Optional[torch.Tensor]) -> None:
    _check(lib().stark_kv_append_reorg(byref(shape), level, n_new, _ptr(k_new), _ptr(v_new), _ptr(parent),
                                       _ptr(k_suffix), _ptr(v_suffix), _ptr(anc), _stream()),
           "stark_kv_append_reorg")


def stark_workspace_bytes(shape: Shape, call: int, n_q: int, total_tokens: int) -> int:
    return int(lib().stark_workspace_bytes(byref(shape), call, n_q, total_tokens))


def alloc_suffix(shape: Shape, dtype: torch.dtype, device) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """k_suffix, v_suffix [d,B,Wmax,Hkv,D] and anc [2,B,Wmax,d], sized by the library's own helpers."""
    eb = 4 if dtype == torch.float32 else 2
    n = lib().stark_suffix_bytes(byref(shape)) // eb
    dims = (shape.d, shape.B, shape.Wmax, shape.Hkv, shape.D)
    assert n == shape.d * shape.B * shape.Wmax * shape.Hkv * shape.D
    ks = torch.zeros(dims, dtype=dtype, device=device)
    vs = torch.zeros(dims, dtype=dtype, device=device)
    na = lib().stark_anc_bytes(byref(shape)) // 4
    assert na == 2 * shape.B * shape.Wmax * shape.d
    anc = torch.zeros((2, shape.B, shape.Wmax, shape.d), dtype=torch.int32, device=device)
    return ks, vs, anc
