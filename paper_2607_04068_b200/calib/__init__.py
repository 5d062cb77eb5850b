"""Loader of libstark_calib.so (calib/stark_calib.h): the launch-floor / cold-stream probes of
`bench.py --calibrate`.  Measurement aid, not part of the product library."""
from __future__ import annotations

import ctypes
import os
from ctypes import c_int, c_size_t, c_void_p

import torch

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libstark_calib.so")
EXPORTS = ("stark_calib_empty", "stark_calib_stream_read")
_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2607_04068_b200.build`")
        L = ctypes.CDLL(LIB_PATH)
        L.stark_calib_empty.restype = c_int
        L.stark_calib_empty.argtypes = [c_void_p]
        L.stark_calib_stream_read.restype = c_int
        L.stark_calib_stream_read.argtypes = [c_void_p, c_size_t, c_void_p, c_void_p]
        _lib = L
    return _lib


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def stark_calib_empty() -> None:
    rc = lib().stark_calib_empty(_stream())
    if rc:
        raise RuntimeError(f"stark_calib_empty: {rc}")


def stark_calib_stream_read(src: torch.Tensor, nbytes: int, sink: torch.Tensor) -> None:
    rc = lib().stark_calib_stream_read(src.data_ptr(), nbytes, sink.data_ptr(), _stream())
    if rc:
        raise RuntimeError(f"stark_calib_stream_read: {rc}")
