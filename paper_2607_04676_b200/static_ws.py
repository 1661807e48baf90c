"""Thin ctypes binding of pici_compress_static (include/pici_static.h): pici_compress with the scan scratch inside the
library - no workspace argument, nothing allocated by the call.  Argument marshalling only; no CPU path."""
from __future__ import annotations

import ctypes

import torch

from . import pici as _pk
from .pici import Pici, _DT, _check, _dev, _p, _stream

EXPORTS = ("pici_static_limits", "pici_compress_static")

_bound = False


def lib() -> ctypes.CDLL:
    global _bound
    L = _pk.lib()
    if not _bound:
        u64, p, ci = ctypes.c_uint64, ctypes.c_void_p, ctypes.c_int
        L.pici_static_limits.argtypes, L.pici_static_limits.restype = [p, p], ci
        L.pici_compress_static.argtypes, L.pici_compress_static.restype = [p, u64, ci, p, p, p, u64, p], ci
        _bound = True
    return L


def limits() -> tuple[int, int]:
    """(largest n accepted, bytes of the library's static scratch array)"""
    n, b = ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().pici_static_limits(ctypes.byref(n), ctypes.byref(b)), "pici_static_limits")
    return int(n.value), int(b.value)


def compress(dense: torch.Tensor, out: Pici, stream=None) -> Pici:
    """dense -> out (B, I, A) on the device; calls that may overlap on the GPU race on the shared scratch."""
    _dev(dense, out.B, out.I, out.A)
    n = dense.numel()
    assert n == out.n and _DT[dense.dtype] == out.dtype and dense.is_contiguous()
    _check(lib().pici_compress_static(_p(dense), n, out.dtype, _p(out.B), _p(out.I), _p(out.A), out.A.numel(),
                                      _stream(stream)), f"pici_compress_static (n <= {limits()[0]})")
    return out
