"""Thin ctypes binding of the prune entry points of libpici_b200 (include/pici_prune.h).
Argument marshalling only; no CPU path."""
from __future__ import annotations

import ctypes

import torch

from . import pici as _pk
from .pici import Pici, _check, _dev, _p, _stream

EXPORTS = ("pici_prune_sizes", "pici_prune_threshold", "pici_prune_compress")

_bound = False


def lib() -> ctypes.CDLL:
    global _bound
    L = _pk.lib()
    if not _bound:
        u64, p, ci, f = ctypes.c_uint64, ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.pici_prune_sizes.argtypes, L.pici_prune_sizes.restype = [u64, u64, p], ci
        L.pici_prune_threshold.argtypes, L.pici_prune_threshold.restype = [p, p, u64, f, p, u64, u64, p, p, u64, p], ci
        L.pici_prune_compress.argtypes, L.pici_prune_compress.restype = [p, p, u64, f, p, p, p, p, u64, p, u64, p], ci
        _bound = True
    return L


def workspace_bytes(n: int, m: int) -> int:
    ws = ctypes.c_uint64()
    _check(lib().pici_prune_sizes(n, m, ctypes.byref(ws)), "pici_prune_sizes")
    return int(ws.value)


def alloc_workspace(n: int, m: int, device="cuda", stream=None) -> torch.Tensor:
    ws = torch.empty(workspace_bytes(n, m), dtype=torch.uint8, device=device)
    _check(lib().pici_workspace_init(_p(ws), ws.numel(), _stream(stream)), "pici_workspace_init")
    return ws


def threshold(g: torch.Tensor, e: torch.Tensor, leak: float, sample: torch.Tensor, k: int, d_tau: torch.Tensor,
              ws: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(g, e, sample, d_tau, ws)
    assert g.dtype == e.dtype == torch.float32 and sample.dtype == torch.int32 and g.numel() == e.numel()
    _check(lib().pici_prune_threshold(_p(g), _p(e), g.numel(), leak, _p(sample), sample.numel(), k, _p(d_tau), _p(ws),
                                      ws.numel(), _stream(stream)), "pici_prune_threshold")
    return d_tau


def prune_compress(g: torch.Tensor, e_inout: torch.Tensor, leak: float, d_tau: torch.Tensor, out: Pici, ws: torch.Tensor,
                   stream=None) -> Pici:
    _dev(g, e_inout, d_tau, out.B, ws)
    assert g.dtype == e_inout.dtype == torch.float32 and g.numel() == e_inout.numel() == out.n
    _check(lib().pici_prune_compress(_p(g), _p(e_inout), out.n, leak, _p(d_tau), _p(out.B), _p(out.I), _p(out.A),
                                     out.A.numel(), _p(ws), ws.numel(), _stream(stream)), "pici_prune_compress")
    return out
