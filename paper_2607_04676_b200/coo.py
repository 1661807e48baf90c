"""Thin ctypes binding of the COO entry points of libpici_b200 (include/pici_coo.h).
Argument marshalling only; no CPU path.  Function names mirror the C ABI (pici_coo_compress -> compress, ...)."""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

import torch

from . import pici as _pk
from .pici import _check, _dev, _p, _stream

EXPORTS = ("pici_coo_sizes", "pici_coo_compress", "pici_coo_decompress", "pici_coo_reduce_sd", "pici_coo_reduce_ss")

_bound = False


def lib() -> ctypes.CDLL:
    global _bound
    L = _pk.lib()
    if not _bound:
        u64, p, ci = ctypes.c_uint64, ctypes.c_void_p, ctypes.c_int
        sig = {
            "pici_coo_sizes": ([u64, p, p], ci),
            "pici_coo_compress": ([p, u64, p, p, u64, p, p, u64, p], ci),
            "pici_coo_decompress": ([p, p, p, u64, p, p, u64, p], ci),
            "pici_coo_reduce_sd": ([p, p, p, u64, p, p], ci),
            "pici_coo_reduce_ss": ([p, p, p, p, p, p, u64, p, p, u64, p, p, u64, p], ci),
        }
        for name, (args, res) in sig.items():
            f = getattr(L, name)
            f.argtypes, f.restype = args, res
        _bound = True
    return L


def sizes(n: int) -> tuple[int, int]:
    """(capacity in elements, workspace bytes) for an n-element buffer."""
    cap, ws = ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().pici_coo_sizes(n, ctypes.byref(cap), ctypes.byref(ws)), "pici_coo_sizes")
    return int(cap.value), int(ws.value)


@dataclass
class Coo:
    """Device-side COO object of an n-element fp32 buffer: caller-owned idx, val (capacity n) and the nnz word."""
    n: int
    idx: torch.Tensor      # int32[n]   (bit pattern of uint32), first nnz valid, ascending
    val: torch.Tensor      # float32[n], first nnz valid
    nnz: torch.Tensor      # int32[1] on the device

    def nnz_host(self) -> int:
        return int(self.nnz.item()) & 0xFFFFFFFF

    def to_host(self):
        """(idx uint32[nnz], val raw bits uint32[nnz]) as numpy arrays (synchronises)."""
        import numpy as np
        k = self.nnz_host()
        return (self.idx[:k].cpu().numpy().view(np.uint32), self.val[:k].cpu().view(torch.int32).numpy().view(np.uint32))


def alloc_coo(n: int, device="cuda") -> Coo:
    cap, _ = sizes(n)
    return Coo(n, torch.empty(max(cap, 4), dtype=torch.int32, device=device),
               torch.empty(max(cap, 4), dtype=torch.float32, device=device),
               torch.zeros(1, dtype=torch.int32, device=device))


def alloc_workspace(n: int, device="cuda", stream=None) -> torch.Tensor:
    ws = torch.empty(max(sizes(n)[1], 16), dtype=torch.uint8, device=device)
    _check(lib().pici_workspace_init(_p(ws), ws.numel(), _stream(stream)), "pici_workspace_init")
    return ws


def compress(dense: torch.Tensor, out: Coo, ws: torch.Tensor, stream=None) -> Coo:
    _dev(dense, out.idx, out.val, out.nnz, ws)
    assert dense.dtype == torch.float32 and dense.is_contiguous() and dense.numel() == out.n
    _check(lib().pici_coo_compress(_p(dense), out.n, _p(out.idx), _p(out.val), out.idx.numel(), _p(out.nnz), _p(ws),
                                   ws.numel(), _stream(stream)), "pici_coo_compress")
    return out


def decompress(x: Coo, dense_out: torch.Tensor, ws: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(x.idx, x.val, x.nnz, dense_out, ws)
    assert dense_out.dtype == torch.float32 and dense_out.is_contiguous() and dense_out.numel() == x.n
    _check(lib().pici_coo_decompress(_p(x.idx), _p(x.val), _p(x.nnz), x.n, _p(dense_out), _p(ws), ws.numel(),
                                     _stream(stream)), "pici_coo_decompress")
    return dense_out


def reduce_sd(x: Coo, dense_inout: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(x.idx, x.val, x.nnz, dense_inout)
    assert dense_inout.dtype == torch.float32 and dense_inout.is_contiguous() and dense_inout.numel() == x.n
    _check(lib().pici_coo_reduce_sd(_p(x.idx), _p(x.val), _p(x.nnz), x.n, _p(dense_inout), _stream(stream)),
           "pici_coo_reduce_sd")
    return dense_inout


def reduce_ss(x: Coo, y: Coo, out: Coo, ws: torch.Tensor, stream=None) -> Coo:
    _dev(x.idx, y.idx, out.idx, ws)
    assert x.n == y.n == out.n
    _check(lib().pici_coo_reduce_ss(_p(x.idx), _p(x.val), _p(x.nnz), _p(y.idx), _p(y.val), _p(y.nnz), x.n, _p(out.idx),
                                    _p(out.val), out.idx.numel(), _p(out.nnz), _p(ws), ws.numel(), _stream(stream)),
           "pici_coo_reduce_ss")
    return out
