"""Thin ctypes binding of libpici_b200 (include/pici.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams.

There is NO CPU fallback: importing works without a GPU (so the symbol table can be checked), but
every compute call raises unless the library is loaded and the tensors live on a CUDA device.
Function names mirror the C ABI (pici_compress -> compress, ...).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

from . import build as _build

F32, BF16 = 0, 1
FMT_PICI, FMT_DENSE = 0, 1
TILE = 4096

_DT = {torch.float32: F32, torch.bfloat16: BF16}

EXPORTS = (
    "pici_version", "pici_strerror", "pici_sizes", "pici_workspace_init", "pici_compress", "pici_decompress", "pici_reduce_sd",
    "pici_reduce_ss", "pici_nnz", "pici_nnz_dense", "pici_maybe_densify", "pici_compress_gated",
    "pici_reduce_ss_gated", "pici_maybe_densify_gated", "pici_dense_add_gated", "pici_reduce_sd_out_gated",
    "pici_decompress_gated", "pici_dense_copy_gated", "pici_compress_host", "pici_decompress_host",
    "pici_probe_random_rmw", "pici_ring_arena_bytes", "pici_ring_layout", "pici_ring_reduce_scatter", "pici_ring_all_gather", "pici_ring_all_reduce",
)

_lib = None


class PiciError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {lib().pici_strerror(code).decode()} ({code})")


def lib() -> ctypes.CDLL:
    """Load (building first if stale) the in-tree shared library.  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        so = _build.SO
        if os.environ.get("PICI_NO_BUILD") != "1":
            so = _build.build()
        if not os.path.exists(so):
            raise RuntimeError(f"{so} is missing: run `python -m paper_2607_04676_b200.build`")
        L = ctypes.CDLL(so)
        u64, p, i32, ci = ctypes.c_uint64, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int
        sig = {
            "pici_version": ([], ci),
            "pici_strerror": ([ci], ctypes.c_char_p),
            "pici_sizes": ([u64, ci, p, p, p, p], ci),
            "pici_workspace_init": ([p, u64, p], ci),
            "pici_compress": ([p, u64, ci, p, p, p, u64, p, u64, p], ci),
            "pici_compress_gated": ([p, u64, ci, p, p, p, u64, p, u64, p, i32, p], ci),
            "pici_decompress": ([p, p, p, u64, ci, p, p], ci),
            "pici_decompress_gated": ([p, p, p, u64, ci, p, p, i32, p], ci),
            "pici_reduce_sd": ([p, p, p, u64, ci, p, p], ci),
            "pici_reduce_sd_out_gated": ([p, p, p, p, u64, ci, p, p, i32, p], ci),
            "pici_reduce_ss": ([p, p, p, p, p, p, u64, ci, p, p, p, u64, p, u64, p], ci),
            "pici_reduce_ss_gated": ([p, p, p, p, p, p, u64, ci, p, p, p, u64, p, u64, p, i32, p], ci),
            "pici_nnz": ([p, u64, p, p], ci),
            "pici_nnz_dense": ([p, u64, ci, p, p, u64, p], ci),
            "pici_maybe_densify": ([p, p, p, u64, ci, u64, p, p, p], ci),
            "pici_maybe_densify_gated": ([p, p, p, u64, ci, u64, p, p, p, i32, p], ci),
            "pici_dense_add_gated": ([p, p, u64, ci, p, p, p, i32, p], ci),
            "pici_dense_copy_gated": ([p, p, u64, ci, p, i32, p], ci),
            "pici_compress_host": ([p, u64, ci, p, p, p, p, p, p, p, p, p, u64, p], ci),
            "pici_decompress_host": ([p, p, p, u64, u64, ci, p, p, p, p, p, p], ci),
            "pici_probe_random_rmw": ([p, u64, p, u64, p], ci),
            "pici_ring_arena_bytes": ([p, p], ci),
            "pici_ring_layout": ([p, p], ci),
            "pici_ring_reduce_scatter": ([p, p, p, p, u64, p, p], ci),
            "pici_ring_all_gather": ([p, p, p, p, u64, p, p], ci),
            "pici_ring_all_reduce": ([p, p, p, p, u64, p, p], ci),
        }
        for name, (args, res) in sig.items():
            f = getattr(L, name)
            f.argtypes, f.restype = args, res
        _lib = L
    return _lib


def version() -> int:
    return lib().pici_version()


def num_tiles(n: int) -> int:
    return (n + TILE - 1) // TILE


def sizes(n: int, dtype: int = F32) -> tuple[int, int, int, int]:
    """(bitvec_words, index_entries, values_capacity, workspace_bytes) for an n-element buffer."""
    out = [ctypes.c_uint64() for _ in range(4)]
    rc = lib().pici_sizes(n, dtype, *[ctypes.byref(o) for o in out])
    if rc:
        raise PiciError(rc, "pici_sizes")
    return tuple(int(o.value) for o in out)


def _stream(stream=None) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream if hasattr(s, "cuda_stream") else int(s)


def _p(t) -> int | None:
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _dev(*ts):
    for t in ts:
        if t is not None and not isinstance(t, int) and not t.is_cuda:
            raise RuntimeError("pici: tensors must live on a CUDA device (there is no CPU path)")


def _check(rc: int, where: str):
    if rc:
        raise PiciError(rc, where)


@dataclass
class Pici:
    """Device-side Pici object for an n-element buffer: the caller-owned B, I, A."""
    n: int
    dtype: int                 # F32 | BF16
    B: torch.Tensor            # int64[64*T] (bit pattern of uint64)
    I: torch.Tensor            # int32[T+1]  (bit pattern of uint32)
    A: torch.Tensor            # float32[n] | bfloat16[n]: capacity n, first nnz valid

    @property
    def T(self) -> int:
        return num_tiles(self.n)

    def nnz_host(self) -> int:
        """Reads I[T] back (synchronises): for reporting and tests, never inside timed regions."""
        return int(self.I[self.T].item()) & 0xFFFFFFFF

    def to_host(self):
        """(B uint64[64T], I uint32[T+1], A raw bits[nnz]) as numpy arrays."""
        import numpy as np
        nnz = self.nnz_host()
        B = self.B.cpu().numpy().view(np.uint64)
        I = self.I.cpu().numpy().view(np.uint32)
        a = self.A[:nnz].cpu()
        A = a.view(torch.int32).numpy().view(np.uint32) if self.dtype == F32 else a.view(torch.int16).numpy().view(np.uint16)
        return B, I, A


def alloc_pici(n: int, dtype: int = F32, device="cuda") -> Pici:
    words, entries, cap, _ = sizes(n, dtype)
    tdt = torch.float32 if dtype == F32 else torch.bfloat16
    return Pici(n, dtype,
                torch.empty(max(words, 2), dtype=torch.int64, device=device),
                torch.empty(entries, dtype=torch.int32, device=device),
                torch.empty(max(cap, 8), dtype=tdt, device=device))


def alloc_workspace(n: int, device="cuda", stream=None) -> torch.Tensor:
    """Scratch for compress / reduce_ss of up to n elements, cleared once (pici_workspace_init)."""
    ws = torch.empty(max(sizes(n, F32)[3], 16), dtype=torch.uint8, device=device)
    _check(lib().pici_workspace_init(_p(ws), ws.numel(), _stream(stream)), "pici_workspace_init")
    return ws


def compress(dense: torch.Tensor, out: Pici, ws: torch.Tensor, stream=None, gate=None, gate_value: int = 0) -> Pici:
    _dev(dense, out.B, out.I, out.A, ws, gate)
    n = dense.numel()
    assert n == out.n and _DT[dense.dtype] == out.dtype and dense.is_contiguous()
    if gate is None:
        rc = lib().pici_compress(_p(dense), n, out.dtype, _p(out.B), _p(out.I), _p(out.A), out.A.numel(),
                                 _p(ws), ws.numel(), _stream(stream))
    else:
        rc = lib().pici_compress_gated(_p(dense), n, out.dtype, _p(out.B), _p(out.I), _p(out.A), out.A.numel(),
                                       _p(ws), ws.numel(), _p(gate), gate_value, _stream(stream))
    _check(rc, "pici_compress")
    return out


def decompress(x: Pici, dense_out: torch.Tensor, stream=None, gate=None, gate_value: int = 0) -> torch.Tensor:
    _dev(x.B, x.I, x.A, dense_out, gate)
    assert dense_out.numel() == x.n and _DT[dense_out.dtype] == x.dtype and dense_out.is_contiguous()
    if gate is None:
        rc = lib().pici_decompress(_p(x.B), _p(x.I), _p(x.A), x.n, x.dtype, _p(dense_out), _stream(stream))
    else:
        rc = lib().pici_decompress_gated(_p(x.B), _p(x.I), _p(x.A), x.n, x.dtype, _p(dense_out), _p(gate),
                                         gate_value, _stream(stream))
    _check(rc, "pici_decompress")
    return dense_out


def reduce_sd(x: Pici, dense_inout: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(x.B, x.I, x.A, dense_inout)
    assert dense_inout.numel() == x.n and dense_inout.is_contiguous()
    _check(lib().pici_reduce_sd(_p(x.B), _p(x.I), _p(x.A), x.n, _DT[dense_inout.dtype], _p(dense_inout),
                                _stream(stream)), "pici_reduce_sd")
    return dense_inout


def reduce_sd_out(x: Pici, local: torch.Tensor, out: torch.Tensor, stream=None, gate=None, gate_value: int = 0):
    _dev(x.B, x.I, x.A, local, out, gate)
    assert local.numel() == x.n == out.numel() and local.is_contiguous() and out.is_contiguous()
    _check(lib().pici_reduce_sd_out_gated(_p(x.B), _p(x.I), _p(x.A), _p(local), x.n, _DT[out.dtype], _p(out),
                                          _p(gate), gate_value, _stream(stream)), "pici_reduce_sd_out_gated")
    return out


def reduce_ss(x: Pici, y: Pici, out: Pici, ws: torch.Tensor, stream=None, gate=None, gate_value: int = 0) -> Pici:
    _dev(x.B, y.B, out.B, ws, gate)
    assert x.n == y.n == out.n
    args = (_p(x.B), _p(x.I), _p(x.A), _p(y.B), _p(y.I), _p(y.A), x.n, out.dtype, _p(out.B), _p(out.I), _p(out.A),
            out.A.numel(), _p(ws), ws.numel())
    if gate is None:
        rc = lib().pici_reduce_ss(*args, _stream(stream))
    else:
        rc = lib().pici_reduce_ss_gated(*args, _p(gate), gate_value, _stream(stream))
    _check(rc, "pici_reduce_ss")
    return out


def nnz(x: Pici, d_nnz: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(x.I, d_nnz)
    _check(lib().pici_nnz(_p(x.I), x.n, _p(d_nnz), _stream(stream)), "pici_nnz")
    return d_nnz


def nnz_dense(dense: torch.Tensor, d_nnz: torch.Tensor, stream=None) -> torch.Tensor:
    _dev(dense, d_nnz)
    assert dense.is_contiguous()
    _check(lib().pici_nnz_dense(_p(dense), dense.numel(), _DT[dense.dtype], _p(d_nnz), None, 0, _stream(stream)),
           "pici_nnz_dense")
    return d_nnz


def maybe_densify(x: Pici, nnz_switch: int, dense_out: torch.Tensor | None, d_switched: torch.Tensor, stream=None,
                  gate=None, gate_value: int = 0) -> torch.Tensor:
    _dev(x.B, x.I, x.A, dense_out, d_switched, gate)
    assert dense_out is None or (dense_out.numel() == x.n and dense_out.is_contiguous())
    if gate is None:
        rc = lib().pici_maybe_densify(_p(x.B), _p(x.I), _p(x.A), x.n, x.dtype, int(nnz_switch), _p(dense_out),
                                      _p(d_switched), _stream(stream))
    else:
        rc = lib().pici_maybe_densify_gated(_p(x.B), _p(x.I), _p(x.A), x.n, x.dtype, int(nnz_switch), _p(dense_out),
                                            _p(d_switched), _p(gate), gate_value, _stream(stream))
    _check(rc, "pici_maybe_densify")
    return d_switched


def dense_add(recv: torch.Tensor, local: torch.Tensor, out: torch.Tensor, d_fmt_out=None, stream=None, gate=None,
              gate_value: int = 0) -> torch.Tensor:
    _dev(recv, local, out, d_fmt_out, gate)
    assert recv.numel() == local.numel() == out.numel()
    _check(lib().pici_dense_add_gated(_p(recv), _p(local), out.numel(), _DT[out.dtype], _p(out), _p(d_fmt_out),
                                      _p(gate), gate_value, _stream(stream)), "pici_dense_add_gated")
    return out


def dense_copy(src: torch.Tensor, dst: torch.Tensor, stream=None, gate=None, gate_value: int = 0) -> torch.Tensor:
    _dev(src, dst, gate)
    assert src.numel() == dst.numel() and src.dtype == dst.dtype and src.is_contiguous() and dst.is_contiguous()
    _check(lib().pici_dense_copy_gated(_p(src), _p(dst), dst.numel(), _DT[dst.dtype], _p(gate), gate_value,
                                       _stream(stream)), "pici_dense_copy_gated")
    return dst


def probe_random_rmw(idx: torch.Tensor, dense_inout: torch.Tensor, stream=None) -> torch.Tensor:
    """Measurement aid (pici_probe_random_rmw): dense_inout[idx[i]] += 1 for distinct int32 indices idx."""
    _dev(idx, dense_inout)
    assert idx.dtype == torch.int32 and idx.is_contiguous() and dense_inout.dtype == torch.float32
    _check(lib().pici_probe_random_rmw(_p(idx), idx.numel(), _p(dense_inout), dense_inout.numel(), _stream(stream)),
           "pici_probe_random_rmw")
    return dense_inout


@dataclass
class HostPici:
    """Host-side (pinned) B, I, A buffers for the end-to-end calls."""
    n: int
    dtype: int
    B: torch.Tensor
    I: torch.Tensor
    A: torch.Tensor
    nnz: int = 0


def alloc_host_pici(n: int, dtype: int = F32, pin: bool = True) -> HostPici:
    words, entries, cap, _ = sizes(n, dtype)
    tdt = torch.float32 if dtype == F32 else torch.bfloat16
    mk = lambda k, d: torch.empty(k, dtype=d, pin_memory=pin)
    return HostPici(n, dtype, mk(max(words, 2), torch.int64), mk(entries, torch.int32), mk(max(cap, 8), tdt))


def compress_host(h_dense: torch.Tensor, h_out: HostPici, d_dense: torch.Tensor, d_scratch: Pici, ws: torch.Tensor,
                  stream=None) -> HostPici:
    """End-to-end: HOST dense buffer -> HOST (B, I, A).  Copies run inside the call; it synchronises."""
    _dev(d_dense, d_scratch.B, ws)
    assert not h_dense.is_cuda and h_dense.is_contiguous() and h_dense.numel() == h_out.n == d_scratch.n
    nnz_out = ctypes.c_uint64()
    _check(lib().pici_compress_host(_p(h_dense), h_out.n, h_out.dtype, _p(h_out.B), _p(h_out.I), _p(h_out.A),
                                    ctypes.addressof(nnz_out), _p(d_dense), _p(d_scratch.B), _p(d_scratch.I),
                                    _p(d_scratch.A), _p(ws), ws.numel(), _stream(stream)), "pici_compress_host")
    h_out.nnz = int(nnz_out.value)
    return h_out


def decompress_host(h_x: HostPici, h_dense_out: torch.Tensor, d_scratch: Pici, d_dense: torch.Tensor,
                    stream=None) -> torch.Tensor:
    """End-to-end: HOST (B, I, A[nnz]) -> HOST dense buffer."""
    _dev(d_dense, d_scratch.B)
    assert not h_dense_out.is_cuda and h_dense_out.numel() == h_x.n == d_scratch.n
    _check(lib().pici_decompress_host(_p(h_x.B), _p(h_x.I), _p(h_x.A), h_x.nnz, h_x.n, h_x.dtype, _p(h_dense_out),
                                      _p(d_scratch.B), _p(d_scratch.I), _p(d_scratch.A), _p(d_dense),
                                      _stream(stream)), "pici_decompress_host")
    return h_dense_out
