"""TEST INFRASTRUCTURE - numpy front-end of oracle/coo_oracle.c (the plain CPU oracle of the paper's COO
variant).  Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import
this; it shares no code with paper_2607_04676_b200/ and never imports it.  Values travel as raw fp32 bits."""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "coo_oracle.c")
_SO = os.path.join(_HERE, "libcoo_oracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fno-fast-math", "-ffp-contract=off",
                               "-fPIC", "-shared", "-o", _SO, _SRC])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        u64, p = ctypes.c_uint64, ctypes.c_void_p
        for name, args, res in [
            ("oracle_coo_compress_f32", [p, u64, p, p], u64),
            ("oracle_coo_decompress_f32", [p, p, u64, u64, p], None),
            ("oracle_coo_reduce_sd_f32", [p, p, u64, p], None),
            ("oracle_coo_reduce_ss_f32", [p, p, u64, p, p, u64, u64, p, p, p], u64),
        ]:
            f = getattr(_lib, name)
            f.argtypes, f.restype = args, res
    return _lib


def _ptr(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p) if a.size else None


@dataclass
class Coo:
    """Flat-index COO of an n-element fp32 buffer: ascending idx, value bits in the same order."""
    n: int
    idx: np.ndarray       # uint32[nnz]
    val: np.ndarray       # uint32[nnz] (fp32 bits)

    @property
    def nnz(self) -> int:
        return int(self.idx.size)

    def message_bytes(self) -> int:
        """32-bit index + 32-bit value per nonzero."""
        return 8 * self.nnz


def _bits(dense: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(dense).view(np.uint32).reshape(-1)


def compress(dense_bits: np.ndarray) -> Coo:
    d = _bits(dense_bits)
    idx = np.empty(max(d.size, 1), np.uint32)
    val = np.empty(max(d.size, 1), np.uint32)
    k = lib().oracle_coo_compress_f32(_ptr(d), d.size, _ptr(idx), _ptr(val))
    return Coo(d.size, idx[:k].copy(), val[:k].copy())


def decompress(x: Coo) -> np.ndarray:
    D = np.empty(x.n, np.uint32)
    lib().oracle_coo_decompress_f32(_ptr(x.idx), _ptr(x.val), x.nnz, x.n, _ptr(D))
    return D


def reduce_sd(x: Coo, dense_inout_f32: np.ndarray) -> None:
    assert dense_inout_f32.dtype == np.float32 and dense_inout_f32.size == x.n
    lib().oracle_coo_reduce_sd_f32(_ptr(x.idx), _ptr(x.val), x.nnz, _ptr(dense_inout_f32))


def reduce_ss(x: Coo, y: Coo) -> Coo:
    assert x.n == y.n
    n = x.n
    io = np.empty(max(n, 1), np.uint32)
    vo = np.empty(max(n, 1), np.uint32)
    scratch = np.empty(2 * max(n, 1), np.float32)
    k = lib().oracle_coo_reduce_ss_f32(_ptr(x.idx), _ptr(x.val), x.nnz, _ptr(y.idx), _ptr(y.val), y.nnz, n,
                                       _ptr(io), _ptr(vo), _ptr(scratch))
    return Coo(n, io[:k].copy(), vo[:k].copy())
