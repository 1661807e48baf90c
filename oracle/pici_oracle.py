"""TEST INFRASTRUCTURE - numpy front-end of oracle/pici_oracle.c (the plain CPU Pici oracle).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It shares no code with paper_2607_04676_b200/ and never imports it.
All arrays are numpy, host memory; values travel as raw bit patterns (uint32 for fp32, uint16
for bf16) so that "copied bit for bit" is literal.  See pici_oracle.c for the
citations of every operation.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pici_oracle.c")
_SO = os.path.join(_HERE, "libpici_oracle.so")

TILE = 4096


def build(force: bool = False) -> str:
    """gcc -O2, single translation unit, no OpenMP: the oracle is single-threaded by definition."""
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
            ("oracle_compress_f32", [p, u64, p, p, p], u64),
            ("oracle_compress_b16", [p, u64, p, p, p], u64),
            ("oracle_decompress_f32", [p, p, p, u64, p], u64),
            ("oracle_decompress_b16", [p, p, p, u64, p], u64),
            ("oracle_decompress_via_index_f32", [p, p, p, u64, p], u64),
            ("oracle_reduce_sd_f32", [p, p, p, u64, p], u64),
            ("oracle_reduce_ss_f32", [p, p, p, p, p, p, u64, p, p, p, p], u64),
            ("oracle_nnz_pici", [p, u64], u64),
            ("oracle_nnz_dense_f32", [p, u64], u64),
            ("oracle_nnz_dense_b16", [p, u64], u64),
            ("oracle_maybe_densify_f32", [p, p, p, u64, u64, p], ctypes.c_int),
            ("oracle_dense_add_f32", [p, p, u64, p], None),
            ("oracle_reduce_sd_b16", [p, p, p, u64, p], u64),
            ("oracle_dense_add_b16", [p, p, u64, p], None),
        ]:
            f = getattr(_lib, name)
            f.argtypes, f.restype = args, res
    return _lib


def _ptr(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def num_tiles(n: int) -> int:
    return (n + TILE - 1) // TILE


@dataclass
class Pici:
    """The three Pici components for an n-element dense buffer."""
    n: int
    dtype: str            # "f32" | "bf16"
    B: np.ndarray         # uint64[64*T]
    I: np.ndarray         # uint32[T+1]
    A: np.ndarray         # uint32[nnz] (f32 bits) | uint16[nnz] (bf16 bits)

    @property
    def nnz(self) -> int:
        return int(self.I[-1])

    def message_bytes(self) -> int:
        """Exact wire size: s*nnz + 8*64*T + 4*(T+1) (reading C9 #15; Eq. 4)."""
        return self.A.itemsize * self.nnz + self.B.nbytes + self.I.nbytes


def as_bits(dense: np.ndarray, dtype: str) -> np.ndarray:
    """View a dense host buffer as raw bit patterns.  Accepts float32, or uint16/uint32 bits."""
    if dtype == "f32":
        return np.ascontiguousarray(dense).view(np.uint32).reshape(-1)
    if dtype == "bf16":
        a = np.ascontiguousarray(dense)
        assert a.dtype.itemsize == 2
        return a.view(np.uint16).reshape(-1)
    raise ValueError(dtype)


def compress(dense_bits: np.ndarray, dtype: str = "f32") -> Pici:
    d = as_bits(dense_bits, dtype)
    n, T = d.size, num_tiles(d.size)
    B = np.zeros(64 * T, np.uint64)
    I = np.zeros(T + 1, np.uint32)
    A = np.empty(max(n, 1), d.dtype)
    fn = lib().oracle_compress_f32 if dtype == "f32" else lib().oracle_compress_b16
    nnz = fn(_ptr(d), n, _ptr(B), _ptr(I), _ptr(A))
    return Pici(n, dtype, B, I, A[:nnz].copy())


def decompress(x: Pici) -> np.ndarray:
    """Returns raw bits (uint32 / uint16) of the n-element dense buffer."""
    D = np.empty(x.n, x.A.dtype)
    fn = lib().oracle_decompress_f32 if x.dtype == "f32" else lib().oracle_decompress_b16
    used = fn(_ptr(x.B), _ptr(x.I), _ptr(x.A) if x.A.size else None, x.n, _ptr(D))
    assert used == x.A.size
    return D


def decompress_via_index(x: Pici) -> np.ndarray:
    assert x.dtype == "f32"
    D = np.empty(x.n, np.uint32)
    used = lib().oracle_decompress_via_index_f32(_ptr(x.B), _ptr(x.I),
                                                 _ptr(x.A) if x.A.size else None, x.n, _ptr(D))
    assert used == x.A.size
    return D


def reduce_sd(x: Pici, dense_inout: np.ndarray) -> None:
    """dense[i] = dense[i] + a_i on set bits, in place: float32, or bf16 bits as uint16 (add in fp32, round RNE)."""
    assert dense_inout.size == x.n
    if x.dtype == "f32":
        assert dense_inout.dtype == np.float32
        lib().oracle_reduce_sd_f32(_ptr(x.B), _ptr(x.I), _ptr(x.A) if x.A.size else None, x.n, _ptr(dense_inout))
    else:
        assert dense_inout.dtype == np.uint16
        lib().oracle_reduce_sd_b16(_ptr(x.B), _ptr(x.I), _ptr(x.A) if x.A.size else None, x.n, _ptr(dense_inout))


def reduce_ss(x: Pici, y: Pici) -> Pici:
    assert x.dtype == y.dtype == "f32" and x.n == y.n
    n, T = x.n, num_tiles(x.n)
    Bo = np.zeros(64 * T, np.uint64)
    Io = np.zeros(T + 1, np.uint32)
    Ao = np.empty(max(n, 1), np.uint32)
    scratch = np.empty(2 * max(n, 1), np.float32)
    nnz = lib().oracle_reduce_ss_f32(_ptr(x.B), _ptr(x.I), _ptr(x.A) if x.A.size else None,
                                     _ptr(y.B), _ptr(y.I), _ptr(y.A) if y.A.size else None,
                                     n, _ptr(Bo), _ptr(Io), _ptr(Ao), _ptr(scratch))
    return Pici(n, "f32", Bo, Io, Ao[:nnz].copy())


def nnz_pici(x: Pici) -> int:
    return int(lib().oracle_nnz_pici(_ptr(x.I), x.n))


def nnz_dense(dense_bits: np.ndarray, dtype: str = "f32") -> int:
    d = as_bits(dense_bits, dtype)
    fn = lib().oracle_nnz_dense_f32 if dtype == "f32" else lib().oracle_nnz_dense_b16
    return int(fn(_ptr(d), d.size))


def maybe_densify(x: Pici, nnz_switch: int, dense_out_bits: np.ndarray) -> bool:
    """switched = (nnz >= nnz_switch); dense_out is written only if switched."""
    assert x.dtype == "f32" and dense_out_bits.dtype == np.uint32 and dense_out_bits.size == x.n
    return bool(lib().oracle_maybe_densify_f32(_ptr(x.B), _ptr(x.I), _ptr(x.A) if x.A.size else None,
                                               x.n, int(nnz_switch), _ptr(dense_out_bits)))


def dense_add(recv: np.ndarray, local: np.ndarray) -> np.ndarray:
    """recv + local elementwise: float32, or bf16 bits as uint16 (add in fp32, round RNE)."""
    assert recv.dtype == local.dtype and recv.size == local.size and recv.dtype in (np.float32, np.uint16)
    out = np.empty_like(recv)
    fn = lib().oracle_dense_add_f32 if recv.dtype == np.float32 else lib().oracle_dense_add_b16
    fn(_ptr(recv), _ptr(local), recv.size, _ptr(out))
    return out
