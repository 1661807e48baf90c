"""TEST INFRASTRUCTURE - numpy front-end of oracle/prune_oracle.c (sampled top-k pruning with leaky error feedback,
PAPER.md:315-317).  Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "prune_oracle.c")
_SO = os.path.join(_HERE, "libprune_oracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fno-fast-math", "-ffp-contract=off",
                               "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        u64, p, f = ctypes.c_uint64, ctypes.c_void_p, ctypes.c_float
        _lib.oracle_prune_threshold_f32.argtypes = [p, p, u64, f, p, u64, u64, p]
        _lib.oracle_prune_threshold_f32.restype = f
        _lib.oracle_prune_ef_f32.argtypes = [p, p, u64, f, f, p, p]
        _lib.oracle_prune_ef_f32.restype = u64
    return _lib


def _ptr(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def threshold(g: np.ndarray, e: np.ndarray, leak: float, sample: np.ndarray, k: int) -> np.float32:
    assert g.dtype == e.dtype == np.float32 and sample.dtype == np.uint32 and 1 <= k <= sample.size
    scratch = np.empty(sample.size, np.float32)
    return np.float32(lib().oracle_prune_threshold_f32(_ptr(g), _ptr(e), g.size, leak, _ptr(sample), sample.size, k,
                                                       _ptr(scratch)))


def prune_ef(g: np.ndarray, e: np.ndarray, leak: float, tau) -> tuple[np.ndarray, np.ndarray, int]:
    """(sent, e', number sent)"""
    sent, e_out = np.empty_like(g), np.empty_like(g)
    c = lib().oracle_prune_ef_f32(_ptr(g), _ptr(e), g.size, leak, float(tau), _ptr(sent), _ptr(e_out))
    return sent, e_out, int(c)
