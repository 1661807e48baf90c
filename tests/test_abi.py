"""CPU-side checks of the C-ABI boundary (no GPU, no compute): libpici_b200.so builds for sm_100a and loads,
exports every function include/pici.h declares, reports the sizes the format fixes, and
rejects bad arguments with error codes before any CUDA call is made (include/pici.h "Errors").
"""
import ctypes
import os
import re

import pytest

from paper_2607_04676_b200 import coo, pici, prune, static_ws

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared() -> list[str]:
    """Function names declared between the extern "C" braces of include/*.h."""
    names = set()
    for h in sorted(os.listdir(os.path.join(ROOT, "include"))):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(pici_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_every_declared_symbol_is_exported_and_bound():
    names = _declared()
    assert {"pici_compress", "pici_decompress", "pici_reduce_ss", "pici_reduce_sd", "pici_nnz",
            "pici_maybe_densify"} <= set(names)              # the six names north_star fixes
    lib = pici.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/pici.h but not exported"
    assert set(names) == set(pici.EXPORTS) | set(coo.EXPORTS) | set(prune.EXPORTS) | set(static_ws.EXPORTS), "the Python binding and the header disagree on the entry points"
    assert lib.pici_version() == 100
    coo.lib()                                                # binds the pici_coo_* signatures
    L = prune.lib()
    INVALID, ALIGN, CAPACITY, WORKSPACE = -1, -3, -4, -5
    n, m = 8192, 8
    ws = prune.workspace_bytes(n, m)
    assert ws >= pici.sizes(n)[3] + 4 * m and ws % 16 == 0
    a, b, c, w = 0x10000, 0x20000, 0x30000, 0x40000
    assert L.pici_prune_threshold(a, b, n, 1.0, c, m, 0, w, w + 0x1000, ws, None) == INVALID        # k >= 1
    assert L.pici_prune_threshold(a, b, n, 1.0, c, m, m + 1, w, w + 0x1000, ws, None) == INVALID    # k <= m
    assert L.pici_prune_threshold(a, b, n, 1.0, c, m, 1, w, w + 0x1000, ws - 16, None) == WORKSPACE
    assert L.pici_prune_threshold(a + 4, b, n, 1.0, c, m, 1, w, w + 0x1000, ws, None) == ALIGN
    assert L.pici_prune_compress(a, a, n, 1.0, w, b, c, c + 0x1000, n, w + 0x1000, ws, None) == INVALID   # g must not be e
    assert L.pici_prune_compress(a, b, n, 1.0, w, c, c + 0x1000, c + 0x2000, n - 1, w + 0x1000, ws, None) == CAPACITY


def test_coo_calls_validate_before_any_cuda_call():
    """include/pici_coo.h: sizes follow the format (capacity n: one index per nonzero in the worst case,
    PAPER.md:275) and bad arguments are rejected on the host."""
    lib = coo.lib()
    INVALID, ALIGN, CAPACITY, WORKSPACE = -1, -3, -4, -5
    n = 8192
    cap, ws = coo.sizes(n)
    assert cap == n and ws % 16 == 0 and ws > pici.sizes(n)[3]
    assert lib.pici_coo_sizes(1 << 32, None, None) == INVALID
    a, b, c, w = 0x10000, 0x20000, 0x30000, 0x40000
    C = lib.pici_coo_compress
    assert C(None, n, b, c, n, w, w + 0x1000, ws, None) == INVALID
    assert C(a, n, b, c, n, None, w + 0x1000, ws, None) == INVALID
    assert C(a, n, b + 4, c, n, w, w + 0x1000, ws, None) == ALIGN
    assert C(a, n, b, c, n - 1, w, w + 0x1000, ws, None) == CAPACITY
    assert C(a, n, b, c, n, w, w + 0x1000, ws - 1, None) == WORKSPACE
    assert lib.pici_coo_decompress(b, c, w, n, None, w + 0x1000, ws, None) == INVALID
    assert lib.pici_coo_reduce_sd(b, c, w, n, a + 8, None) == ALIGN
    S = lib.pici_coo_reduce_ss
    assert S(a, a + 0x1000, w, b, b + 0x1000, w + 16, n, a, c + 0x1000, n, w + 32, w + 0x1000, ws, None) == INVALID   # io == ix
    assert S(a, a + 0x1000, w, b, b + 0x1000, w + 16, n, c, c + 0x1000, n - 1, w + 32, w + 0x1000, ws, None) == CAPACITY


def test_oracle_and_product_share_no_code():
    """Neither side imports, includes or links the other (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_2607_04676_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(from|import)\s+\S*oracle", text, flags=re.M), f"{f} imports the oracle"
                assert not re.search(r"#\s*include\s*[<\"].*oracle", text), f"{f} includes the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2607_04676_b200", text, flags=re.M), f
            assert not re.search(r"#\s*include\s*[<\"].*(csrc|pici\.h|pici_common)", text), f


@pytest.mark.parametrize("n", [0, 1, 4095, 4096, 4097, 8192, 1 << 20, (1 << 28), (1 << 32) - 1])
@pytest.mark.parametrize("dtype", [pici.F32, pici.BF16])
def test_sizes_follow_the_format(n, dtype):
    lib = pici.lib()
    bw, ie, cap, ws = (ctypes.c_uint64() for _ in range(4))
    assert lib.pici_sizes(n, dtype, ctypes.byref(bw), ctypes.byref(ie), ctypes.byref(cap), ctypes.byref(ws)) == 0
    T = (n + 4095) // 4096
    assert bw.value == 64 * T            # one 64-bit word per column of every 64x64 tile
    assert ie.value == T + 1             # exclusive prefix per tile + total nnz
    assert cap.value == n                # worst case: every element stored
    assert ws.value >= 8 * T and ws.value % 16 == 0
    if n and n % 4096 == 0:              # metadata / fp32 dense = (1/8 + 4/4096) / 4 + 4 bytes
        assert 8 * bw.value + 4 * ie.value == n // 8 + n // 1024 + 4
    assert lib.pici_sizes(n, dtype, None, None, None, None) == 0          # every output is optional


def test_sizes_and_calls_reject_bad_arguments_without_touching_the_device():
    lib = pici.lib()
    INVALID, DTYPE, ALIGN, CAPACITY, WORKSPACE = -1, -2, -3, -4, -5
    assert lib.pici_sizes(1 << 32, pici.F32, None, None, None, None) == INVALID      # n < 2^32 (32-bit I)
    assert lib.pici_sizes(16, 7, None, None, None, None) == DTYPE
    a = 0x1000                                                                      # a fake, 16-aligned "pointer"
    n = 8192
    ws = ctypes.c_uint64()
    lib.pici_sizes(n, pici.F32, None, None, None, ctypes.byref(ws))
    C = lib.pici_compress
    assert C(a, n, 9, a, a, a, n, a, ws.value, None) == DTYPE
    assert C(a, 1 << 32, pici.F32, a, a, a, 1 << 32, a, ws.value, None) == INVALID
    assert C(None, n, pici.F32, a, a, a, n, a, ws.value, None) == INVALID
    assert C(a, n, pici.F32, a, None, a, n, a, ws.value, None) == INVALID
    assert C(a + 4, n, pici.F32, a, a, a, n, a, ws.value, None) == ALIGN
    assert C(a, n, pici.F32, a + 8, a, a, n, a, ws.value, None) == ALIGN
    assert C(a, n, pici.F32, a, a + 2, a, n, a, ws.value, None) == ALIGN
    assert C(a, n, pici.F32, a, a, a, n - 1, a, ws.value, None) == CAPACITY
    assert C(a, n, pici.F32, a, a, a, n, a, ws.value - 1, None) == WORKSPACE
    assert C(a, n, pici.F32, a, a, a, n, None, ws.value, None) == WORKSPACE
    S = lib.pici_reduce_ss
    assert S(a, a, a, a, a, a, n, pici.BF16, a, a, a, n, a, ws.value, None) == DTYPE       # reductions are fp32 only
    assert S(a, a, a, a, a, a, n, pici.F32, a, a, a, n - 1, a, ws.value, None) == CAPACITY
    assert S(a, a, a, a, None, a, n, pici.F32, a, a, a, n, a, ws.value, None) == INVALID
    assert lib.pici_reduce_sd(a, a, a, n, 7, a, None) == DTYPE                               # unknown dtype (bf16 sums exist)
    assert lib.pici_decompress(a, a, a, n, pici.F32, None, None) == INVALID
    assert lib.pici_decompress(a, a, a, n, pici.F32, a + 4, None) == ALIGN
    for code in (0, INVALID, DTYPE, ALIGN, CAPACITY, WORKSPACE, -6, -99):
        assert lib.pici_strerror(code)                                               # always a string, never NULL


def test_reduce_ss_rejects_aliased_outputs_and_host_forms_check_their_scratch():
    """include/pici.h: "Outputs must not alias inputs" (pici_reduce_ss) and the *_host calls' device scratch
    pointers are checked on the host, before any CUDA call."""
    lib = pici.lib()
    INVALID, ALIGN, WORKSPACE = -1, -3, -5
    n = 8192
    ws_bytes = ctypes.c_uint64()
    assert lib.pici_sizes(n, pici.F32, None, None, None, ctypes.byref(ws_bytes)) == 0
    a, b, c, w = 0x10000, 0x20000, 0x30000, 0x40000              # fake, 16-aligned "device pointers"
    big = 1 << 40
    ok_args = lambda Bo, Io, Ao: (a, a + 0x1000, a + 0x2000, b, b + 0x1000, b + 0x2000, n, pici.F32, Bo, Io, Ao, n, w, big, None)
    assert lib.pici_reduce_ss(*ok_args(a, c + 0x1000, c + 0x2000)) == INVALID          # Bo == Bx
    assert lib.pici_reduce_ss(*ok_args(c, b + 0x1000, c + 0x2000)) == INVALID          # Io == Iy
    assert lib.pici_reduce_ss(*ok_args(c, c + 0x1000, a + 0x2000)) == INVALID          # Ao == Ax
    h = (ctypes.c_uint64 * 4)()                                                          # any host memory
    hp, nnz = ctypes.addressof(h), ctypes.c_uint64()
    host = lambda d_dense, d_B, d_I, d_A, ws, wsb: lib.pici_compress_host(hp, n, pici.F32, hp, hp, hp, ctypes.byref(nnz),
                                                                          d_dense, d_B, d_I, d_A, ws, wsb, None)
    assert host(None, a, b, c, w, big) == INVALID
    assert host(a, None, b, c, w, big) == INVALID
    assert host(a, b, None, c, w, big) == INVALID
    assert host(a + 4, b, c, c + 0x1000, w, big) == ALIGN
    assert host(a, b, c, c + 0x1000, w, 16) == WORKSPACE
    back = lambda d_B, d_I, d_A, d_dense: lib.pici_decompress_host(hp, hp, hp, 1, n, pici.F32, hp, d_B, d_I, d_A, d_dense, None)
    assert back(None, a, b, c) == INVALID
    assert back(a, b, c, None) == INVALID
    assert back(a, b + 2, c, w) == ALIGN


def test_ring_entry_points_validate_before_any_cuda_call():
    """pici_ring_* reject bad configurations / pointers on the host (no GPU needed: nothing is launched)."""
    from paper_2607_04676_b200 import ring
    lib = pici.lib()
    INVALID, ALIGN, WORKSPACE = -1, -3, -5
    good = ring._Config(4, 0, 0, 0, 8192, 8193, 8193, 0.6, 0.5, 0.1, 2, 0)
    nbytes = ctypes.c_uint64()
    assert lib.pici_ring_arena_bytes(ctypes.byref(good), ctypes.byref(nbytes)) == 0 and nbytes.value % 256 == 0
    info = ring._Layout()
    assert lib.pici_ring_layout(ctypes.byref(good), ctypes.byref(info)) == 0
    assert info.rs_records == 3 * 4 and info.records == 3 * 4 + 4 and info.slots == 3 * 4     # two RS sets + one AG set
    keep = ring._Config(4, 0, 0, 1, 8192, 8193, 8193, 0.6, 0.5, 0.1, 2, 0)
    lib.pici_ring_layout(ctypes.byref(keep), ctypes.byref(info))
    assert info.slots == info.records
    for bad in (ring._Config(1, 0, 0, 0, 8192, 0, 0, 0, 0, 0, 1, 0), ring._Config(17, 0, 0, 0, 8192, 0, 0, 0, 0, 0, 1, 0),
                ring._Config(4, 0, 0, 0, 4097, 0, 0, 0, 0, 0, 1, 0), ring._Config(4, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 0)):
        assert lib.pici_ring_arena_bytes(ctypes.byref(bad), ctypes.byref(nbytes)) == INVALID
    ptrs = (ctypes.c_void_p * 4)(0x1000, 0x2000, 0x3000, 0x4000)
    arena = 0x10000
    for fn in (lib.pici_ring_reduce_scatter, lib.pici_ring_all_gather, lib.pici_ring_all_reduce):
        assert fn(None, ptrs, ptrs, arena, 1 << 40, None, None) == INVALID
        assert fn(ctypes.byref(good), None, ptrs, arena, 1 << 40, None, None) == INVALID
        assert fn(ctypes.byref(good), ptrs, ptrs, None, 1 << 40, None, None) == INVALID
        assert fn(ctypes.byref(good), ptrs, ptrs, arena + 16, 1 << 40, None, None) == ALIGN
        assert fn(ctypes.byref(good), ptrs, ptrs, arena, 1024, None, None) == WORKSPACE
        odd = (ctypes.c_void_p * 4)(0x1000, 0x2004, 0x3000, 0x4000)
        assert fn(ctypes.byref(good), odd, ptrs, arena, 1 << 40, None, None) == ALIGN
        strat = ring._Config(4, 7, 0, 0, 8192, 0, 0, 0, 0, 0, 1, 0)
        assert fn(ctypes.byref(strat), ptrs, ptrs, arena, 1 << 40, None, None) == INVALID
