"""Pins for oracle/pici_oracle.c against what the paper and the mathematics fix.

None of these re-type the oracle's loop: they use (a) a hand-derived worked example stored as a
text fixture, (b) a reduction to library routines (numpy transpose + packbits + boolean-mask
compaction, i.e. the textbook BV format of PAPER.md:78 applied after the tile-local transpose),
(c) closed forms printed in the paper, (d) invariants, (e) brute force on tiny inputs.
"""
import os

import numpy as np
import pytest
import torch

import workloads as wl
from oracle import pici_oracle as po

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def f32bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int32).numpy().view(np.uint32)


def b16bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def nz_np(bits: np.ndarray) -> np.ndarray:
    """IEEE x != 0 evaluated by the floating-point unit (not by the oracle's bit trick)."""
    if bits.dtype == np.uint32:
        with np.errstate(invalid="ignore"):
            return bits.view(np.float32) != 0.0
    # bf16 -> fp32 is exact: place the 16 bits in the high half
    with np.errstate(invalid="ignore"):
        return (bits.astype(np.uint32) << 16).view(np.float32) != 0.0


def library_pici(bits: np.ndarray):
    """Pici via library routines: pad to whole tiles, tile-local transpose pi, then textbook BV."""
    n = bits.size
    T = (n + 4095) // 4096
    pad = np.zeros(T * 4096, bits.dtype)
    pad[:n] = bits
    dpi = pad.reshape(T, 64, 64).swapaxes(1, 2).reshape(-1)      # column-major inside each tile
    m = nz_np(dpi)
    B = np.packbits(m, bitorder="little").view(np.uint64) if T else np.zeros(0, np.uint64)
    A = dpi[m]
    counts = m.reshape(T, 4096).sum(axis=1) if T else np.zeros(0, np.int64)
    I = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
    return B, I, A


# ---------------------------------------------------------------------------------------------
# (a) worked example, tests/golden/worked_example_n8192.txt
# ---------------------------------------------------------------------------------------------

def _load_example():
    D = np.zeros(8192, np.float32)
    B = np.zeros(128, np.uint64)
    I = A = None
    for line in open(os.path.join(GOLDEN, "worked_example_n8192.txt")):
        tok = line.split()
        if not tok or tok[0].startswith("#"):
            continue
        if tok[0] == "D":
            D[int(tok[1])] = float(tok[2])
        elif tok[0] == "B":
            B[int(tok[1])] = np.uint64(int(tok[2], 16))
        elif tok[0] == "I":
            I = np.array([int(x) for x in tok[1:]], np.uint32)
        elif tok[0] == "A":
            A = np.array([float(x) for x in tok[1:]], np.float32)
    return D, B, I, A


def test_worked_example_layout():
    D, B, I, A = _load_example()
    p = po.compress(D, "f32")
    assert np.array_equal(p.B, B)
    assert np.array_equal(p.I, I)
    assert np.array_equal(p.A.view(np.float32), A)
    assert np.array_equal(po.decompress(p).view(np.float32), D)
    # Fig. 1 shape: two tiles -> 128 words, 3 index entries
    assert p.B.size == 128 and p.I.size == 3


# ---------------------------------------------------------------------------------------------
# (b) reduction to library routines, random + ragged + special values
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", wl.edge_sizes() + (1 << 16, (1 << 16) + 4095))
@pytest.mark.parametrize("density", [0.0, 0.01, 0.5, 1.0])
def test_compress_equals_library_bv_after_tile_transpose_f32(n, density):
    d = f32bits(wl.sparse_buffer(n, density, seed=n % 97 + 1))
    p = po.compress(d, "f32")
    B, I, A = library_pici(d)
    assert np.array_equal(p.B, B) and np.array_equal(p.I, I) and np.array_equal(p.A, A)


@pytest.mark.parametrize("n", [1, 4097, 1 << 15])
@pytest.mark.parametrize("density", [0.05, 0.9])
def test_compress_equals_library_bf16(n, density):
    d = b16bits(wl.sparse_buffer(n, density, seed=5, dtype="bf16"))
    p = po.compress(d, "bf16")
    B, I, A = library_pici(d)
    assert np.array_equal(p.B, B) and np.array_equal(p.I, I) and np.array_equal(p.A, A)
    assert np.array_equal(po.decompress(p), d)


def test_special_values_predicate_and_roundtrip():
    sv = wl.special_values_f32()
    d = np.zeros(4096 + 100, np.uint32)
    bits = f32bits(sv)
    pos = np.arange(bits.size) * 37 + 3
    d[pos] = bits
    p = po.compress(d, "f32")
    B, I, A = library_pici(d)
    assert np.array_equal(p.B, B) and np.array_equal(p.I, I) and np.array_equal(p.A, A)
    # -0.0 and +0.0 are not stored; NaN (quiet, signalling, payloads), Inf, subnormals are
    stored = set(int(x) for x in p.A)
    assert 0x80000000 not in stored and 0 not in stored
    for b in (0x7F800000, 0xFF800000, 0x7FC00001, 0xFFC12345, 0x7F800001, 0x00000001, 0x807FFFFF):
        assert b in stored
    back = po.decompress(p)
    expect = d.copy()
    expect[expect == 0x80000000] = 0          # -0.0 decompresses to +0.0 (C1)
    assert np.array_equal(back, expect)        # NaN payloads preserved bit for bit


def test_bf16_special_values():
    d = np.zeros(5000, np.uint16)
    d[[0, 70, 4095, 4096, 4999]] = [0x8000, 0x7FC1, 0x0001, 0xFF80, 0x8000]
    p = po.compress(d, "bf16")
    assert p.nnz == 3 and list(p.I) == [0, 2, 3]
    e = d.copy()
    e[e == 0x8000] = 0
    assert np.array_equal(po.decompress(p), e)


# ---------------------------------------------------------------------------------------------
# (c) closed forms the paper prints
# ---------------------------------------------------------------------------------------------

def test_metadata_closed_forms():
    # PAPER.md:116 "index overhead ... only ~0.78% relative to the bitvector"; "total overhead
    # relative to a 32-bit dense representation is only ~3.15%"; PAPER.md:78 BV 3.125%.
    for n in (4096, 8192, 1 << 20):
        p = po.compress(np.zeros(n, np.float32), "f32")
        assert p.B.nbytes == n // 8
        assert p.I.nbytes == n // 1024 + 4
        assert (p.I.nbytes - 4) / p.B.nbytes == 0.0078125
        assert (p.B.nbytes + p.I.nbytes - 4) / (4 * n) == 0.031494140625
        assert p.B.nbytes / (4 * n) == 0.03125
        assert p.message_bytes() == n // 8 + n // 1024 + 4
    assert round(0.031494140625, 4) == 0.0315           # omega in Eq. 4
    assert abs(0.99 ** 256 - 0.0763) < 5e-4


def test_message_size_matches_eq4():
    # Eq. 4: n' = n (1 - sigma + omega)
    n = 1 << 20
    d = f32bits(wl.sparse_buffer(n, 0.05, seed=3))
    p = po.compress(d, "f32")
    sigma = 1.0 - p.nnz / n
    assert abs(p.message_bytes() - 4 * n * (1 - sigma + 0.031494140625)) <= 4


# ---------------------------------------------------------------------------------------------
# (d) invariants
# ---------------------------------------------------------------------------------------------

def popcount64(a: np.ndarray) -> np.ndarray:
    return np.unpackbits(a.view(np.uint8)).reshape(a.size, 64).sum(axis=1)


@pytest.mark.parametrize("density", [0.001, 0.1, 0.5])
def test_index_invariants(density):
    n = 40 * 4096 + 123
    d = f32bits(wl.sparse_buffer(n, density, seed=11))
    p = po.compress(d, "f32")
    T = po.num_tiles(n)
    assert p.I[0] == 0
    per_tile = popcount64(p.B).reshape(T, 64).sum(axis=1)
    assert np.array_equal(np.diff(p.I.astype(np.int64)), per_tile)
    assert int(p.I[T]) == int(popcount64(p.B).sum()) == p.A.size == int(nz_np(d).sum())
    assert po.nnz_pici(p) == po.nnz_dense(d, "f32") == p.A.size
    # bits beyond n are zero (virtual padding, C9 #4)
    tail_rows = np.unpackbits(p.B[-64:].view(np.uint8), bitorder="little").reshape(64, 64)  # [col][row]
    idx = (T - 1) * 4096 + np.arange(64)[None, :] * 64 + np.arange(64)[:, None]
    assert not tail_rows[idx >= n].any()


def test_nnz_dense_bf16_counts_ieee_nonzeros():
    """Pin for oracle_nnz_dense_b16 (predicate C1): the count of a bf16 buffer equals
    (a) the FPU's `x != 0` over the same bits widened exactly to fp32, (b) a brute-force Python loop on
    the hand-listed special patterns, (c) len(A) of the bf16 compressor - on ragged sizes."""
    special = np.array([0x0000, 0x8000, 0x0001, 0x8001, 0x007F, 0x0080, 0x7F80, 0xFF80, 0x7FC0, 0xFFC1, 0x7F81,
                        0x3F80, 0xBF80, 0x7FFF, 0xFFFF], np.uint16)
    # by hand: only +0 (0x0000) and -0 (0x8000) are zeros; subnormals, Inf and every NaN count
    assert po.nnz_dense(special, "bf16") == special.size - 2
    assert po.nnz_dense(special, "bf16") == sum(1 for b in special.tolist() if (b & 0x7FFF) != 0)
    for k in range(special.size + 1):                 # every prefix: a dropped / doubled element shows
        assert po.nnz_dense(special[:k].copy(), "bf16") == int(nz_np(special[:k]).sum())
    for n, dens, seed in ((0, 0.5, 1), (1, 1.0, 2), (63, 0.3, 3), (4097, 0.01, 4), (3 * 4096 + 17, 0.5, 5),
                          (40 * 4096 + 123, 0.1, 6)):
        d = b16bits(wl.sparse_buffer(n, dens, seed=seed, dtype="bf16")).copy()
        if n > 20:
            d[3], d[7], d[n - 1] = 0x8000, 0x0001, 0x7FC0        # -0.0, smallest subnormal, NaN
        want = int(nz_np(d).sum())
        assert po.nnz_dense(d, "bf16") == want
        assert po.compress(d, "bf16").A.size == want == po.nnz_pici(po.compress(d, "bf16"))
    # an fp32 buffer viewed as twice as many 16-bit words is NOT the same count: the two variants differ
    f = f32bits(wl.sparse_buffer(4096, 0.5, seed=9))
    assert po.nnz_dense(f, "f32") != po.nnz_dense(f.view(np.uint16).copy(), "bf16")


def test_index_is_a_random_access_offset_table():
    n = 9 * 4096 + 5
    d = f32bits(wl.sparse_buffer(n, 0.3, seed=2))
    p = po.compress(d, "f32")
    assert np.array_equal(po.decompress_via_index(p), po.decompress(p))
    assert np.array_equal(po.decompress(p), d)


def test_all_zero_and_all_nonzero():
    n = 3 * 4096
    p = po.compress(np.zeros(n, np.float32), "f32")
    assert p.A.size == 0 and not p.B.any() and not p.I.any()
    d = np.arange(1, n + 1, dtype=np.float32)
    p = po.compress(d, "f32")
    assert (p.B == np.uint64(0xFFFFFFFFFFFFFFFF)).all()
    assert np.array_equal(p.I, np.arange(4) * 4096)
    assert np.array_equal(p.A.view(np.float32), d.reshape(3, 64, 64).swapaxes(1, 2).reshape(-1))


def test_tile_corners():
    n = 2 * 4096
    for t in range(2):
        for (r, c) in [(0, 0), (0, 63), (63, 0), (63, 63)]:
            d = np.zeros(n, np.float32)
            d[4096 * t + 64 * r + c] = -2.5
            p = po.compress(d, "f32")
            assert p.nnz == 1
            assert p.B[64 * t + c] == np.uint64(1) << np.uint64(r)
            assert np.count_nonzero(p.B) == 1
            assert list(p.I) == [0, 0 if t == 1 else 1, 1]


def test_pici_bitvector_differs_from_plain_bv_only_by_the_tile_transpose():
    # PAPER.md:112 "the bitvectors of Pici and BV are generally not identical"
    n = 4096
    d = f32bits(wl.sparse_buffer(n, 0.2, seed=8))
    p = po.compress(d, "f32")
    bv = np.packbits(nz_np(d), bitorder="little").view(np.uint64)
    assert not np.array_equal(bv, p.B)
    bits_pici = np.unpackbits(p.B.view(np.uint8), bitorder="little").reshape(64, 64)   # [c][r]
    bits_bv = np.unpackbits(bv.view(np.uint8), bitorder="little").reshape(64, 64)      # [r][c]
    assert np.array_equal(bits_pici.T, bits_bv)


# ---------------------------------------------------------------------------------------------
# (e) reductions: brute force against numpy dense arithmetic
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 64, 4097, 5 * 4096])
@pytest.mark.parametrize("dx,dy", [(0.01, 0.01), (0.3, 0.6), (1.0, 0.0)])
def test_reduce_sd_is_dense_add(n, dx, dy):
    x = wl.sparse_buffer(n, dx, seed=21).numpy()
    y = wl.sparse_buffer(n, dy, seed=22).numpy()
    px = po.compress(x, "f32")
    acc = y.copy()
    po.reduce_sd(px, acc)
    assert np.array_equal(acc.view(np.uint32), (y + x).view(np.uint32))
    # untouched where x has no bit: a -0.0 there must survive
    y2 = y.copy()
    hole = np.flatnonzero(x == 0)
    if hole.size:
        y2[hole[0]] = -0.0
        acc = y2.copy()
        po.reduce_sd(px, acc)
        assert acc.view(np.uint32)[hole[0]] == 0x80000000


@pytest.mark.parametrize("n", [1, 4096, 4097, 6 * 4096 + 9])
@pytest.mark.parametrize("dx,dy", [(0.01, 0.02), (0.4, 0.5), (0.0, 0.3), (1.0, 1.0)])
def test_reduce_ss_is_compress_of_dense_sum(n, dx, dy):
    x = wl.sparse_buffer(n, dx, seed=31).numpy()
    y = wl.sparse_buffer(n, dy, seed=32).numpy()
    px, py = po.compress(x, "f32"), po.compress(y, "f32")
    o = po.reduce_ss(px, py)
    B, I, A = library_pici((x + y).view(np.uint32))
    assert np.array_equal(o.B, B) and np.array_equal(o.I, I) and np.array_equal(o.A, A)
    o2 = po.reduce_ss(py, px)                                   # commutative bitwise (non-NaN)
    assert np.array_equal(o.B, o2.B) and np.array_equal(o.I, o2.I) and np.array_equal(o.A, o2.A)


def test_reduce_ss_identity_and_cancellation():
    n = 2 * 4096 + 77
    x = wl.sparse_buffer(n, 0.1, seed=41).numpy()
    px = po.compress(x, "f32")
    empty = po.compress(np.zeros(n, np.float32), "f32")
    o = po.reduce_ss(px, empty)
    assert np.array_equal(o.B, px.B) and np.array_equal(o.I, px.I) and np.array_equal(o.A, px.A)
    # exact cancellation: x + (-x) is not stored; popcount(B) == I[T] == len(A) still holds
    y = -x
    keep = np.flatnonzero(x)[::3]
    y[keep] = 1.0
    o = po.reduce_ss(px, po.compress(y, "f32"))
    assert o.nnz == keep.size == int(popcount64(o.B).sum()) == o.A.size
    assert np.array_equal(po.decompress(o).view(np.float32), x + y)


def test_maybe_densify_brute_force():
    n = 4096 * 3
    x = wl.sparse_buffer(n, 0.25, seed=51).numpy()
    p = po.compress(x, "f32")
    for sw in (0, 1, p.nnz - 1, p.nnz, p.nnz + 1, n, n + 1):
        out = np.full(n, 0xDEADBEEF, np.uint32)
        switched = po.maybe_densify(p, sw, out)
        assert switched == (p.nnz >= sw)                        # inclusive (C9 #9)
        if switched:
            assert np.array_equal(out, x.view(np.uint32))
        else:
            assert (out == 0xDEADBEEF).all()                    # not written
    assert wl.nnz_switch_from_permille(1000, 400) == 400
    assert wl.nnz_switch_from_permille(1001, 25) == 26          # ceil


def test_tiny_brute_force_python_loops():
    """Independent pure-Python restatement from the prose of PAPER.md:108-112 on a tiny input:
    'ordered first by their parent tile, next by their parent column, and finally by their
    intra-column position'."""
    rng = np.random.default_rng(0)
    n = 4096 + 300
    d = np.where(rng.random(n) < 0.07, rng.standard_normal(n), 0.0).astype(np.float32)
    triples = sorted((i // 4096, (i % 4096) % 64, (i % 4096) // 64, float(d[i]))
                     for i in range(n) if d[i] != 0)
    p = po.compress(d, "f32")
    assert [v for *_, v in triples] == [float(v) for v in p.A.view(np.float32)]
    for t, c, r, _ in triples:
        assert (int(p.B[64 * t + c]) >> r) & 1
    assert sum(bin(int(w)).count("1") for w in p.B) == len(triples)


# ---------------------------------------------------------------------------------------------
# bf16 reductions: "add in fp32, round-to-nearest-even" - pinned by torch's bf16 addition, a library
# routine that widens to fp32, adds and rounds RNE
# ---------------------------------------------------------------------------------------------

def test_bf16_dense_add_and_reduce_sd_are_torch_bf16_addition():
    n = 3 * 4096 + 17
    a = wl.sparse_buffer(n, 0.3, seed=21, dtype="bf16")
    b = wl.sparse_buffer(n, 0.6, seed=22, dtype="bf16")
    b[::5] = -a[::5]                                                  # cancellations
    a[7], b[7] = 1.0, 2.0 ** -8                                       # a tie: 1 + 2^-8 rounds to even (1.0)
    a[8], b[8] = 1.0 + 2.0 ** -7, 2.0 ** -8                           # a tie that rounds up to even
    a[9], b[9] = 3.0e38, 3.0e38                                       # overflow to +inf
    want = (a + b)                                                    # torch: fp32 add, RNE to bf16
    got = po.dense_add(b16bits(a), b16bits(b))
    assert np.array_equal(got, b16bits(want))
    assert got[7] == 0x3F80 and got[8] == 0x3F82 and got[9] == 0x7F80
    x = po.compress(b16bits(a), "bf16")
    acc = b16bits(b).copy()
    po.reduce_sd(x, acc)
    mask = (a != 0).numpy()
    ref = np.where(mask, b16bits(a + b), b16bits(b))                  # untouched where a has no value
    assert np.array_equal(acc, ref)
    nan = po.dense_add(np.array([0x7FC1, 0x7F80], np.uint16), np.array([0x3F80, 0xFF80], np.uint16))
    assert (nan[0] & 0x7FFF) > 0x7F80 and (nan[1] & 0x7FFF) > 0x7F80  # NaN + 1 and inf - inf are NaN
