"""Pins for oracle/coo_oracle.c (the paper's COO variant) against what the paper and the
mathematics fix: a hand-derived example (tests/golden/coo_example_n16.txt), reduction to numpy library routines
(flatnonzero / fancy indexing / add.at), the paper's size statements, an independent two-pointer merge written here,
and agreement with the Pici oracle on the dense meaning of every object."""
import os

import numpy as np
import pytest
import torch

import workloads as wl
from oracle import coo_oracle as co
from oracle import pici_oracle as po

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def f32bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int32).numpy().view(np.uint32)


def nz_np(bits):
    with np.errstate(invalid="ignore"):
        return bits.view(np.float32) != 0.0          # the FPU's x != 0, not the oracle's bit trick


def _example():
    ex = {}
    for line in open(os.path.join(GOLDEN, "coo_example_n16.txt")):
        tok = line.split()
        if tok and not tok[0].startswith("#"):
            ex[tok[0]] = tok[1:]
    n = int(ex["N"][0])
    mk = lambda k: co.Coo(n, np.array(ex[k + ".idx"], np.uint32), np.array(ex[k + ".val"], np.float32).view(np.uint32))
    return n, mk("X"), mk("Y"), mk("O"), np.array(ex["SD"], np.float32)


def _dense_of(c: co.Coo) -> np.ndarray:
    d = np.zeros(c.n, np.float32)
    d[c.idx] = c.val.view(np.float32)
    return d


def test_worked_example():
    n, X, Y, O, SD = _example()
    for c in (X, Y, O):
        got = co.compress(_dense_of(c))
        assert np.array_equal(got.idx, c.idx) and np.array_equal(got.val, c.val)
        assert np.array_equal(co.decompress(c).view(np.float32), _dense_of(c))
    got = co.reduce_ss(X, Y)
    assert np.array_equal(got.idx, O.idx) and np.array_equal(got.val, O.val)        # index 4 cancelled
    d = np.ones(n, np.float32)
    co.reduce_sd(X, d)
    assert np.array_equal(d, SD)


@pytest.mark.parametrize("n", [0, 1, 63, 4096, 4097, 70001])
@pytest.mark.parametrize("density", [0.0, 0.01, 0.5, 1.0])
def test_compress_is_flatnonzero(n, density):
    bits = f32bits(wl.sparse_buffer(n, density, seed=n + 17))
    c = co.compress(bits)
    want = np.flatnonzero(nz_np(bits)).astype(np.uint32)
    assert np.array_equal(c.idx, want) and np.array_equal(c.val, bits[want])
    assert c.message_bytes() == 8 * want.size
    assert np.array_equal(co.decompress(c), bits)                                     # round trip (no -0.0 here)
    if n:
        assert np.array_equal(co.decompress(c), po.decompress(po.compress(bits, "f32")))   # same dense meaning as Pici


def test_special_values():
    v = np.array([0.0, -0.0, np.nan, np.inf, -np.inf, 1e-45, -1e-45, 1.0], np.float32)
    bits = v.view(np.uint32).copy()
    bits[2] = 0x7FC12345                                                              # NaN payload survives
    c = co.compress(bits)
    assert list(c.idx) == [2, 3, 4, 5, 6, 7]                                          # +-0 are zeros, the rest is stored
    assert np.array_equal(c.val, bits[2:])
    back = co.decompress(c)
    assert back[1] == 0 and np.array_equal(back[2:], bits[2:])                        # -0.0 -> +0.0


def test_size_statements_of_the_paper():
    n = 1 << 20
    # "below 96.875 % sparsity, BV is more space-efficient than COO": equal at nnz = n / 32
    nnz = n // 32
    d = np.zeros(n, np.float32)
    d[:: 32] = 1.0
    c, p = co.compress(d), po.compress(d, "f32")
    assert c.nnz == nnz == p.nnz
    bv_bytes = 4 * nnz + n // 8                                                       # values + one bit per element
    assert c.message_bytes() == bv_bytes
    assert c.message_bytes() < p.message_bytes()                                      # Pici = BV + I: a little above
    assert p.message_bytes() - bv_bytes == 4 * (n // 4096 + 1)
    assert 1.0 - nnz / n == 0.96875
    # "At 50 % sparsity, COO requires the same amount of space as the dense representation"
    d[:] = 0
    d[::2] = 2.0
    assert co.compress(d).message_bytes() == 4 * n


def _two_pointer_merge(X: co.Coo, Y: co.Coo) -> co.Coo:
    """Independent statement: merge of two ascending lists, equal indices added (x + y), zeros dropped."""
    i = j = 0
    oi, ov = [], []
    xv, yv = X.val.view(np.float32), Y.val.view(np.float32)
    while i < X.nnz or j < Y.nnz:
        if j >= Y.nnz or (i < X.nnz and X.idx[i] < Y.idx[j]):
            k, s = X.idx[i], xv[i]; i += 1
        elif i >= X.nnz or Y.idx[j] < X.idx[i]:
            k, s = Y.idx[j], yv[j]; j += 1
        else:
            k, s = X.idx[i], np.float32(xv[i] + yv[j]); i += 1; j += 1
        if s != 0 or np.isnan(s):
            oi.append(k); ov.append(s)
    return co.Coo(X.n, np.array(oi, np.uint32), np.array(ov, np.float32).view(np.uint32))


@pytest.mark.parametrize("n,dx,dy", [(1, 1.0, 1.0), (5000, 0.02, 0.03), (9000, 0.5, 0.5), (4096, 0.0, 0.1), (8192, 1.0, 0.3)])
def test_reduce_ss_and_sd(n, dx, dy):
    xb, yb = wl.sparse_buffer(n, dx, seed=3), wl.sparse_buffer(n, dy, seed=4)
    yb[::7] = -xb[::7]                                                                # exact cancellations where both are set
    X, Y = co.compress(f32bits(xb)), co.compress(f32bits(yb))
    O = co.reduce_ss(X, Y)
    dense = (xb.numpy() + yb.numpy())
    want = co.compress(dense)                                                         # numpy's dense add, recompressed
    assert np.array_equal(O.idx, want.idx) and np.array_equal(O.val, want.val)
    tp = _two_pointer_merge(X, Y)
    assert np.array_equal(O.idx, tp.idx) and np.array_equal(O.val, tp.val)
    P = po.reduce_ss(po.compress(f32bits(xb), "f32"), po.compress(f32bits(yb), "f32"))
    assert np.array_equal(co.decompress(O), po.decompress(P))                         # Pici's merge means the same
    R = co.reduce_ss(Y, X)
    assert np.array_equal(R.idx, O.idx) and np.array_equal(R.val, O.val)              # commutative (no NaN here)
    E = co.reduce_ss(X, co.compress(np.zeros(n, np.float32)))
    assert np.array_equal(E.idx, X.idx) and np.array_equal(E.val, X.val)              # + empty = identity
    acc = yb.numpy().copy()
    co.reduce_sd(X, acc)
    ref = yb.numpy().copy()
    np.add.at(ref, X.idx.astype(np.int64), X.val.view(np.float32))                    # library scatter-add
    assert np.array_equal(acc.view(np.uint32), ref.view(np.uint32))
    untouched = np.ones(n, bool); untouched[X.idx] = False
    assert np.array_equal(acc.view(np.uint32)[untouched], f32bits(yb)[untouched])
