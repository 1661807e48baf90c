"""Pins for oracle/prune_oracle.c (sampled top-k pruning + leaky error feedback): a hand-worked
example, numpy's sort as the selection routine, the conservation law sent + e' == acc, the leak = 0 / leak = 1 special
cases and the kept fraction the recipe promises (1 % of the sample above the threshold)."""
import os

import numpy as np
import pytest

import workloads as wl
from oracle import pici_oracle as po
from oracle import prune_oracle as pr

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _example():
    ex = {}
    for line in open(os.path.join(GOLDEN, "prune_example_n12.txt")):
        tok = line.split()
        if tok and not tok[0].startswith("#"):
            ex[tok[0]] = tok[1:]
    f = lambda k: np.array(ex[k], np.float32)
    return f("G"), f("E"), float(ex["LEAK"][0]), np.array(ex["SAMPLE"], np.uint32), int(ex["K"][0]), f("TAU")[0], f("ACC"), f("SENT"), f("EOUT")


def test_worked_example():
    g, e, leak, sample, k, tau, acc, sent, eout = _example()
    assert np.array_equal(g + np.float32(leak) * e, acc)
    assert pr.threshold(g, e, leak, sample, k) == tau
    s, eo, c = pr.prune_ef(g, e, leak, tau)
    assert np.array_equal(s, sent) and np.array_equal(eo, eout) and c == 4
    p = po.compress(s.view(np.uint32), "f32")                                   # the message: Pici of what is sent
    assert p.nnz == 4 and np.array_equal(po.decompress(p), s.view(np.uint32))


@pytest.mark.parametrize("n,leak", [(1000, 0.0), (50_000, 1.0), (200_003, 0.9)])
def test_threshold_is_numpy_selection_and_ef_conserves(n, leak):
    g = wl.values(n, seed=1).numpy()
    e = (wl.values(n, seed=2).numpy() * np.float32(0.3)).astype(np.float32)
    rng = np.random.default_rng(n)
    m = max(8, n // 1000)
    sample = np.sort(rng.choice(n, size=m, replace=False)).astype(np.uint32)
    k = max(1, -(-m // 100))
    acc = (g + (np.float32(leak) * e).astype(np.float32)).astype(np.float32)     # two roundings, numpy fp32
    want = np.sort(np.abs(acc[sample]))[::-1][k - 1]
    tau = pr.threshold(g, e, leak, sample, k)
    assert tau == want
    sent, eout, c = pr.prune_ef(g, e, leak, tau)
    keep = np.abs(acc) >= tau
    assert c == int(keep.sum())
    assert np.array_equal(sent, np.where(keep, acc, np.float32(0)))
    assert np.array_equal(eout, np.where(keep, np.float32(0), acc))
    assert np.array_equal((sent + eout).view(np.uint32), (acc + np.float32(0)).view(np.uint32))   # nothing is lost
    assert (np.abs(acc[sample]) >= tau).sum() >= k                               # at least k of the sample pass
    if leak == 0.0:
        assert np.array_equal(sent, np.where(np.abs(g) >= tau, g, np.float32(0)))    # plain magnitude pruning of g


def test_kept_fraction_is_about_one_percent():
    """The recipe: sample 0.1 %, keep the top 1 % of the sample -> about 99 % sparsity of the message."""
    n = 1 << 22
    g = wl.values(n, seed=5).numpy()
    e = np.zeros(n, np.float32)
    sample = np.arange(0, n, 1000, dtype=np.uint32)
    k = -(-sample.size // 100)
    tau = pr.threshold(g, e, 1.0, sample, k)
    _, _, c = pr.prune_ef(g, e, 1.0, tau)
    assert 0.006 < c / n < 0.015                                                 # 1 % +- the sampling error of a 4195-element sample
    assert abs(float(tau) - 2.576) < 0.15                                        # the 99.5th percentile of |N(0,1)|


def test_nan_and_zero_threshold():
    g = np.array([np.nan, 0.0, -0.0, 1.0, -3.0, 0.5], np.float32)
    e = np.zeros(6, np.float32)
    sent, eout, c = pr.prune_ef(g, e, 1.0, 1.0)
    assert c == 2 and np.isnan(eout[0]) and sent[0] == 0                          # a NaN is never sent, it stays in e'
    assert list(sent[3:]) == [1.0, -3.0, 0.0] and list(eout[3:]) == [0.0, 0.0, 0.5]
    sent, eout, c = pr.prune_ef(g, e, 1.0, 0.0)                                  # tau = 0: everything but the NaN "passes"
    assert c == 5 and po.compress(sent.view(np.uint32), "f32").nnz == 3
    assert pr.threshold(g, e, 1.0, np.array([0, 3, 4], np.uint32), 1) == np.inf   # a NaN in the sample counts as large
