"""Pins for the paper's adaptive policy in oracle/ring_oracle.py (Eq. 7):
a hand-derived trace (tests/golden/policy_sandwich_p4.txt), exactness against the dense left fold whatever the
format decisions, the two degenerate policies that reduce to already-pinned collectives, and the fill-in law."""
import os

import numpy as np
import pytest

import workloads as wl
from oracle import pici_oracle as po
from oracle import ring_oracle as ro

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "policy_sandwich_p4.txt")


def biteq(a, b):
    return np.array_equal(a.view(np.uint32), b.view(np.uint32))


def disjoint_inputs(P=4, n=16384):
    """Rank r: every chunk has a nonzero exactly where i mod 8 == r (values never 0, never cancelling)."""
    X = []
    i = np.arange(P * n)
    for r in range(P):
        v = (1.0 + 0.25 * r + (i % 97) / 128.0).astype(np.float32)
        X.append(np.where(i % 8 == r, v, np.float32(0.0)).astype(np.float32))
    return X


def load_golden():
    rows, final = [], {}
    for line in open(GOLDEN):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "final":
            final[int(f[1])] = float(f[2])
        else:
            rows.append((int(f[0]), int(f[1]), int(f[2]), f[3], float(f[4]), f[5], None if f[6] == "-" else int(f[6])))
    return rows, final


def test_worked_example_sandwich():
    pol = ro.Policy(intra_thresh=0.8, inter_thresh=0.6, ag_thresh=0.1, ranks_per_node=2)
    X = disjoint_inputs()
    out, log, sigma0, sigma = ro.ring_reduce_scatter_policy(X, pol)
    rows, final = load_golden()
    assert len(rows) == len(log.entries)
    for (step, rank, chunk, link, dec, fmt, nnz) in rows:
        e = log.at("rs", step, rank)
        assert (e.chunk, e.fmt, e.nnz) == (chunk, fmt, nnz), (step, rank)
        assert e.extrapolated_sparsity == dec, (step, rank, e.extrapolated_sparsity)   # dyadic: exact in fp64
        assert pol.link_thresh(rank, 4) == (0.8 if link == "intra" else 0.6)
    assert sigma0 == [0.875] * 4
    assert sigma == [final[r] for r in range(4)]
    # the sandwich on chunk 0 and the collective's exactness
    assert [log.at("rs", s, r).fmt for s, r in ((0, 1), (1, 2), (2, 3))] == ["pici", "dense", "pici"]
    ref = ro.reduce_scatter_definition(X)
    assert all(biteq(out[r], ref[r]) for r in range(4))
    # a message sent after a dense one is the compression of the dense partial sum (re-calibrated count)
    m = log.at("rs", 2, 3).msg
    part = po.dense_add(po.dense_add(X[1][:16384].copy(), X[2][:16384].copy()), X[3][:16384].copy())
    assert biteq(po.decompress(m.pici).view(np.float32), part) and m.nnz == 3 * 2048


@pytest.mark.parametrize("P,rpn", [(2, 1), (3, 2), (4, 2), (8, 2), (8, 4)])
@pytest.mark.parametrize("intra,inter", [(0.6, 0.5), (0.95, 0.9), (0.9, 0.99), (0.0, 0.0), (1.0, 1.0), (0.93, 0.2)])
def test_policy_collectives_are_exact(P, rpn, intra, inter):
    cfg = wl.RingConfig("small", P, P * 4096 * 2, 0.02, 0.03, "normal", 1.0, 3)
    X = [b.numpy() for b in cfg.buffers()]
    pol = ro.Policy(intra, inter, 0.85, rpn)
    out, log, sigma0, sigma = ro.ring_reduce_scatter_policy(X, pol)
    ref = ro.reduce_scatter_definition(X)
    assert all(biteq(out[r], ref[r]) for r in range(P))
    n = cfg.chunk
    for e in log.entries:
        tau = pol.link_thresh(e.rank, P)
        assert (e.fmt == "dense") == (e.extrapolated_sparsity <= tau)
        assert e.chunk == (e.rank - 1 - e.step) % P                              # C8 schedule
        if e.fmt == "pici":
            assert e.nnz == e.msg.pici.nnz == int(np.count_nonzero(po.decompress(e.msg.pici).view(np.float32)))
        else:
            assert e.nnz is None                                                 # no count after a dense send
    outs, log2 = ro.ring_all_reduce_policy(X, pol)
    want = np.concatenate(ref)
    assert all(biteq(o, want) for o in outs)
    for e in (e for e in log2.entries if e.phase == "ar.ag" and e.step == 0):
        assert (e.fmt == "dense") == (e.extrapolated_sparsity <= pol.ag_thresh)


def test_degenerate_policies_reduce_to_the_pinned_collectives():
    P = 4
    cfg = wl.RingConfig("small", P, P * 4096 * 3, 0.0, 0.05, "normal", 1.0, 1)
    X = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    # thresholds 0: sparsity is never <= 0 here, every send is Pici = the measured-nnz algorithm that never switches
    _, log, _, _ = ro.ring_reduce_scatter_policy(X, ro.Policy(0.0, 0.0, 0.0, 2))
    _, ref = ro.ring_reduce_scatter(X, n + 1)
    assert len(log.entries) == len(ref.entries)
    for e in log.entries:
        w = ref.at("rs", e.step, e.rank)
        assert e.fmt == w.fmt == "pici" and e.nnz == w.nnz
        assert np.array_equal(e.msg.pici.B, w.msg.pici.B) and np.array_equal(e.msg.pici.A, w.msg.pici.A)
    # thresholds 1: every send is dense = the dense ring (partial left folds)
    _, log1, _, _ = ro.ring_reduce_scatter_policy(X, ro.Policy(1.0, 1.0, 1.0, 2))
    for e in log1.entries:
        assert e.fmt == "dense"
        acc = X[(e.chunk + 1) % P][e.chunk * n:(e.chunk + 1) * n].copy()
        for k in range(2, e.step + 2):
            acc = po.dense_add(acc, np.ascontiguousarray(X[(e.chunk + k) % P][e.chunk * n:(e.chunk + 1) * n]))
        assert biteq(e.msg.dense, acc)


def test_calibration_follows_the_fill_in_law():
    """Independent supports: the count-calibrated sparsity after k contributions is sigma_0^k (Eq. 7) within
    Bernoulli noise, which is what makes the extrapolation a usable predictor."""
    P = 8
    cfg = wl.RingConfig("small", P, P * 4096 * 8, 0.0, 0.05, "normal", 1.0, 5)
    X = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    _, log, sigma0, _ = ro.ring_reduce_scatter_policy(X, ro.Policy(0.0, 0.0, 0.0, 2))
    for e in log.entries:
        k = e.step + 1
        d = 1.0 - 0.95 ** k
        assert abs(ro.measured_sparsity(e.nnz, n) - 0.95 ** k) < 6.0 * (d * (1 - d) / n) ** 0.5
        if e.step > 0:                                   # decision value = previous calibrated value * sigma_0
            assert abs(e.extrapolated_sparsity - 0.95 ** k) < 0.01
