"""Pins for oracle/ring_oracle.py: the paper's sparse ring algorithm (scatter-add + recompress +
threshold switch) must equal the plain definition of the collective - a dense left fold in ring
order - bit for bit ("SpCCL collectives are exact"), and match an fp64 sum in
any order to 1e-6 * sum|x|.  Also the schedule (C8), the fill-in law Eq. 7 and the
switch behaviour."""
import numpy as np
import pytest

import workloads as wl
from oracle import pici_oracle as po
from oracle import ring_oracle as ro


def small_cfg(P=4, n_per_rank=4 * 4096 * 4, private=0.05, common=0.0, seed=0, dist="normal"):
    return wl.RingConfig("small", P, n_per_rank, common, private, dist, 1.0, seed)


def bufs(cfg):
    return [b.numpy() for b in cfg.buffers()]


def biteq(a, b):
    return np.array_equal(a.view(np.uint32), b.view(np.uint32))


@pytest.mark.parametrize("P", [2, 3, 4, 8])
@pytest.mark.parametrize("switch_permille", [0, 60, 120, 1001])
def test_reduce_scatter_algorithm_equals_left_fold(P, switch_permille):
    cfg = small_cfg(P=P, n_per_rank=P * 4096 * 2)
    X = bufs(cfg)
    n = cfg.chunk
    sw = wl.nnz_switch_from_permille(n, switch_permille)
    out, log = ro.ring_reduce_scatter(X, sw)
    ref = ro.reduce_scatter_definition(X)
    for r in range(P):
        assert biteq(out[r], ref[r])
    # any-order fp64 sum within 1e-6 * sum |x| (north_star tolerance)
    Xs = np.stack(X).astype(np.float64)
    tot, mag = Xs.sum(0), np.abs(Xs).sum(0)
    got = np.concatenate(out).astype(np.float64)
    assert (np.abs(got - tot) <= 1e-6 * mag + 1e-300).all()


def test_reduce_scatter_schedule_and_switch_monotone():
    P = 4
    cfg = small_cfg(P=P, n_per_rank=P * 4096 * 4, private=0.05)
    X = bufs(cfg)
    n = cfg.chunk
    sw = wl.nnz_switch_from_permille(n, 120)      # density .05,.0975,.1426 -> switch at 3rd contribution
    out, log = ro.ring_reduce_scatter(X, sw)
    for e in log.entries:
        assert e.chunk == (e.rank - 1 - e.step) % P          # C8 schedule
        assert e.msg.chunk == e.chunk
    for c in range(P):
        fmts = [e.fmt for e in sorted((e for e in log.entries if e.chunk == c), key=lambda e: e.step)]
        assert fmts == ["pici", "pici", "dense"], fmts       # once dense stays dense
        assert log.switch_step[c] == 2
    # never: default theta = 0.4 (intra_thresh 0.6 sparsity)
    out2, log2 = ro.ring_reduce_scatter(X, wl.nnz_switch_from_permille(n, 400))
    assert all(e.fmt == "pici" for e in log2.entries)
    assert all(v is None for v in log2.switch_step.values())
    for r in range(P):
        assert biteq(out[r], out2[r])                        # the format never changes the result
    # always dense from step 0
    out3, log3 = ro.ring_reduce_scatter(X, 0)
    assert all(e.fmt == "dense" for e in log3.entries)
    for r in range(P):
        assert biteq(out[r], out3[r])


def test_messages_are_the_running_partial_sums():
    P = 4
    cfg = small_cfg(P=P, n_per_rank=P * 4096)
    X = bufs(cfg)
    n = cfg.chunk
    _, log = ro.ring_reduce_scatter(X, n + 1)
    for e in log.entries:
        # message sent by rank r at step s carries chunk c summed over ranks r-s .. r (left fold)
        c, r, s = e.chunk, e.rank, e.step
        acc = X[(r - s) % P][c * n:(c + 1) * n].copy()
        for j in range(s - 1, -1, -1):
            acc = acc + X[(r - j) % P][c * n:(c + 1) * n]
        assert np.array_equal(po.decompress(e.msg.pici), acc.view(np.uint32))
        assert e.nnz == np.count_nonzero(acc) == e.msg.pici.nnz


def test_fill_in_law_config1():
    """Eq. 7: independent supports, density after k contributions = 1 - sigma0^k.
    Config 1: 99% -> 0.0100, 0.0199, 0.0297 (and 0.0394 in the output)."""
    cfg = wl.config1()
    X = bufs(cfg)
    n = cfg.chunk
    out, log = ro.ring_reduce_scatter(X, n + 1, keep_messages=False)
    for e in log.entries:
        k = e.step + 1
        d = 1 - 0.99 ** k
        assert abs(e.nnz / n - d) < 5 * np.sqrt(d * (1 - d) / n), (k, e.nnz / n)
        assert abs(e.nnz / n - cfg.expected_density(k)) < 5 * np.sqrt(d / n)
        # Eq. 7 extrapolation logged beside the measurement is close to it
        assert abs((1 - e.extrapolated_sparsity) - e.nnz / n) < 2e-3
    d4 = np.mean([np.count_nonzero(o) / n for o in out])
    assert abs(d4 - (1 - 0.99 ** 4)) < 1e-3
    ref = ro.reduce_scatter_definition(X)
    for r in range(cfg.ranks):
        assert biteq(out[r], ref[r])


def test_config1_switch_at_2p5_percent():
    """theta = 2.5% -> the switch happens after the 3rd contribution
    (density 0.0297), i.e. the message sent at step 2 is dense."""
    cfg = wl.config1()
    X = bufs(cfg)
    n = cfg.chunk
    out, log = ro.ring_reduce_scatter(X, wl.nnz_switch_from_permille(n, 25), keep_messages=False)
    assert all(v == 2 for v in log.switch_step.values())
    ref = ro.reduce_scatter_definition(X)
    for r in range(cfg.ranks):
        assert biteq(out[r], ref[r])


def test_all_gather_is_concatenation():
    P = 4
    cfg = small_cfg(P=P, n_per_rank=4096 * 3, private=0.2)
    shards = bufs(cfg)
    outs, log = ro.ring_all_gather(shards)
    ref = ro.all_gather_definition(shards)
    for r in range(P):
        assert biteq(outs[r], ref)
    for e in log.entries:
        assert e.chunk == (e.rank - e.step) % P and e.fmt == "pici"
    # 1 compress + (P-1) decompress per rank (Eq. 5)
    assert sum(1 for e in log.entries if e.step == 0) == P
    assert sum(1 for e in log.entries if e.step > 0) == P * (P - 1)
    # -0.0 in a remote shard arrives as +0.0, own slot is a plain copy (C9 #12)
    shards[1][5] = -0.0
    outs, _ = ro.ring_all_gather(shards)
    n = shards[0].size
    assert outs[1].view(np.uint32)[n + 5] == 0x80000000
    assert outs[0].view(np.uint32)[n + 5] == 0


@pytest.mark.parametrize("ag_permille", [0, 900, 1001])
def test_all_reduce_equals_definition_and_all_ranks_identical(ag_permille):
    P = 4
    cfg = small_cfg(P=P, n_per_rank=P * 4096 * 2, private=0.05, common=0.05, dist="uniform")
    X = bufs(cfg)
    n = cfg.chunk
    outs, log = ro.ring_all_reduce(X, wl.nnz_switch_from_permille(n, 150),
                                   wl.nnz_switch_from_permille(n, ag_permille))
    ref = ro.all_reduce_definition(X)
    for r in range(P):
        assert biteq(outs[r], ref)
    ag0 = [e for e in log.entries if e.phase == "ar.ag" and e.step == 0]
    assert len(ag0) == P
    want = "dense" if ag_permille == 0 else "pici"             # ag_thresh decision
    assert all(e.fmt == want for e in ag0)
    # shared support fills in more slowly than independent supports (config 4 recipe)
    rs = [e for e in log.entries if e.phase == "rs" and e.nnz is not None]
    for e in rs:
        k = e.step + 1
        assert abs(e.nnz / n - cfg.expected_density(k)) < 0.02
