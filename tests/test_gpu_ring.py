"""GPU parity of the host ring driver (paper_2607_04676_b200/ring.py) against oracle/ring_oracle.py,
MESSAGE BY MESSAGE: for every (phase, step, rank) the format word, the measured nnz and the full
message (B, I, A or the dense buffer) must equal the oracle's log bit for bit, and the outputs must
equal the dense left fold in ring order bit for bit.  Both strategies of the
reduce-scatter step are covered: "paper" (scatter-add + recompress) and "fused"
(sparse+sparse merge, north_star).
"""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import pici_oracle as po
from oracle import ring_oracle as ro

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from paper_2607_04676_b200 import pici, ring
    pici.lib()
    return pici, ring


def _u32(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int32).numpy().view(np.uint32)


def _check_records(pk, res, log: ro.RingLog):
    fmts = res.formats()
    nnz = res.nnz.cpu().numpy().view(np.uint32)
    for rec, f in zip(res.records, fmts):
        e = log.at(rec.phase, rec.step, rec.rank)
        assert e.chunk == rec.chunk, (rec.phase, rec.step, rec.rank)
        assert e.fmt == f, (rec.phase, rec.step, rec.rank, e.fmt, f)
        if e.nnz is not None:
            assert int(nnz[rec.nnz_index]) == e.nnz
        if rec.msg is None or e.msg is None:
            continue
        if e.fmt == "pici":
            B, I, A = rec.msg.pici.to_host()
            w = e.msg.pici
            assert np.array_equal(I[:w.I.size], w.I) and np.array_equal(B[:w.B.size], w.B)
            assert np.array_equal(A, w.A)
        else:
            assert np.array_equal(_u32(rec.msg.dense), e.msg.dense.view(np.uint32))


def _small(P, chunk_tiles, private, common=0.0, seed=0, dist="normal"):
    return wl.RingConfig("small", P, P * chunk_tiles * wl.TILE, common, private, dist, 1.0, seed)


@pytest.mark.parametrize("strategy", ["fused", "paper"])
@pytest.mark.parametrize("P,permille", [(4, 400), (4, 120), (3, 60), (8, 150), (2, 1000)])
def test_reduce_scatter_message_by_message(mods, strategy, P, permille):
    pk, ring = mods
    cfg = _small(P, 5, 0.05, seed=P)
    Xh = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    sw = wl.nnz_switch_from_permille(n, permille)
    want, log = ro.ring_reduce_scatter(Xh, sw)
    drv = ring.RingDriver(P, n, strategy=strategy, keep_messages=True)
    res = drv.reduce_scatter([torch.from_numpy(x).cuda() for x in Xh], sw)
    torch.cuda.synchronize()
    _check_records(pk, res, log)
    fold = ro.reduce_scatter_definition(Xh)
    for r in range(P):
        assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))
        assert np.array_equal(_u32(res.outputs[r]), fold[r].view(np.uint32))
    assert res.switch_steps("rs") == log.switch_step


def test_config1_round_trip_and_reduce_scatter(mods):
    """BASELINE.json configs[0]: P=4, N=2^20 per rank, 99% sparsity, seed 0; default theta (never
    switches) and theta = 2.5% (switch after the third contribution)."""
    pk, ring = mods
    cfg = wl.config1()
    Xh = [b.numpy() for b in cfg.buffers()]
    Xd = [torch.from_numpy(x).cuda() for x in Xh]
    n = cfg.chunk
    for x_h, x_d in zip(Xh, Xd):                       # Pici round trip of each rank's buffer
        want = po.compress(x_h.view(np.uint32), "f32")
        got = pk.alloc_pici(x_d.numel(), pk.F32)
        pk.compress(x_d, got, pk.alloc_workspace(x_d.numel()))
        B, I, A = got.to_host()
        assert np.array_equal(B[:want.B.size], want.B) and np.array_equal(I[:want.I.size], want.I)
        assert np.array_equal(A, want.A)
        back = torch.empty_like(x_d)
        pk.decompress(got, back)
        assert np.array_equal(_u32(back), x_h.view(np.uint32))
    for permille, strategy in ((400, "fused"), (25, "fused"), (25, "paper")):
        sw = wl.nnz_switch_from_permille(n, permille)
        want, log = ro.ring_reduce_scatter(Xh, sw)
        drv = ring.RingDriver(cfg.ranks, n, strategy=strategy, keep_messages=True)
        res = drv.reduce_scatter(Xd, sw)
        torch.cuda.synchronize()
        _check_records(pk, res, log)
        for r in range(cfg.ranks):
            assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))
        assert res.switch_steps("rs") == log.switch_step
        if permille == 25:
            assert set(log.switch_step.values()) == {2}


@pytest.mark.parametrize("P", [2, 4, 8])
def test_all_gather_message_by_message(mods, P):
    pk, ring = mods
    n = 3 * wl.TILE
    shards_h = [wl.sparse_buffer(n, 0.02 * (r + 1), seed=50 + r).numpy() for r in range(P)]
    sw = wl.nnz_switch_from_permille(n, 30)             # shard 0 (2 %) travels as Pici, the others dense
    want, log = ro.ring_all_gather(shards_h, sw)
    drv = ring.RingDriver(P, n, keep_messages=True)
    res = drv.all_gather([torch.from_numpy(x).cuda() for x in shards_h], sw)
    torch.cuda.synchronize()
    _check_records(pk, res, log)
    cat = ro.all_gather_definition(shards_h)
    for r in range(P):
        assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))
        assert np.array_equal(_u32(res.outputs[r]), cat.view(np.uint32))
    assert {"pici", "dense"} <= set(res.formats())


@pytest.mark.parametrize("strategy", ["fused", "paper"])
@pytest.mark.parametrize("rs_permille,ag_permille", [(400, 900), (200, 900), (200, 250)])
def test_all_reduce_matches_oracle_and_all_ranks_identical(mods, strategy, rs_permille, ag_permille):
    """Config-4 style supports (shared + private masks, U(-1,1)) at a small size."""
    pk, ring = mods
    cfg = _small(4, 4, 1.0 - 0.90 / 0.95, common=0.05, seed=4, dist="uniform")
    Xh = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    sw_rs = wl.nnz_switch_from_permille(n, rs_permille)
    sw_ag = wl.nnz_switch_from_permille(n, ag_permille)
    want, log = ro.ring_all_reduce(Xh, sw_rs, sw_ag)
    drv = ring.RingDriver(cfg.ranks, n, strategy=strategy, keep_messages=True)
    res = drv.all_reduce([torch.from_numpy(x).cuda() for x in Xh], sw_rs, sw_ag)
    torch.cuda.synchronize()
    _check_records(pk, res, log)
    ref = ro.all_reduce_definition(Xh)
    for r in range(cfg.ranks):
        assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))
        assert np.array_equal(_u32(res.outputs[r]), ref.view(np.uint32))
    # any-order check (north_star): |out - fp64 sum| <= 1e-6 * sum |x_r|
    s64 = np.sum([x.astype(np.float64) for x in Xh], axis=0)
    sabs = np.sum([np.abs(x.astype(np.float64)) for x in Xh], axis=0)
    got = res.outputs[0].cpu().numpy().astype(np.float64)
    assert np.all(np.abs(got - s64) <= 1e-6 * sabs + 1e-300)


def test_pooled_buffers_give_the_same_outputs(mods):
    """keep_messages=False (the timed configuration: a fixed pool of 2P message buffers) must not
    change any output."""
    pk, ring = mods
    cfg = _small(8, 2, 0.03, seed=7)
    Xh = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    sw = wl.nnz_switch_from_permille(n, 100)
    want, _ = ro.ring_all_reduce(Xh, sw, wl.nnz_switch_from_permille(n, 900))
    drv = ring.RingDriver(cfg.ranks, n, strategy="fused", keep_messages=False)
    Xd = [torch.from_numpy(x).cuda() for x in Xh]
    for _ in range(2):                                  # reuse of the pool across collectives
        res = drv.all_reduce(Xd, sw, wl.nnz_switch_from_permille(n, 900))
        torch.cuda.synchronize()
        for r in range(cfg.ranks):
            assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))


def test_ring_is_cuda_graph_capturable(mods):
    """The whole collective - per-rank streams, gated kernels, cooperative launches, workspace memsets - is
    captured into ONE CUDA graph; replays give the oracle's outputs again (no host decision inside)."""
    pk, ring = mods
    cfg = _small(4, 6, 0.03, seed=21)
    Xh = [b.numpy() for b in cfg.buffers()]
    n = cfg.chunk
    sw = wl.nnz_switch_from_permille(n, 70)
    want_out, _ = ro.ring_reduce_scatter(Xh, sw, keep_messages=False)
    X = [torch.from_numpy(v).cuda() for v in Xh]
    drv = ring.RingDriver(cfg.ranks, n)
    drv.reduce_scatter(X, sw)                       # warm-up outside the capture (lazy one-time setup)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        res = drv.reduce_scatter(X, sw)
    for _ in range(3):
        for o in res.outputs:
            o.fill_(7.0)
        g.replay()
        torch.cuda.synchronize()
        for r in range(cfg.ranks):
            assert np.array_equal(_u32(res.outputs[r]), want_out[r].view(np.uint32))


# ---------------------------------------------------------------------------------------------------
# The paper's adaptive policy on the device against
# oracle/ring_oracle.py ring_*_policy: formats, counts, decision sparsities (fp64, bit for bit) and every message.
# ---------------------------------------------------------------------------------------------------
def _check_policy_records(pk, res, log: ro.RingLog):
    fmts = res.formats()
    nnz = res.nnz.cpu().numpy().view(np.uint32)
    sigma = res.sigma.cpu().numpy()
    for rec, f in zip(res.records, fmts):
        e = log.at(rec.phase, rec.step, rec.rank)
        key = (rec.phase, rec.step, rec.rank)
        assert e.chunk == rec.chunk and e.fmt == f, (key, e.fmt, f)
        assert float(sigma[rec.fmt_index]) == e.extrapolated_sparsity, (key, sigma[rec.fmt_index], e.extrapolated_sparsity)
        assert int(nnz[rec.nnz_index]) == (e.nnz if e.nnz is not None else 0xFFFFFFFF), key
        if rec.msg is None or e.msg is None:
            continue
        if e.fmt == "pici":
            B, I, A = rec.msg.pici.to_host()
            w = e.msg.pici
            assert np.array_equal(I[:w.I.size], w.I) and np.array_equal(B[:w.B.size], w.B) and np.array_equal(A, w.A), key
        else:
            assert np.array_equal(_u32(rec.msg.dense), e.msg.dense.view(np.uint32)), key


def _disjoint_inputs(P=4, n=16384):
    """tests/golden/policy_sandwich_p4.txt: rank r holds a nonzero exactly where i mod 8 == r."""
    i = np.arange(P * n)
    return [np.where(i % 8 == r, (1.0 + 0.25 * r + (i % 97) / 128.0).astype(np.float32), np.float32(0.0)).astype(np.float32)
            for r in range(P)]


@pytest.mark.parametrize("strategy", ["fused", "paper"])
def test_policy_worked_example_sandwich(mods, strategy):
    """The hand-derived trace: a dense send sandwiched between sparse ones, re-calibrated counts."""
    pk, ring = mods
    Xh = _disjoint_inputs()
    pol = ro.Policy(0.8, 0.6, 0.1, 2)
    want, log, _, _ = ro.ring_reduce_scatter_policy(Xh, pol)
    drv = ring.RingDriver(4, 16384, strategy=strategy, keep_messages=True, policy=ring.Policy(0.8, 0.6, 0.1, 2))
    res = drv.reduce_scatter([torch.from_numpy(x).cuda() for x in Xh])
    torch.cuda.synchronize()
    _check_policy_records(pk, res, log)
    assert [f for rec, f in zip(res.records, res.formats()) if rec.chunk == 0] == ["pici", "dense", "pici"]
    for r in range(4):
        assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))


@pytest.mark.parametrize("strategy", ["fused", "paper"])
@pytest.mark.parametrize("P,rpn,intra,inter,ag", [(4, 2, 0.6, 0.5, 0.1), (8, 2, 0.93, 0.2, 0.85), (8, 4, 0.9, 0.99, 0.5),
                                                  (3, 2, 0.0, 0.0, 0.0), (2, 1, 1.0, 1.0, 1.0), (8, 2, 0.95, 0.9, 0.7)])
def test_policy_collectives_message_by_message(mods, strategy, P, rpn, intra, inter, ag):
    pk, ring = mods
    cfg = wl.RingConfig("small", P, P * 5 * wl.TILE, 0.02, 0.03, "normal", 1.0, 11 + P)
    Xh = [b.numpy() for b in cfg.buffers()]
    Xd = [torch.from_numpy(x).cuda() for x in Xh]
    n = cfg.chunk
    pol = ro.Policy(intra, inter, ag, rpn)
    want, log, _, _ = ro.ring_reduce_scatter_policy(Xh, pol)
    drv = ring.RingDriver(P, n, strategy=strategy, keep_messages=True, policy=ring.Policy(intra, inter, ag, rpn))
    res = drv.reduce_scatter(Xd)
    torch.cuda.synchronize()
    _check_policy_records(pk, res, log)
    fold = ro.reduce_scatter_definition(Xh)
    for r in range(P):
        assert np.array_equal(_u32(res.outputs[r]), want[r].view(np.uint32))
        assert np.array_equal(_u32(res.outputs[r]), fold[r].view(np.uint32))
    # all-reduce: the ag_thresh decision and the gathered result
    want_ar, log_ar = ro.ring_all_reduce_policy(Xh, pol)
    res = drv.all_reduce(Xd)
    torch.cuda.synchronize()
    _check_policy_records(pk, res, log_ar)
    for r in range(P):
        assert np.array_equal(_u32(res.outputs[r]), want_ar[r].view(np.uint32))


def test_ring_engine_launch_count_and_reuse(mods):
    """One launch per kernel family per ring step, whatever P is; the arena is reusable without clearing."""
    pk, ring = mods
    for P in (4, 8):
        cfg = _small(P, 4, 0.05, seed=2)
        Xd = [b.cuda() for b in cfg.buffers()]
        drv = ring.RingDriver(P, cfg.chunk, strategy="fused")
        sw = wl.nnz_switch_from_permille(cfg.chunk, 120)
        first = drv.reduce_scatter(Xd, sw)
        assert first.launches == 3 + 5 * (P - 2) + 2                 # step 0: 3, middle steps: 5, last step: 2
        ref = [o.clone() for o in first.outputs]
        for _ in range(3):
            again = drv.reduce_scatter(Xd, sw)
            torch.cuda.synchronize()
            assert all(torch.equal(a.view(torch.int32), b.view(torch.int32)) for a, b in zip(again.outputs, ref))
