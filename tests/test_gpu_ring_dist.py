"""The real multi-rank ring (ring_dist.py) run by SEVERAL PROCESSES against the oracle's ring.
This box has one GPU, so the ranks share cuda:0 and talk over gloo with payloads staged through pinned host memory
(the transport's non-NCCL path); no kernel of one rank ever waits for a kernel of another - every wait is a host-side
receive.  Outputs are compared bit for bit with oracle/ring_oracle.py, and with one segment per chunk every message
(format, nnz, B, I, A) with the oracle's log."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as wl
from oracle import ring_oracle as ro

pytestmark = pytest.mark.gpu


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q, case):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2607_04676_b200 import ring_dist as rd
        torch.cuda.set_device(0)
        coll, strategy, segments, chunk, density, sw_rs, sw_ag = case
        cfg = wl.RingConfig("dist", world, world * chunk, 0.0, density, "normal", 1.0, 3)
        x = cfg.buffers()[rank].cuda()
        ring = rd.DistRing(chunk, "cuda", strategy=strategy, segments=segments, keep_messages=(segments == 1))
        if coll == "rs":
            out = torch.full((chunk,), 7.0, device="cuda")
            ring.reduce_scatter(x, out, sw_rs)
        elif coll == "ag":
            out = torch.full((world * chunk,), 7.0, device="cuda")
            ring.all_gather(x[rank * chunk:(rank + 1) * chunk].contiguous(), out, sw_ag)
        else:
            out = torch.full((world * chunk,), 7.0, device="cuda")
            ring.all_reduce(x, out, sw_rs, sw_ag)
        sent = [(s.phase, s.step, s.segment, s.chunk, s.fmt, s.nnz, s.payload_bytes, s.copy) for s in ring.log.sent]
        q.put((rank, out.cpu().numpy(), sent))
    finally:
        dist.destroy_process_group()


def _run(world, case):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q, case)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in ps:
        p.join(120)
        assert p.exitcode == 0
    return res


CASES = [
    # collective, strategy, segments, chunk, density, nnz_switch_rs, nnz_switch_ag
    (2, ("rs", "paper", 1, 8 * 4096, 0.05, None, None)),
    (2, ("rs", "fused", 1, 8 * 4096, 0.05, None, None)),
    (3, ("rs", "paper", 1, 4 * 4096, 0.10, int(0.15 * 4 * 4096), None)),     # switches to dense on the way
    (3, ("rs", "fused", 2, 4 * 4096, 0.10, int(0.15 * 2 * 4096), None)),     # two segments per chunk
    (3, ("ag", "paper", 1, 4 * 4096, 0.02, None, None)),
    (2, ("ag", "paper", 2, 8 * 4096, 0.60, None, int(0.5 * 4 * 4096))),      # dense shards
    (3, ("ar", "paper", 1, 4 * 4096, 0.10, int(0.15 * 4 * 4096), int(0.9 * 4 * 4096))),
    (2, ("ar", "fused", 4, 16 * 4096, 0.01, None, None)),
]


@pytest.mark.timeout(600)
@pytest.mark.parametrize("world,case", CASES)
def test_multi_process_ring_matches_oracle(world, case):
    coll, strategy, segments, chunk, density, sw_rs, sw_ag = case
    cfg = wl.RingConfig("dist", world, world * chunk, 0.0, density, "normal", 1.0, 3)
    X = [b.numpy() for b in cfg.buffers()]
    res = _run(world, case)
    never = chunk + 1
    if coll == "rs":
        want, log = ro.ring_reduce_scatter(X, never if sw_rs is None else sw_rs)
        for r, out, _ in res:
            assert np.array_equal(out.view(np.uint32), want[r].view(np.uint32))
    elif coll == "ag":
        shards = [np.ascontiguousarray(X[r][r * chunk:(r + 1) * chunk]) for r in range(world)]
        want, log = ro.ring_all_gather(shards, sw_ag)
        for r, out, _ in res:
            assert np.array_equal(out.view(np.uint32), want[r].view(np.uint32))
    else:
        want, log = ro.ring_all_reduce(X, never if sw_rs is None else sw_rs, never if sw_ag is None else sw_ag)
        for r, out, _ in res:
            assert np.array_equal(out.view(np.uint32), want[r].view(np.uint32))
        assert all(np.array_equal(res[0][1], o) for _, o, _ in res)              # every rank ends bit-identical
    if segments != 1:
        return
    # message by message (one segment per chunk = the oracle's messages)
    for r, _, sent in res:
        for phase, step, seg, ch, fmt, nnz, nbytes, copy in sent:
            e = log.at(phase, step, r)
            assert e.chunk == ch and (e.fmt == "dense") == (fmt == 1)
            if fmt == 0:
                assert nnz == e.msg.pici.nnz if e.msg is not None else True
                if e.msg is not None:
                    B, I, A = copy
                    T = chunk // 4096
                    assert np.array_equal(B[:64 * T], e.msg.pici.B) and np.array_equal(I[:T + 1], e.msg.pici.I)
                    assert np.array_equal(A, e.msg.pici.A)
            elif e.msg is not None and e.msg.dense is not None:
                assert np.array_equal(copy[0].view(np.uint32), e.msg.dense.view(np.uint32))
