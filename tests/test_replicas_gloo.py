"""N > 1 host logic on CPU: world_size-2 gloo run of the replicas plumbing bench.py uses (max-over-ranks
timing, summed units, distinct per-replica seeds).  No CUDA involved."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as wl
from paper_2607_04676_b200 import replicas


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
        thr, ms_max = replicas.whole_job_throughput(1000.0 * (rank + 1), ms)
        seeds = replicas.rank_seeds(0, rank, 2)
        x = wl.sparse_buffer(8192, 0.05, seed=seeds[0])
        g = [torch.zeros(8192) for _ in range(world)]
        dist.all_gather(g, x)
        q.put((rank, thr, ms_max, seeds, bool(torch.equal(g[0], g[1]))))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, thr, ms_max, seeds, same in res:
        assert ms_max == 20.0                        # max over ranks
        assert abs(thr - 3000.0 / 0.020) < 1e-6     # sum of units / max time
        assert not same                              # replicas draw different buffers
    assert set(res[0][3]).isdisjoint(res[1][3])


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_throughput(10.0, 5.0) == (2000.0, 5.0)
    assert replicas.rank_seeds(0, 0, 2) == [wl.stream_seed(0, 0), wl.stream_seed(0, 1)]
    # no two (config seed, replica) pairs share a stream: replica 1 of seed 0 is not replica 0 of seed 1
    seen = [tuple(replicas.rank_seeds(S, r, 8)) for S in range(6) for r in range(8)]
    flat = [v for t in seen for v in t]
    assert len(set(flat)) == len(flat)
