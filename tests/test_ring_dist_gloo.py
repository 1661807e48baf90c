"""Host logic of the real multi-rank ring (paper_2607_04676_b200/ring_dist.py) on CPU: the 48-byte
header, the message layout against the format's sizes, the ring schedule, and a world-size-2 / 3 gloo run
of the transport that moves framed variable-size messages round the ring.  No CUDA, no kernels: payloads are bytes."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import pici_oracle as po
from paper_2607_04676_b200 import ring_dist as rd


def test_header_is_48_bytes_and_round_trips():
    assert rd.HEADER_BYTES == 48
    lay = rd.Layout(3 * 4096)
    for h in (lay.header(5, 17, 1234), lay.dense_header(2, 3), rd.Header(0, 0, 65535, 65535, (1 << 32) - 1, (1 << 32) - 1, 1, 2, 3, 1 << 40)):
        raw = h.pack()
        assert len(raw) == 48 and rd.Header.unpack(raw) == h
    with pytest.raises(RuntimeError):
        rd.Header.unpack(b"\0" * 48)


@pytest.mark.parametrize("n", [4096, 8192, 5 * 4096, 1 << 20])
def test_layout_matches_the_format(n):
    """Payload = B (512 T bytes) + I (4 (T + 1), padded to 16) + 4 nnz: the oracle's message size plus the padding; the
    receive buffer holds the worst case."""
    lay = rd.Layout(n)
    T = n // 4096
    x = np.zeros(n, np.float32)
    x[::37] = 1.0
    p = po.compress(x, "f32")
    pad = (-(4 * (T + 1))) % 16
    assert lay.off_I == p.B.nbytes and lay.off_A == p.B.nbytes + p.I.nbytes + pad
    assert lay.payload_bytes(p.nnz) == p.message_bytes() + pad
    assert lay.capacity_bytes == lay.payload_bytes(n) and lay.off_A % 16 == 0
    assert lay.dense_header(0, 0).payload_bytes == 4 * n


@pytest.mark.parametrize("P", [2, 3, 4, 8, 16])
def test_schedule_is_consistent(P):
    """What rank r sends at step s is what rank r + 1 expects at step s + 1; reduce-scatter ends with chunk r on rank
    r after every rank has contributed once; all-gather visits every slot once."""
    for r in range(P):
        for s in range(P - 1):
            assert rd.rs_chunk(r, s, P) == rd.rs_chunk((r + 1) % P, s + 1, P)
            assert rd.ag_chunk(r, s, P) == rd.ag_chunk((r + 1) % P, s + 1, P)
        assert rd.rs_chunk(r, 0, P) == (r - 1) % P and rd.rs_chunk(r, P - 1, P) == r
        assert sorted(rd.ag_chunk(r, s, P) for s in range(P)) == list(range(P))
    for c in range(P):                                                 # chunk c is started by rank c + 1 and passes every rank
        holders = [r for s in range(P) for r in range(P) if rd.rs_chunk(r, s, P) == c]
        assert sorted(holders) == list(range(P))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _payload(rank: int, step: int, nbytes: int) -> torch.Tensor:
    g = torch.Generator().manual_seed(1000 * rank + step)
    return torch.randint(0, 256, (nbytes,), dtype=torch.uint8, generator=g)


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        tp = rd.Transport()
        lay = rd.Layout(8 * 4096)
        recv = torch.zeros(lay.capacity_bytes, dtype=torch.uint8)
        ok = tp.staged and tp.next == (rank + 1) % world and tp.prev == (rank - 1) % world
        prev = (rank - 1) % world
        for step in range(5):                                          # sizes differ per rank and step, known to the sender only
            nnz = 100 * (rank + 1) + 7 * step
            dense = step == 3 and rank == 0
            hdr = lay.dense_header(step, rank) if dense else lay.header(step, rank, nnz)
            send = _payload(rank, step, hdr.payload_bytes)
            got = tp.exchange_headers(hdr, "cpu")
            pn = 100 * (prev + 1) + 7 * step
            want = lay.dense_header(step, prev) if (step == 3 and prev == 0) else lay.header(step, prev, pn)
            ok = ok and got == want
            tp.exchange(send, recv[:got.payload_bytes])()
            ok = ok and torch.equal(recv[:got.payload_bytes], _payload(prev, step, got.payload_bytes))
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_framed_messages_go_round_the_ring_gloo(world):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]
