"""SpCCL's sparse ring collectives over REAL ranks: one process per GPU, variable-size Pici messages between ring
neighbours (PAPER.md:207-219 the ring algorithms, 263-275 the message protocol, 289-291 the
staging of received sparse data).  The per-element work is the C-ABI kernels (pici.py); this module is the host side:
framing, buffers, schedule, transport.

What the paper fixes and how it is mapped here
  * "we extend the Simple protocol by prepending a 48-byte header to all messages.  The header contains format and
    message size metadata, as well as offsets indicating where different components of our sparse formats begin"
      ->  `Header` below: 48 bytes, sent ahead of every payload.
  * "the collective cannot determine message sizes or message format in advance for any individual receipt ... we
    also enlarge the FIFO buffers to ensure that even a worst-case compressed slice fits"  ->  every
    receive buffer holds the worst case (B + I + n values); the payload that travels is B + I + the nnz values only.
  * "we first copy the received data into a staging buffer and perform the scatter-add from local memory"
      ->  the receive buffer IS local HBM (the transport's receive is the copy); kernels never read a
    peer's memory.
  * compression "at the slice level ... the slice is the unit of pipelining" with a block-local scan per segment
      ->  `segments`: a chunk is cut into S independent Pici objects (each with its own I), sent as S
    messages per ring step; the payload of segment j + 1 is in flight while segment j is reduced and recompressed.
  * schedule: NCCL's: rank r sends to r + 1, ends owning chunk r; sums in ring order
    acc = received + local, so the result equals oracle/ring_oracle.py bit for bit.
  * format switch: on the measured nnz (readings C9 #9/#10): a message travels dense once nnz >= nnz_switch, and a
    chunk that went dense stays dense for the rest of the reduce-scatter.

Transport: torch.distributed point-to-point.  With the NCCL backend device buffers are handed to isend / irecv
directly (NVLink 5 / NVSwitch inside a node).  With the gloo backend (the CPU test rig, and two processes sharing one
GPU) payloads are staged through pinned host memory.  A message's size is only known on the device, so the sender
reads nnz back before it can post the payload - one host synchronisation per message, which is what the header
round trip costs in this form (a peer-mapped FIFO written by the kernel, as NCCLX has it, would remove it).
"""
from __future__ import annotations

import struct
from dataclasses import dataclass, field

import torch
import torch.distributed as dist

TILE = 4096
FMT_PICI, FMT_DENSE = 0, 1
MAGIC = 0x49434950            # "PICI"
_HDR = struct.Struct("<IHHHHQQIIIQ")
HEADER_BYTES = _HDR.size
assert HEADER_BYTES == 48


@dataclass
class Header:
    fmt: int                  # FMT_PICI | FMT_DENSE
    dtype: int                # pici.F32
    step: int
    chunk: int                # chunk id * segments + segment
    n: int                    # elements the message stands for
    nnz: int                  # stored values (0xFFFF... for a dense message: no count is computed)
    off_B: int = 0            # byte offsets of the components inside the payload
    off_I: int = 0
    off_A: int = 0
    payload_bytes: int = 0

    def pack(self) -> bytes:
        return _HDR.pack(MAGIC, self.fmt, self.dtype, self.step, self.chunk, self.n, self.nnz, self.off_B, self.off_I,
                         self.off_A, self.payload_bytes)

    @staticmethod
    def unpack(raw: bytes) -> "Header":
        magic, fmt, dtype, step, chunk, n, nnz, oB, oI, oA, pb = _HDR.unpack(raw)
        if magic != MAGIC:
            raise RuntimeError("ring_dist: bad message header")
        return Header(fmt, dtype, step, chunk, n, nnz, oB, oI, oA, pb)


NO_COUNT = (1 << 64) - 1


@dataclass(frozen=True)
class Layout:
    """Byte layout of one Pici message of n elements inside its (worst-case sized) buffer."""
    n: int

    @property
    def T(self) -> int:
        return (self.n + TILE - 1) // TILE

    @property
    def off_B(self) -> int:
        return 0

    @property
    def off_I(self) -> int:
        return 512 * self.T

    @property
    def off_A(self) -> int:
        return self.off_I + ((4 * (self.T + 1) + 15) & ~15)

    @property
    def capacity_bytes(self) -> int:          # worst case: every element stored
        return self.off_A + 4 * self.n

    def payload_bytes(self, nnz: int) -> int:
        return self.off_A + 4 * nnz

    def header(self, step: int, chunk: int, nnz: int) -> Header:
        return Header(FMT_PICI, 0, step, chunk, self.n, nnz, self.off_B, self.off_I, self.off_A, self.payload_bytes(nnz))

    def dense_header(self, step: int, chunk: int) -> Header:
        return Header(FMT_DENSE, 0, step, chunk, self.n, NO_COUNT, 0, 0, 0, 4 * self.n)


def rs_chunk(rank: int, step: int, P: int) -> int:
    """Reduce-scatter: the chunk rank `rank` SENDS at step `step` (0 .. P-2) = the one it reduced at that step
    (step 0: its own contribution to chunk rank-1).  Rank r receives chunk rs_chunk(r-1, s-1) at step s."""
    return (rank - 1 - step) % P


def ag_chunk(rank: int, step: int, P: int) -> int:
    """All-gather: the shard rank `rank` sends at step `step` (0 .. P-2): its own at step 0, then what it received."""
    return (rank - step) % P


class Transport:
    """Point-to-point exchange with the ring neighbours.  `staged`: payloads go through pinned host buffers (gloo)."""

    def __init__(self, group=None, staged: bool | None = None):
        self.group = group
        self.rank = dist.get_rank(group)
        self.P = dist.get_world_size(group)
        self.next = dist.get_global_rank(group, (self.rank + 1) % self.P) if group is not None else (self.rank + 1) % self.P
        self.prev = dist.get_global_rank(group, (self.rank - 1) % self.P) if group is not None else (self.rank - 1) % self.P
        self.staged = (dist.get_backend(group) != "nccl") if staged is None else staged
        self._pin: dict[tuple[str, int], torch.Tensor] = {}

    def _host(self, kind: str, slot: int, nbytes: int) -> torch.Tensor:
        key = (kind, slot)
        buf = self._pin.get(key)
        if buf is None or buf.numel() < nbytes:
            buf = torch.empty(max(nbytes, 64), dtype=torch.uint8)
            if torch.cuda.is_available():
                buf = buf.pin_memory()
            self._pin[key] = buf
        return buf[:nbytes]

    def _post(self, send: torch.Tensor, recv: torch.Tensor):
        if dist.get_backend(self.group) == "nccl":
            return dist.batch_isend_irecv([dist.P2POp(dist.isend, send, self.next, self.group),
                                           dist.P2POp(dist.irecv, recv, self.prev, self.group)])
        return [dist.isend(send, self.next, self.group), dist.irecv(recv, self.prev, self.group)]

    def exchange(self, send: torch.Tensor, recv: torch.Tensor, slot: int = 0):
        """Post `send` (uint8 view, exact size) to the next rank and `recv` (uint8 view, exact size) from the previous
        one; returns a callable that completes both (and, when staged, lands the bytes in `recv`)."""
        if not (self.staged and send.is_cuda):
            works = self._post(send, recv)

            def done():
                for w in works:
                    w.wait()
            return done
        hs, hr = self._host("s", slot, send.numel()), self._host("r", slot, recv.numel())
        hs.copy_(send)                                   # device -> pinned host (synchronises the producing stream)
        works = self._post(hs, hr)

        def done():
            for w in works:
                w.wait()
            recv.copy_(hr, non_blocking=True)
            torch.cuda.current_stream().synchronize()    # the pinned buffer is reused by the next message
        return done

    def exchange_headers(self, hdr: Header, device) -> Header:
        raw = torch.frombuffer(bytearray(hdr.pack()), dtype=torch.uint8)
        got = torch.empty(HEADER_BYTES, dtype=torch.uint8)
        if not self.staged:                              # NCCL moves device memory only
            raw, got = raw.to(device), got.to(device)
        for w in self._post(raw, got):
            w.wait()
        return Header.unpack(got.cpu().numpy().tobytes())


@dataclass
class Sent:
    phase: str
    step: int
    segment: int
    chunk: int
    fmt: int
    nnz: int | None
    payload_bytes: int
    copy: tuple | None = None      # keep_messages: (B, I, A) numpy arrays or the dense numpy array


@dataclass
class DistLog:
    sent: list[Sent] = field(default_factory=list)

    def bytes_sent(self) -> int:
        return sum(s.payload_bytes + HEADER_BYTES for s in self.sent)


class _Msg:
    """One message buffer (worst-case sized, device) with Pici views over it and a dense view of its first 4 n bytes."""

    def __init__(self, pk, lay: Layout, device):
        self.lay = lay
        self.flat = torch.empty(lay.capacity_bytes, dtype=torch.uint8, device=device)
        B = self.flat[lay.off_B:lay.off_I].view(torch.int64)
        I = self.flat[lay.off_I:lay.off_I + 4 * (lay.T + 1)].view(torch.int32)
        A = self.flat[lay.off_A:lay.off_A + 4 * lay.n].view(torch.float32)
        self.pici = pk.Pici(lay.n, pk.F32, B, I, A)
        self.dense = self.flat[:4 * lay.n].view(torch.float32)
        self.fmt = FMT_PICI
        self.nnz = 0
        self.dense_src: torch.Tensor | None = None     # a dense message may be sent straight from another buffer

    def payload(self) -> torch.Tensor:
        if self.fmt == FMT_DENSE:
            src = self.dense if self.dense_src is None else self.dense_src
            return src.view(torch.uint8)
        return self.flat[:self.lay.payload_bytes(self.nnz)]


class DistRing:
    """Ring reduce-scatter / all-gather / all-reduce of fp32 buffers over the ranks of a process group."""

    def __init__(self, chunk: int, device, group=None, strategy: str = "paper", segments: int = 1,
                 keep_messages: bool = False, staged: bool | None = None):
        from . import pici as pk
        pk.lib()
        assert strategy in ("paper", "fused") and chunk % (segments * TILE) == 0
        self.pk, self.device, self.strategy, self.S, self.keep = pk, device, strategy, segments, keep_messages
        self.tp = Transport(group, staged)
        self.rank, self.P = self.tp.rank, self.tp.P
        self.n, self.sn = chunk, chunk // segments
        self.lay = Layout(self.sn)
        mk = lambda: [_Msg(pk, self.lay, device) for _ in range(segments)]
        self.out_msg = [mk(), mk()]                     # what this rank sends: double-buffered by step parity
        self.in_msg = [mk(), mk()]                      # what it receives
        self.acc = [[torch.empty(self.sn, dtype=torch.float32, device=device) for _ in range(segments)] for _ in range(2)]
        self.loc = pk.alloc_pici(self.sn, pk.F32, device) if strategy == "fused" else None
        self.ws = pk.alloc_workspace(self.sn, device)
        self.log = DistLog()

    # ---- helpers -------------------------------------------------------------------------------------------
    def _seg(self, x: torch.Tensor, chunk: int, g: int) -> torch.Tensor:
        lo = chunk * self.n + g * self.sn
        return x[lo:lo + self.sn]

    def _record(self, phase: str, step: int, g: int, chunk: int, m: _Msg):
        copy = None
        if self.keep:
            copy = m.pici.to_host() if m.fmt == FMT_PICI else (m.payload().view(torch.float32).cpu().numpy().copy(),)
        self.log.sent.append(Sent(phase, step, g, chunk, m.fmt, m.nnz if m.fmt == FMT_PICI else None,
                                  m.payload().numel(), copy))

    def _encode(self, dense: torch.Tensor, m: _Msg, nnz_switch: int):
        """compress `dense` into m; the message travels dense (straight from `dense`) once nnz >= nnz_switch."""
        self.pk.compress(dense, m.pici, self.ws)
        m.nnz = m.pici.nnz_host()                       # the size of the send is decided on the host
        m.fmt = FMT_DENSE if m.nnz >= nnz_switch else FMT_PICI
        m.dense_src = dense if m.fmt == FMT_DENSE else None

    def _swap(self, phase: str, step: int, send: list[_Msg], recv: list[_Msg], chunk_out: int):
        """One ring step of the transport: headers, then payloads, segment by segment; returns per-segment waiters so
        that segment g + 1 is in flight while segment g is processed."""
        waits = []
        for g, (ms, mr) in enumerate(zip(send, recv)):
            hdr = (self.lay.header(step, chunk_out * self.S + g, ms.nnz) if ms.fmt == FMT_PICI
                   else self.lay.dense_header(step, chunk_out * self.S + g))
            self._record(phase, step, g, chunk_out, ms)
            got = self.tp.exchange_headers(hdr, self.device)
            assert got.n == self.sn and got.step == step
            mr.fmt, mr.nnz, mr.dense_src = got.fmt, (got.nnz if got.fmt == FMT_PICI else 0), None
            waits.append(self.tp.exchange(ms.payload(), mr.flat[:got.payload_bytes], slot=g))
        return waits

    # ---- collectives ---------------------------------------------------------------------------------------
    def reduce_scatter(self, x: torch.Tensor, out: torch.Tensor, nnz_switch: int | None = None) -> torch.Tensor:
        """x: this rank's P * chunk elements; out: chunk elements = the reduced chunk `rank` (ring-order sum)."""
        pk, P, r, S = self.pk, self.P, self.rank, self.S
        assert x.numel() == P * self.n and out.numel() == self.n and x.dtype == torch.float32
        sw = self.sn + 1 if nnz_switch is None else nnz_switch
        cur = self.out_msg[0]
        c0 = rs_chunk(r, 0, P)
        for g in range(S):                               # step 0 always compresses
            self._encode(self._seg(x, c0, g), cur[g], sw)
        for s in range(1, P):
            c = rs_chunk(r, s, P)                        # the chunk received and reduced at this step
            rcv, nxt, acc = self.in_msg[s & 1], self.out_msg[s & 1], self.acc[s & 1]
            waits = self._swap("rs", s - 1, cur, rcv, rs_chunk(r, s - 1, P))
            last = s == P - 1
            for g in range(S):
                local = self._seg(x, c, g)
                if self.strategy == "fused" and not last:
                    pk.compress(local, self.loc, self.ws)          # independent of the message: overlaps its transfer
                waits[g]()
                m, o = rcv[g], nxt[g]
                dst = out[g * self.sn:(g + 1) * self.sn] if last else acc[g]
                if m.fmt == FMT_DENSE:                   # once dense, the chunk stays dense (C8)
                    pk.dense_add(m.dense, local, dst)
                    o.fmt, o.nnz, o.dense_src = FMT_DENSE, 0, dst
                elif last:
                    pk.reduce_sd_out(m.pici, local, dst)
                elif self.strategy == "fused":           # sparse + sparse merge, no dense scratch
                    pk.reduce_ss(m.pici, self.loc, o.pici, self.ws)
                    o.nnz = o.pici.nnz_host()
                    o.fmt, o.dense_src = FMT_PICI, None
                    if o.nnz >= sw:
                        pk.decompress(o.pici, dst)
                        o.fmt, o.dense_src = FMT_DENSE, dst
                else:                                    # the paper's step: scatter-add into dense, recompress
                    pk.reduce_sd_out(m.pici, local, dst)
                    self._encode(dst, o, sw)
            cur = nxt
        if x.is_cuda:
            torch.cuda.current_stream().synchronize()
        return out

    def all_gather(self, shard: torch.Tensor, out: torch.Tensor, nnz_switch: int | None = None, phase: str = "ag") -> torch.Tensor:
        """shard: this rank's chunk elements; out: P * chunk elements, identical on every rank."""
        pk, P, r, S = self.pk, self.P, self.rank, self.S
        assert shard.numel() == self.n and out.numel() == P * self.n
        sw = self.sn + 1 if nnz_switch is None else nnz_switch
        cur = self.out_msg[0]
        for g in range(S):                               # compress once, forward unchanged
            self._encode(shard[g * self.sn:(g + 1) * self.sn], cur[g], sw)
        out[r * self.n:(r + 1) * self.n].copy_(shard)    # own slot: plain copy (C9 #12)
        other = self.in_msg[0]
        for s in range(1, P):
            c = ag_chunk(r, s, P)
            rcv = other
            waits = self._swap(phase, s - 1, cur, rcv, ag_chunk(r, s - 1, P))
            for g in range(S):
                waits[g]()                               # completes the send of cur[g] as well
                m = rcv[g]
                dst = self._seg(out, c, g)
                if m.fmt == FMT_DENSE:
                    pk.dense_copy(m.dense, dst)
                else:
                    pk.decompress(m.pici, dst)
            cur, other = rcv, cur                        # forwarded unchanged at the next step
        if out.is_cuda:
            torch.cuda.current_stream().synchronize()
        return out

    def all_reduce(self, x: torch.Tensor, out: torch.Tensor, nnz_switch_rs: int | None = None,
                   nnz_switch_ag: int | None = None) -> torch.Tensor:
        """RS, then the reduced chunk re-decides its format with the all-gather threshold, then AG."""
        red = out[self.rank * self.n:(self.rank + 1) * self.n]
        self.reduce_scatter(x, red, nnz_switch_rs)
        shard = red.clone()
        return self.all_gather(shard, out, nnz_switch_ag, phase="ar.ag")
