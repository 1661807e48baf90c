"""Ring collectives over P LOGICAL ranks held as separate buffers in one B200's HBM (BASELINE.json north_star;
SURVEY.md S8(a) a9, S8(c) C8): a thin binding of the C ring engine (include/pici.h "Ring engine",
csrc/ring.cu).  No NCCL, no inter-GPU traffic: a "send" is a pointer hand-off inside the engine's arena.

This file marshals arguments and exposes the engine's log - it enqueues nothing itself.  One call =
one C call = the whole collective on the current stream: one kernel launch per kernel family per ring step
(each launch handles all P ranks' jobs), every format decision taken on the device.

    drv = RingDriver(P, n, strategy="fused" | "paper", keep_messages=False, policy=None | Policy(...))
    res = drv.reduce_scatter(X, nnz_switch)          # X[r]: rank r's P*n fp32 elements -> res.outputs[r]: chunk r
    res = drv.all_gather(shards, nnz_switch=None)    # -> res.outputs[r]: P*n elements, identical on every rank
    res = drv.all_reduce(X, nnz_switch_rs, nnz_switch_ag)

policy=None decides on the MEASURED nnz (a message travels dense once nnz >= nnz_switch, PAPER.md:227 with the
readings C9 #9/#10); policy=Policy(intra, inter, ag, ranks_per_node) is the paper's adaptive rule (Eq. 7
extrapolation, link-aware and phase-aware thresholds) and ignores the nnz_switch arguments.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass, field

import torch

from . import pici as pk

FUSED, PAPER = 0, 1
MEASURED, POLICY = 0, 1
NO_COUNT = 0xFFFFFFFF


class _Config(ctypes.Structure):
    _fields_ = [("ranks", ctypes.c_int32), ("strategy", ctypes.c_int32), ("decision", ctypes.c_int32),
                ("keep_messages", ctypes.c_int32), ("chunk", ctypes.c_uint64), ("nnz_switch_rs", ctypes.c_uint64),
                ("nnz_switch_ag", ctypes.c_uint64), ("intra_thresh", ctypes.c_double), ("inter_thresh", ctypes.c_double),
                ("ag_thresh", ctypes.c_double), ("ranks_per_node", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class _Layout(ctypes.Structure):
    _fields_ = [(k, ctypes.c_uint64) for k in
                ("records", "rs_records", "off_fmt", "off_nnz", "off_sigma", "off_messages", "message_bytes", "message_I",
                 "message_A", "message_dense", "off_reduced", "reduced_bytes", "slots")]


@dataclass
class Policy:
    """The paper's thresholds (sparsities): PAPER.md:237 intra 0.6 / inter 0.5 (Pici, fp32 RS), :239 ag 0.1."""
    intra_thresh: float = 0.6
    inter_thresh: float = 0.5
    ag_thresh: float = 0.1
    ranks_per_node: int = 2


@dataclass
class _Msg:
    pici: pk.Pici
    dense: torch.Tensor


@dataclass
class StepRecord:
    phase: str
    step: int
    rank: int
    chunk: int
    msg: _Msg | None          # views of the message's slot in the arena (keep_messages only)
    fmt_index: int            # index of its format word / nnz / decision sparsity in the log arrays
    nnz_index: int


@dataclass
class RingResult:
    outputs: list[torch.Tensor]
    records: list[StepRecord] = field(default_factory=list)
    fmt: torch.Tensor | None = None       # int32 format words, one per record index (device)
    nnz: torch.Tensor | None = None       # int32 (uint32 bits) measured nnz; NO_COUNT after a dense send
    sigma: torch.Tensor | None = None     # float64 decision sparsities (policy mode)
    launches: int = 0                     # kernel launches the collective enqueued

    def formats(self) -> list[str]:
        f = self.fmt.cpu().tolist()
        return ["dense" if f[r.fmt_index] == pk.FMT_DENSE else "pici" for r in self.records]

    def switch_steps(self, phase: str = "rs") -> dict[int, int | None]:
        """chunk -> first step of `phase` whose message travelled dense (None = never)."""
        out: dict[int, int | None] = {}
        for rec, f in zip(self.records, self.formats()):
            if rec.phase != phase:
                continue
            out.setdefault(rec.chunk, None)
            if f == "dense" and out[rec.chunk] is None:
                out[rec.chunk] = rec.step
        return out


def _ptr_array(tensors) -> ctypes.Array:
    return (ctypes.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


class RingDriver:
    """Arena + configuration for P logical ranks with chunk length n (elements, multiple of 4096), fp32."""

    def __init__(self, ranks: int, chunk: int, device="cuda", strategy: str = "fused", keep_messages: bool = False,
                 policy: Policy | None = None, concurrent: bool = True):
        assert chunk % pk.TILE == 0 and ranks >= 2 and strategy in ("fused", "paper")
        del concurrent   # the engine batches the ranks of a step into one launch; kept for call compatibility
        self.P, self.n, self.device, self.strategy, self.keep, self.policy = ranks, chunk, device, strategy, keep_messages, policy
        self.cfg = _Config(ranks, FUSED if strategy == "fused" else PAPER, MEASURED if policy is None else POLICY,
                           1 if keep_messages else 0, chunk, chunk + 1, chunk + 1,
                           policy.intra_thresh if policy else 0.0, policy.inter_thresh if policy else 0.0,
                           policy.ag_thresh if policy else 0.0, policy.ranks_per_node if policy else 1, 0)
        L = pk.lib()
        nbytes = ctypes.c_uint64()
        pk._check(L.pici_ring_arena_bytes(ctypes.byref(self.cfg), ctypes.byref(nbytes)), "pici_ring_arena_bytes")
        self.layout = _Layout()
        pk._check(L.pici_ring_layout(ctypes.byref(self.cfg), ctypes.byref(self.layout)), "pici_ring_layout")
        self.arena = torch.empty(int(nbytes.value), dtype=torch.uint8, device=device)
        pk._check(L.pici_workspace_init(self.arena.data_ptr(), self.arena.numel(), pk._stream()), "pici_workspace_init")
        lay, R = self.layout, int(self.layout.records)
        self.fmt = self.arena[lay.off_fmt:lay.off_fmt + 4 * R].view(torch.int32)
        self.nnz = self.arena[lay.off_nnz:lay.off_nnz + 4 * R].view(torch.int32)
        self.sigma = self.arena[lay.off_sigma:lay.off_sigma + 8 * R].view(torch.float64)

    # ------------------------------------------------------------------------------------------
    def _message(self, slot: int, dense_alias: torch.Tensor | None = None) -> _Msg:
        lay, n = self.layout, self.n
        T = n // pk.TILE
        o = int(lay.off_messages + slot * lay.message_bytes)
        view = lambda off, nbytes, dt: self.arena[o + off:o + off + nbytes].view(dt)
        p = pk.Pici(n, pk.F32, view(0, 64 * T * 8, torch.int64), view(int(lay.message_I), (T + 1) * 4, torch.int32),
                    view(int(lay.message_A), n * 4, torch.float32))
        return _Msg(p, dense_alias if dense_alias is not None else view(int(lay.message_dense), n * 4, torch.float32))

    def _records(self, res: RingResult, phase: str, shards=None) -> None:
        P = self.P
        if phase == "rs":
            for s in range(P - 1):
                for r in range(P):
                    idx = s * P + r
                    res.records.append(StepRecord("rs", s, r, (r - 1 - s) % P, self._message(idx) if self.keep else None, idx, idx))
        else:
            for r in range(P):
                idx = int(self.layout.rs_records) + r
                # a dense all-gather message aliases the shard itself (no copy is made)
                msg = self._message(idx, shards[r]) if self.keep else None
                res.records.append(StepRecord(phase, 0, r, r, msg, idx, idx))

    def _call(self, fn, a, b) -> int:
        launches = ctypes.c_int()
        pk._check(fn(ctypes.byref(self.cfg), _ptr_array(a), _ptr_array(b), self.arena.data_ptr(), self.arena.numel(),
                     ctypes.byref(launches), pk._stream()), fn.__name__)
        return int(launches.value)

    def _result(self, outs, launches) -> RingResult:
        return RingResult(outs, [], self.fmt, self.nnz, self.sigma, launches)

    # ------------------------------------------------------------------------------------------
    def reduce_scatter(self, X: list[torch.Tensor], nnz_switch: int | None = None,
                       outputs: list[torch.Tensor] | None = None) -> RingResult:
        """X[r]: rank r's N = P*n element fp32 buffer.  Returns outputs[r] = reduced chunk r (n elements)."""
        P, n = self.P, self.n
        assert len(X) == P and all(x.numel() == P * n and x.dtype == torch.float32 and x.is_cuda and x.is_contiguous() for x in X)
        outs = outputs or [torch.empty(n, dtype=torch.float32, device=self.device) for _ in range(P)]
        self.cfg.nnz_switch_rs = int(nnz_switch) if nnz_switch is not None else n + 1
        res = self._result(outs, self._call(pk.lib().pici_ring_reduce_scatter, X, outs))
        self._records(res, "rs")
        return res

    def all_gather(self, shards: list[torch.Tensor], nnz_switch: int | None = None,
                   outputs: list[torch.Tensor] | None = None) -> RingResult:
        """shards[r]: rank r's n-element shard.  outputs[r]: P*n elements, identical on every rank."""
        P, n = self.P, self.n
        assert len(shards) == P and all(x.numel() == n and x.dtype == torch.float32 and x.is_cuda and x.is_contiguous() for x in shards)
        outs = outputs or [torch.empty(P * n, dtype=torch.float32, device=self.device) for _ in range(P)]
        self.cfg.nnz_switch_ag = int(nnz_switch) if nnz_switch is not None else n + 1
        res = self._result(outs, self._call(pk.lib().pici_ring_all_gather, shards, outs))
        self._records(res, "ag", shards)
        return res

    def all_reduce(self, X: list[torch.Tensor], nnz_switch_rs: int | None = None, nnz_switch_ag: int | None = None,
                   outputs: list[torch.Tensor] | None = None) -> RingResult:
        """RS, then the ag_thresh decision on each reduced chunk, then AG."""
        P, n = self.P, self.n
        assert len(X) == P and all(x.numel() == P * n and x.dtype == torch.float32 and x.is_cuda and x.is_contiguous() for x in X)
        outs = outputs or [torch.empty(P * n, dtype=torch.float32, device=self.device) for _ in range(P)]
        self.cfg.nnz_switch_rs = int(nnz_switch_rs) if nnz_switch_rs is not None else n + 1
        self.cfg.nnz_switch_ag = int(nnz_switch_ag) if nnz_switch_ag is not None else n + 1
        res = self._result(outs, self._call(pk.lib().pici_ring_all_reduce, X, outs))
        lay = self.layout
        reduced = [self.arena[lay.off_reduced + r * lay.reduced_bytes:lay.off_reduced + r * lay.reduced_bytes + 4 * n].view(torch.float32)
                   for r in range(P)]
        self._records(res, "rs")
        self._records(res, "ar.ag", reduced)
        return res
