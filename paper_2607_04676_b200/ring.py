"""Host driver: SpCCL's sparse ring collectives over P LOGICAL ranks held as separate buffers in one
B200's HBM (BASELINE.json north_star).  No NCCL, no inter-GPU traffic:
a "send" is a pointer hand-off.  This file is host logic only - every byte of data is touched by
the libpici_b200 kernels (through `pici`), and every format decision is taken ON THE DEVICE:

  * each message carries a device-side format word (PICI_FMT_PICI / PICI_FMT_DENSE, the fact the
    paper's 48-byte header carries);
  * for every step the driver enqueues both the sparse-path and the dense-path kernels, each gated
    on the incoming message's format word, so nothing is read back and no stream is synchronised
    until the caller asks for the log (SURVEY.md S7 hard part 6).

Schedule (NCCL's, inherited silently by the paper; S8(c) C8): rank r sends to r+1 and ends owning
chunk r.  reduce-scatter step 0 encodes chunk (r-1) mod P; at step s rank r receives chunk
(r-1-s) mod P, forms acc = received + local and, unless it is the last step, re-encodes.
Two equivalent ways to take the step, both bit-identical to the oracle's messages:
  strategy="paper": scatter-add the received Pici into a dense scratch (pici_reduce_sd), recompress
                    it (pici_compress), PAPER.md:219;
  strategy="fused": compress the local chunk and merge sparse+sparse (pici_reduce_ss), never
                    touching a dense buffer while the chunk stays sparse (north_star).
A chunk that reached nnz >= nnz_switch travels dense from then on (pici_maybe_densify, PAPER.md:227;
once dense it stays dense within the reduce-scatter, C8).

The P ranks' kernels of one ring step are independent of one another, and a chunk is a few thousand tiles -
too little to fill 148 SMs from one launch - so with concurrent=True every logical rank enqueues on its own
CUDA stream and the streams join after every step (SURVEY.md S7 hard part 5).  The whole collective can be
captured into ONE CUDA graph (the cross-stream events become graph edges): bench.py --ring times both.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import torch

from . import pici as pk


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
    msg: _Msg | None          # buffers holding the message sent at this step (valid until reused)
    fmt_index: int            # index of its format word in the driver's flag array
    nnz_index: int


@dataclass
class RingResult:
    outputs: list[torch.Tensor]
    records: list[StepRecord] = field(default_factory=list)
    fmt: torch.Tensor | None = None       # int32 flags, one per record (device)
    nnz: torch.Tensor | None = None       # int32 measured nnz, one per record (device)

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


class RingDriver:
    """Buffers for P logical ranks with chunk length n (elements, multiple of 4096), fp32."""

    def __init__(self, ranks: int, chunk: int, device="cuda", strategy: str = "fused", keep_messages: bool = False,
                 concurrent: bool = True):
        assert chunk % pk.TILE == 0 and ranks >= 2 and strategy in ("fused", "paper")
        self.P, self.n, self.device, self.strategy = ranks, chunk, device, strategy
        self.keep = keep_messages
        self.streams = [torch.cuda.Stream(device=device) for _ in range(ranks)] if concurrent else None
        self._ev_main = torch.cuda.Event()
        self._ev_rank = [torch.cuda.Event() for _ in range(ranks)]
        P = ranks
        n_sets = (2 * P) if not keep_messages else None
        self._pool: list[_Msg] = []
        self._n_sets = n_sets
        self._cursor = 0
        self.local = [pk.alloc_pici(chunk, pk.F32, device) for _ in range(P)] if strategy == "fused" else None
        self.ws = [pk.alloc_workspace(chunk, device) for _ in range(P)]
        max_records = 4 * P * P + 4 * P
        self.fmt = torch.zeros(max_records, dtype=torch.int32, device=device)
        self.nnz = torch.zeros(max_records, dtype=torch.int32, device=device)
        if n_sets is not None:
            for _ in range(n_sets):
                self._pool.append(self._new_msg())

    def _new_msg(self) -> _Msg:
        return _Msg(pk.alloc_pici(self.n, pk.F32, self.device), torch.empty(self.n, dtype=torch.float32, device=self.device))

    def _msg(self) -> _Msg:
        if self._n_sets is None:          # keep every message alive (tests compare them with the oracle's log)
            m = self._new_msg()
            self._pool.append(m)
            return m
        m = self._pool[self._cursor % self._n_sets]
        self._cursor += 1
        return m

    # ------------------------------------------------------------------------------------------
    def _step(self, body) -> None:
        """Run body(r) for every rank r: on rank r's own stream (all forked from the current stream, all joined
        back into it afterwards) when concurrent, else in order on the current stream."""
        if self.streams is None:
            for r in range(self.P):
                body(r)
            return
        main = torch.cuda.current_stream(self.device)
        self._ev_main.record(main)
        for r in range(self.P):
            st = self.streams[r]
            st.wait_event(self._ev_main)
            with torch.cuda.stream(st):
                body(r)
            self._ev_rank[r].record(st)
        for r in range(self.P):
            main.wait_event(self._ev_rank[r])

    def _begin(self) -> RingResult:
        res = RingResult([], [], self.fmt, self.nnz)
        return res

    def _record(self, res: RingResult, phase, step, rank, chunk, msg) -> StepRecord:
        idx = len(res.records)
        assert idx < self.fmt.numel()
        rec = StepRecord(phase, step, rank, chunk, msg if self.keep else None, idx, idx)
        res.records.append(rec)
        return rec

    def _encode(self, res, phase, step, r, chunk, src_dense: torch.Tensor, nnz_switch: int, copy_dense: bool):
        """compress + decide on the measured nnz (the oracle's _encode).  If copy_dense the dense form is
        materialised into the message's own buffer, else the message aliases src_dense."""
        m = self._msg()
        rec = self._record(res, phase, step, r, chunk, m)
        pk.compress(src_dense, m.pici, self.ws[r])
        pk.nnz(m.pici, self.nnz[rec.nnz_index:rec.nnz_index + 1])
        f = self.fmt[rec.fmt_index:rec.fmt_index + 1]
        if copy_dense:
            pk.maybe_densify(m.pici, nnz_switch, m.dense, f)
        else:
            pk.maybe_densify(m.pici, nnz_switch, None, f)
            m = _Msg(m.pici, src_dense)
            rec.msg = m if self.keep else None
        return m, f

    # ------------------------------------------------------------------------------------------
    def reduce_scatter(self, X: list[torch.Tensor], nnz_switch: int, outputs: list[torch.Tensor] | None = None,
                       res: RingResult | None = None) -> RingResult:
        """X[r]: rank r's N = P*n element fp32 buffer.  Returns outputs[r] = reduced chunk r (n elements)."""
        P, n = self.P, self.n
        assert len(X) == P and all(x.numel() == P * n and x.dtype == torch.float32 and x.is_cuda for x in X)
        res = res or self._begin()
        outs = outputs or [torch.empty(n, dtype=torch.float32, device=self.device) for _ in range(P)]
        chunk = lambda r, c: X[r][c * n:(c + 1) * n]

        cur = [None] * P

        def step0(r):                                        # step 0: always compress
            c = (r - 1) % P
            cur[r] = self._encode(res, "rs", 0, r, c, chunk(r, c), nnz_switch, copy_dense=True)
        self._step(step0)

        for s in range(1, P):
            nxt = [None] * P

            def step(r, s=s, cur=cur, nxt=nxt):
                (m_in, f_in) = cur[(r - 1) % P]
                c = (r - 1 - s) % P
                loc = chunk(r, c)
                if s == P - 1:                                # last step: acc is rank r's dense output
                    pk.reduce_sd_out(m_in.pici, loc, outs[r], gate=f_in, gate_value=pk.FMT_PICI)
                    pk.dense_add(m_in.dense, loc, outs[r], None, gate=f_in, gate_value=pk.FMT_DENSE)
                    return
                m = self._msg()
                rec = self._record(res, "rs", s, r, c, m)
                f = self.fmt[rec.fmt_index:rec.fmt_index + 1]
                if self.strategy == "fused":
                    pk.compress(loc, self.local[r], self.ws[r], gate=f_in, gate_value=pk.FMT_PICI)
                    pk.reduce_ss(m_in.pici, self.local[r], m.pici, self.ws[r], gate=f_in, gate_value=pk.FMT_PICI)
                    pk.maybe_densify(m.pici, nnz_switch, m.dense, f, gate=f_in, gate_value=pk.FMT_PICI)
                else:
                    pk.reduce_sd_out(m_in.pici, loc, m.dense, gate=f_in, gate_value=pk.FMT_PICI)
                    pk.compress(m.dense, m.pici, self.ws[r], gate=f_in, gate_value=pk.FMT_PICI)
                    pk.maybe_densify(m.pici, nnz_switch, None, f, gate=f_in, gate_value=pk.FMT_PICI)
                pk.nnz(m.pici, self.nnz[rec.nnz_index:rec.nnz_index + 1])
                pk.dense_add(m_in.dense, loc, m.dense, f, gate=f_in, gate_value=pk.FMT_DENSE)
                nxt[r] = (m, f)
            self._step(step)
            cur = nxt
        res.outputs = outs
        return res

    # ------------------------------------------------------------------------------------------
    def all_gather(self, shards: list[torch.Tensor], nnz_switch: int | None = None,
                   outputs: list[torch.Tensor] | None = None, res: RingResult | None = None,
                   phase: str = "ag") -> RingResult:
        """shards[r]: rank r's n-element shard.  outputs[r]: P*n elements, identical on every rank."""
        P, n = self.P, self.n
        assert len(shards) == P and all(x.numel() == n and x.dtype == torch.float32 and x.is_cuda for x in shards)
        res = res or self._begin()
        outs = outputs or [torch.empty(P * n, dtype=torch.float32, device=self.device) for _ in range(P)]
        switch = nnz_switch if nnz_switch is not None else n + 1
        msgs = [None] * P

        def step0(r):                                        # step 0: compress once
            msgs[r] = self._encode(res, phase, 0, r, r, shards[r], switch, copy_dense=False)
            pk.dense_copy(shards[r], outs[r][r * n:(r + 1) * n])          # own slot: plain copy (C9 #12)
        self._step(step0)
        for s in range(1, P):
            def step(r, s=s):
                c = (r - s) % P                               # forwarded unchanged: still rank c's message
                m, f = msgs[c]
                slot = outs[r][c * n:(c + 1) * n]
                pk.decompress(m.pici, slot, gate=f, gate_value=pk.FMT_PICI)
                pk.dense_copy(m.dense, slot, gate=f, gate_value=pk.FMT_DENSE)
            self._step(step)
        res.outputs = outs
        return res

    # ------------------------------------------------------------------------------------------
    def all_reduce(self, X: list[torch.Tensor], nnz_switch_rs: int, nnz_switch_ag: int) -> RingResult:
        """RS, then the ag_thresh decision on each reduced chunk, then AG."""
        res = self.reduce_scatter(X, nnz_switch_rs)
        reduced = res.outputs
        return self.all_gather(reduced, nnz_switch_ag, None, res, phase="ar.ag")
