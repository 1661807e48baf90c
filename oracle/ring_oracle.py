"""TEST INFRASTRUCTURE - plain CPU oracle of SpCCL's sparse ring collectives over P logical ranks.

Follows the paper step by step (PAPER.md:52-55 ring; 207 all-gather; 219 reduce-scatter and
all-reduce = RS + AG; 227-233 threshold switch; 239 ag_thresh at the RS->AG transition) with the
chunk schedule of SURVEY.md S8(c) C8 (NCCL's: rank r sends to r+1 and ends owning chunk r).
Every per-element operation is a call into oracle/pici_oracle.c; nothing here imports or calls
the CUDA path.  Each collective returns the outputs AND a per-(step, rank) log of the messages so
that the GPU driver can be compared message by message.

Two statements are provided for the reducing collectives:
  * ``*_definition``  - the plain definition: a dense fp32 LEFT FOLD in ring order,
        out_c = ((..(X_{c+1}[c] + X_{c+2}[c]) + ..) + X_{c-1}[c]) + X_c[c]   (indices mod P),
    "the oracle's fixed rank order" (BASELINE.json north_star);
  * ``ring_*``        - the paper's algorithm: scatter-add the received Pici message into the
    dense local chunk, re-compress before the next send, switch to dense once the MEASURED nnz
    reaches nnz_switch (readings C9 #9/#10), stay dense afterwards.
tests/test_oracle_ring.py pins the second to the first bit for bit.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import pici_oracle as po


@dataclass
class Message:
    fmt: str                          # "pici" | "dense"
    chunk: int
    pici: po.Pici | None = None
    dense: np.ndarray | None = None   # float32[n] when fmt == "dense"
    nnz: int | None = None            # measured nnz (None after a dense step: not computed)

    def nbytes(self) -> int:
        return self.pici.message_bytes() if self.fmt == "pici" else self.dense.nbytes


@dataclass
class LogEntry:
    phase: str
    step: int
    rank: int
    chunk: int
    fmt: str
    nnz: int | None
    extrapolated_sparsity: float | None   # Eq. 7 - diagnostic only
    msg: Message | None = None


@dataclass
class RingLog:
    entries: list[LogEntry] = field(default_factory=list)
    switch_step: dict[int, int | None] = field(default_factory=dict)  # chunk -> first step sent dense

    def at(self, phase: str, step: int, rank: int) -> LogEntry:
        for e in self.entries:
            if e.phase == phase and e.step == step and e.rank == rank:
                return e
        raise KeyError((phase, step, rank))


def _chunk(x: np.ndarray, c: int, n: int) -> np.ndarray:
    return x[c * n:(c + 1) * n]


def _encode(acc_f32: np.ndarray, chunk: int, nnz_switch: int) -> Message:
    """Compress, then decide on the measured nnz: Pici iff nnz < nnz_switch (C9 #9)."""
    p = po.compress(acc_f32, "f32")
    if p.nnz >= nnz_switch:
        return Message("dense", chunk, None, acc_f32.copy(), p.nnz)
    return Message("pici", chunk, p, None, p.nnz)


# ------------------------------------------------------------------------------------------------
# Reduce-scatter
# ------------------------------------------------------------------------------------------------

def reduce_scatter_definition(X: list[np.ndarray]) -> list[np.ndarray]:
    """Dense left fold in ring order (C8).  out[c] is rank c's n-element result."""
    P = len(X)
    n = X[0].size // P
    out = []
    for c in range(P):
        acc = _chunk(X[(c + 1) % P], c, n).astype(np.float32, copy=True)
        for j in range(2, P + 1):
            acc = po.dense_add(acc, np.ascontiguousarray(_chunk(X[(c + j) % P], c, n)))
        out.append(acc)
    return out


def ring_reduce_scatter(X: list[np.ndarray], nnz_switch: int, keep_messages: bool = True
                        ) -> tuple[list[np.ndarray], RingLog]:
    """The paper's sparse ring reduce-scatter over P logical ranks."""
    P = len(X)
    N = X[0].size
    assert all(x.dtype == np.float32 and x.size == N for x in X) and N % (P * po.TILE) == 0
    n = N // P
    log = RingLog()
    sigma0 = [None] * P
    sigma = [None] * P

    def record(step, r, m):
        c = m.chunk
        if m.fmt == "dense" and c not in log.switch_step:
            log.switch_step[c] = step
        log.entries.append(LogEntry("rs", step, r, c, m.fmt, m.nnz, sigma[r],
                                    m if keep_messages else None))

    # Step 0: every rank compresses chunk (r-1) mod P of its own input ("Step 0 always executes
    # compression, and the first threshold-informed send decision is based directly on the
    # computed sparsity").
    send = [None] * P
    for r in range(P):
        c = (r - 1) % P
        send[r] = _encode(np.ascontiguousarray(_chunk(X[r], c, n)), c, nnz_switch)
        sigma0[r] = 1.0 - send[r].nnz / n
        sigma[r] = sigma0[r]
        record(0, r, send[r])

    out = [None] * P
    for s in range(1, P):
        recv = [send[(r - 1) % P] for r in range(P)]          # rank r receives from r-1
        nxt = [None] * P
        for r in range(P):
            m = recv[r]
            c = (r - 1 - s) % P
            assert m.chunk == c
            local = np.ascontiguousarray(_chunk(X[r], c, n))
            if m.fmt == "pici":
                acc = local.copy()                              # application buffer reused as scratch
                po.reduce_sd(m.pici, acc)                       # scatter-add
            else:
                acc = po.dense_add(m.dense, local)              # reduceCopy on dense steps
            sigma[r] = sigma[r] * sigma0[r]                     # Eq. 7, logged beside the measurement
            if s == P - 1:
                assert c == r
                out[r] = acc
            elif m.fmt == "dense":
                nxt[r] = Message("dense", c, None, acc, None)   # once dense, stays dense (C8)
                record(s, r, nxt[r])
            else:
                nxt[r] = _encode(acc, c, nnz_switch)            # recompress before the next send
                record(s, r, nxt[r])
        send = nxt
    for c in range(P):
        log.switch_step.setdefault(c, None)
    return out, log


# ------------------------------------------------------------------------------------------------
# All-gather
# ------------------------------------------------------------------------------------------------

def all_gather_definition(shards: list[np.ndarray]) -> np.ndarray:
    return np.concatenate(shards)


def ring_all_gather(shards: list[np.ndarray], nnz_switch: int | None = None, phase: str = "ag",
                    log: RingLog | None = None, keep_messages: bool = True
                    ) -> tuple[list[np.ndarray], RingLog]:
    """Sparse ring all-gather: compress once at step 0, forward unchanged for P-1
    steps, decompress every received shard immediately into the output.  Own slot = plain copy
    (C9 #12).  nnz_switch (count) makes a shard travel dense when nnz >= nnz_switch (used by
    all-reduce's ag_thresh); None = always Pici."""
    P = len(shards)
    n = shards[0].size
    assert all(x.dtype == np.float32 and x.size == n for x in shards) and n % po.TILE == 0
    log = log or RingLog()
    outs = [np.empty(P * n, np.float32) for _ in range(P)]
    send = [None] * P
    for r in range(P):
        own = np.ascontiguousarray(shards[r])
        send[r] = _encode(own, r, nnz_switch if nnz_switch is not None else n + 1)
        outs[r][r * n:(r + 1) * n] = own
        log.entries.append(LogEntry(phase, 0, r, r, send[r].fmt, send[r].nnz, None,
                                    send[r] if keep_messages else None))
    for s in range(1, P):
        recv = [send[(r - 1) % P] for r in range(P)]
        for r in range(P):
            m = recv[r]
            c = (r - s) % P
            assert m.chunk == c
            if m.fmt == "pici":
                outs[r][c * n:(c + 1) * n] = po.decompress(m.pici).view(np.float32)
            else:
                outs[r][c * n:(c + 1) * n] = m.dense
            log.entries.append(LogEntry(phase, s, r, c, m.fmt, m.nnz, None, None))
        send = recv                                             # forwarded unchanged
    return outs, log


# ------------------------------------------------------------------------------------------------
# All-reduce = RS + AG
# ------------------------------------------------------------------------------------------------

def all_reduce_definition(X: list[np.ndarray]) -> np.ndarray:
    return np.concatenate(reduce_scatter_definition(X))


def ring_all_reduce(X: list[np.ndarray], nnz_switch_rs: int, nnz_switch_ag: int,
                    keep_messages: bool = True) -> tuple[list[np.ndarray], RingLog]:
    reduced, log = ring_reduce_scatter(X, nnz_switch_rs, keep_messages)
    # RS->AG transition: each rank re-decides the format of its reduced chunk with the AG
    # threshold on a measured nnz (trial compress).
    outs, log = ring_all_gather(reduced, nnz_switch_ag, "ar.ag", log, keep_messages)
    return outs, log


# ------------------------------------------------------------------------------------------------
# The paper's adaptive policy (SIV-C): extrapolated sparsity (Eq. 7), link-aware
# thresholds (intra_thresh / inter_thresh), phase-aware ag_thresh.  SURVEY.md S8(f) f1.
#
# What the text fixes, restated (readings are listed in DESIGN.md S2):
#   * every rank tracks ONE sparsity sigma.  Step 0 always compresses; sigma_0 = sigma = 1 - nnz / n is the
#     computed sparsity, and the first send decision uses it directly.
#   * at a later step the rank has scatter-added (or densely added) the received data into its local
#     chunk; "the reduction process does not naturally compute the post-reduction sparsity", so the
#     decision "whether to compress data before sending is made based on an extrapolated post-reduction
#     sparsity" sigma_next = sigma_prev * sigma_0 (Eq. 7).
#   * the send is dense when the sparsity used for the decision is <= the threshold of the LINK the send
#     goes over: intra_thresh inside a node, inter_thresh between nodes.
#   * a dense send computes no nonzero count: the extrapolation is carried forward, "where sigma_prev may
#     now represent a prior-step computed sparsity or a previous extrapolation"; "when compressions occur
#     after extrapolations, they calibrate the tracked sparsity using the computed nonzero count"
#     (PAPER.md:247).  Dense sends may therefore be sandwiched between sparse ones.
#   * all-reduce: ag_thresh decides at the RS -> AG transition, on the tracked sparsity extrapolated to
#     the last accumulation, whether the all-gather phase carries Pici or dense data.
# All sparsities are IEEE doubles: 1 - nnz / n (one division, one subtraction) and products; a threshold
# is a double; the compare is `sigma <= tau`.  The CUDA driver evaluates the same expressions in fp64.
# ------------------------------------------------------------------------------------------------

@dataclass
class Policy:
    intra_thresh: float = 0.6       # PAPER.md:237 (Pici, fp32 reduce-scatter)
    inter_thresh: float = 0.5
    ag_thresh: float = 0.1
    ranks_per_node: int = 2         # logical ranks r with the same r // ranks_per_node share a "node"

    def link_thresh(self, r: int, P: int) -> float:
        """Threshold of the link rank r sends over (to rank r + 1 mod P)."""
        same = (r // self.ranks_per_node) == (((r + 1) % P) // self.ranks_per_node)
        return self.intra_thresh if same else self.inter_thresh


def measured_sparsity(nnz: int, n: int) -> float:
    return 1.0 - float(nnz) / float(n)


def ring_reduce_scatter_policy(X: list[np.ndarray], pol: Policy, keep_messages: bool = True
                               ) -> tuple[list[np.ndarray], RingLog, list[float], list[float]]:
    """Reduce-scatter under the paper's policy.  Returns (outputs, log, sigma0 per rank, tracked sigma per
    rank extrapolated to the last accumulation).  LogEntry.extrapolated_sparsity holds the sparsity the send
    decision of that entry was taken on; LogEntry.nnz is None for dense sends (no count is computed)."""
    P = len(X)
    N = X[0].size
    assert all(x.dtype == np.float32 and x.size == N for x in X) and N % (P * po.TILE) == 0
    n = N // P
    log = RingLog()
    sigma0 = [0.0] * P
    sigma = [0.0] * P
    send = [None] * P

    def record(step, r, m, used):
        if m.fmt == "dense" and m.chunk not in log.switch_step:
            log.switch_step[m.chunk] = step
        log.entries.append(LogEntry("rs", step, r, m.chunk, m.fmt, m.nnz, used, m if keep_messages else None))

    for r in range(P):                                   # step 0: always compress, decide on the computed value
        c = (r - 1) % P
        local = np.ascontiguousarray(_chunk(X[r], c, n))
        p = po.compress(local, "f32")
        sigma0[r] = sigma[r] = measured_sparsity(p.nnz, n)
        if sigma[r] <= pol.link_thresh(r, P):
            send[r] = Message("dense", c, None, local.copy(), None)
        else:
            send[r] = Message("pici", c, p, None, p.nnz)
        record(0, r, send[r], sigma[r])

    out = [None] * P
    for s in range(1, P):
        recv = [send[(r - 1) % P] for r in range(P)]
        nxt = [None] * P
        for r in range(P):
            m = recv[r]
            c = (r - 1 - s) % P
            assert m.chunk == c
            local = np.ascontiguousarray(_chunk(X[r], c, n))
            if m.fmt == "pici":
                acc = local.copy()
                po.reduce_sd(m.pici, acc)
            else:
                acc = po.dense_add(m.dense, local)
            ext = sigma[r] * sigma0[r]                    # Eq. 7
            if s == P - 1:
                out[r] = acc
                sigma[r] = ext                            # extrapolated to the last accumulation (used by ag_thresh)
                continue
            if ext <= pol.link_thresh(r, P):              # dense send: no count, the extrapolation is carried
                sigma[r] = ext
                nxt[r] = Message("dense", c, None, acc, None)
            else:                                         # compress: the count calibrates the tracked sparsity
                p = po.compress(acc, "f32")
                sigma[r] = measured_sparsity(p.nnz, n)
                nxt[r] = Message("pici", c, p, None, p.nnz)
            record(s, r, nxt[r], ext)
        send = nxt
    for c in range(P):
        log.switch_step.setdefault(c, None)
    return out, log, sigma0, sigma


def ring_all_reduce_policy(X: list[np.ndarray], pol: Policy, keep_messages: bool = True
                           ) -> tuple[list[np.ndarray], RingLog]:
    """All-reduce under the paper's policy: RS as above, then ag_thresh on the tracked sparsity decides per rank
    whether its reduced chunk travels through the all-gather as Pici or dense."""
    P = len(X)
    reduced, log, _, sigma = ring_reduce_scatter_policy(X, pol, keep_messages)
    n = reduced[0].size
    outs = [np.empty(P * n, np.float32) for _ in range(P)]
    send = [None] * P
    for r in range(P):
        own = np.ascontiguousarray(reduced[r])
        if sigma[r] <= pol.ag_thresh:
            send[r] = Message("dense", r, None, own.copy(), None)
        else:
            p = po.compress(own, "f32")
            send[r] = Message("pici", r, p, None, p.nnz)
        outs[r][r * n:(r + 1) * n] = own
        log.entries.append(LogEntry("ar.ag", 0, r, r, send[r].fmt, send[r].nnz, sigma[r],
                                    send[r] if keep_messages else None))
    for s in range(1, P):
        recv = [send[(r - 1) % P] for r in range(P)]
        for r in range(P):
            m = recv[r]
            c = (r - s) % P
            if m.fmt == "pici":
                outs[r][c * n:(c + 1) * n] = po.decompress(m.pici).view(np.float32)
            else:
                outs[r][c * n:(c + 1) * n] = m.dense
            log.entries.append(LogEntry("ar.ag", s, r, c, m.fmt, m.nnz, None, None))
        send = recv
    return outs, log
