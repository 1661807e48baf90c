#!/usr/bin/env python
"""bench.py - the Pici hot path on B200: one JSON line (contract in the task statement).

A STEP is one pass of the whole hot path over one batch of synthetic input of
BASELINE.json configs[1] (N = 2^28 single buffer, fp32, unstructured Bernoulli sparsity, N(0,1) values):

    compress(X) -> PX ; compress(Y) -> PY          a1-a3   (X, Y: seeds 0 and 1 of the config)
    reduce_ss(PX, PY) -> PO                        a6      sparse + sparse merge
    nnz(PO)                                        a7      on-device count
    maybe_densify(PO, nnz_switch = 0) -> D         a8 + a4 the switch is taken: a full decompress
    reduce_sd(PX, D)                               a5      scatter-add into the dense buffer

`value` = dense-equivalent GB/s = (5 buffers of N*s bytes handled per step) * K / time, inputs resident in
HBM.  `e2e` = the same metric through the C ABI's HOST-buffer calls (pici_compress_host +
pici_decompress_host, pinned host memory, copies inside the timed region): 2 buffers of N*s per step.
`roofline` = the dominant kernel (largest share of the timed region), algorithmic bytes (DESIGN.md
"Algorithmic bytes") / its CUDA-event duration measured inside the timed region, against the measured
HBM copy peak of MEASURED_PEAKS.json.  `sweep` = every kernel at every sparsity of the config (fp32 and
bf16), timed alone with CUDA events after the K steps.  `cpu_baseline` = oracle/ (single-threaded C,
as it stands) on a bounded sample of the same workload, on this box's host cores.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--sparsity 0.99] [--no-sweep]
    python bench.py --impl reference ...     # the oracle timed on the host cores (same metric)
Under torchrun (N > 1) every rank runs the same per-GPU workload on its own GPU (weak scaling; the path
has no data-path collective on one node: SURVEY.md S8(e) "replicas only"), time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import workloads as wl  # noqa: E402

METRIC = "Pici compress/decompress/merge GB/s (dense-equiv) and % of B200 HBM peak vs sparsity"
UNIT = "GB/s (dense-equivalent)"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
OPS_PER_STEP = 5                   # N-element buffers handled per step (2 compress, merge, densify, scatter-add)
TILE = 4096


def measured_peak() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy burst)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic() -> dict:
    """Per-launch DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of each op from the committed
    ncu --set full capture: profiles/traffic.csv, lines `op,read_bytes,write_bytes` (see profiles/*.md)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    out = {}
    if os.path.exists(p):
        with open(p) as f:
            for line in f:
                parts = line.strip().split(",")
                if len(parts) == 3 and parts[1].replace(".", "").isdigit():
                    out[parts[0]] = int(float(parts[1]) + float(parts[2]))
    return out


# ---------------------------------------------------------------------------------------------------
# algorithmic bytes; n multiple of 4096 here
# ---------------------------------------------------------------------------------------------------
def meta_bytes(n: int) -> int:
    T = (n + TILE - 1) // TILE
    return 8 * 64 * T + 4 * (T + 1)


def bytes_compress(n, s, nnz):          # read dense, write B + I + A
    return n * s + meta_bytes(n) + s * nnz


def bytes_decompress(n, s, nnz):        # read B + I + A, write dense
    return n * s + meta_bytes(n) + s * nnz


def bytes_reduce_ss(n, nx, ny, no):     # read 2 x (B, I, A), write (B, I, A)
    return 3 * meta_bytes(n) + 4 * (nx + ny + no)


def bytes_reduce_sd(n, nnz, touched_sectors=None):
    """Sparse operand + the cheaper of (a) streaming the dense buffer through (read + write n*4) and
    (b) read-modify-write of only the touched 32-byte sectors (2 x 32 B each)."""
    stream = 8 * n
    if touched_sectors is None:
        return meta_bytes(n) + 4 * nnz + stream
    return meta_bytes(n) + 4 * nnz + min(stream, 64 * touched_sectors)


# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows]
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric/config/unit."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import numpy as np
    from oracle import pici_oracle as po
    n = args.ref_n
    d = 1.0 - args.sparsity
    x = wl.sparse_buffer(n, d, seed=wl.stream_seed(0, 0)).numpy()
    y = wl.sparse_buffer(n, d, seed=wl.stream_seed(0, 1)).numpy()

    with PinnedCore() as pin:
        for _ in range(args.warmup):
            oracle_step(po, np, x, y, n)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            oracle_step(po, np, x, y, n)
        dt = time.perf_counter() - t0
        where = pin.describe()
    val = OPS_PER_STEP * n * 4 * args.steps / dt / 1e9
    sample = f"first-principles sample: N=2^{n.bit_length() - 1} elements of the same recipe per step (full workload N=2^28)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[1] Pici hot path, fp32, sparsity {args.sparsity}, seeds 0/1; oracle on host cores",
                   "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cores_available": os.cpu_count(), **where},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


class HotPath:
    """Buffers + the step of the hot path for one (n, dtype=f32, sparsity)."""

    def __init__(self, pk, n: int, density: float, seed_x: int, seed_y: int, device):
        self.pk, self.n = pk, n
        self.x = wl.sparse_buffer(n, density, seed=seed_x, device=device)
        self.y = wl.sparse_buffer(n, density, seed=seed_y, device=device)
        self.px, self.py, self.po = (pk.alloc_pici(n, pk.F32, device) for _ in range(3))
        self.ws = pk.alloc_workspace(n, device)
        self.dense = torch.empty(n, dtype=torch.float32, device=device)
        self.cnt = torch.zeros(1, dtype=torch.int32, device=device)
        self.flag = torch.zeros(1, dtype=torch.int32, device=device)
        self.launches_per_step = 7      # compress x2, reduce_ss, nnz, expand (densify), scatter_add_sparse + expand (reduce_sd)

    OPS = ("compress", "compress", "reduce_ss", "nnz", "maybe_densify", "reduce_sd")

    def step(self, ev=None):
        pk = self.pk
        calls = (
            lambda: pk.compress(self.x, self.px, self.ws),
            lambda: pk.compress(self.y, self.py, self.ws),
            lambda: pk.reduce_ss(self.px, self.py, self.po, self.ws),
            lambda: pk.nnz(self.po, self.cnt),
            lambda: pk.maybe_densify(self.po, 0, self.dense, self.flag),
            lambda: pk.reduce_sd(self.px, self.dense),
        )
        if ev is None:
            for c in calls:
                c()
            return
        for i, c in enumerate(calls):
            ev[i][0].record()
            c()
            ev[i][1].record()

    def counts(self):
        torch.cuda.synchronize()
        return self.px.nnz_host(), self.py.nnz_host(), self.po.nnz_host()


def touched_sectors_f32(mask_dense: torch.Tensor) -> int:
    """Number of 32-byte sectors (8 fp32) of a dense buffer holding at least one nonzero."""
    n8 = mask_dense.numel() // 8 * 8
    return int((mask_dense[:n8].view(-1, 8) != 0).any(dim=1).sum().item())


NO_GRAPH = False      # --no-graph: time eager launches with events (the form the ncu captures profile)


def graph_time(fns, launches: int, replays: int = 5, warm: int = 5):
    """Per-launch time of a kernel with no host cost inside the timed region: `launches` calls - call i uses
    fns[i % len(fns)], i.e. the buffer sets are rotated so that nothing is re-read from L2 - are captured into ONE
    CUDA graph, replayed `replays` times between CUDA events (after `warm` eager calls per set and one replay).
    Returns (median, min) over the replays of ms per launch."""
    for _ in range(max(1, (warm + len(fns) - 1) // len(fns))):
        for f in fns:
            f()
    torch.cuda.synchronize()
    if NO_GRAPH:
        ts = []
        for i in range(launches):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fns[i % len(fns)](); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ts.sort()
        return ts[len(ts) // 2], ts[0]
    st = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            for i in range(launches):
                fns[i % len(fns)]()
    g.replay()
    torch.cuda.synchronize()
    ts = []
    for _ in range(replays):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); g.replay(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b) / launches)
    ts.sort()
    return ts[len(ts) // 2], ts[0]


L2_BYTES = 126e6                     # B200 L2 (B200_PROFILING.md)


def run_sweep(pk, n: int, peak: float, launches: int, device, dtypes=("f32", "bf16"), sparsities=None,
              ops=("compress", "decompress", "reduce_ss", "reduce_sd"), seeds=(0, 1, 2, 3, 4)) -> list[dict]:
    """Every kernel alone at every sparsity of configs[1], fp32: all ops, bf16: compress / decompress.
    Seeds 0-4 of the config are five buffer sets; launch i of the timed CUDA graph works on set i mod 5, so every
    launch reads inputs that at least four other launches' traffic (> 2x L2 for every op) has pushed out of L2,
    and the reported time is the mean over the seeds (SURVEY.md S8(d) Timing: >= 5 warm-ups, >= 100 timed launches,
    rotate buffer sets when the working set is < 2x L2)."""
    rows = []
    for dtype in dtypes:
        s = 4 if dtype == "f32" else 2
        D = pk.F32 if dtype == "f32" else pk.BF16
        ws = pk.alloc_workspace(n, device)
        for sp in (sparsities or wl.CONFIG2_SPARSITIES):
            d = 1.0 - sp
            merge = dtype == "f32" and ("reduce_ss" in ops or "reduce_sd" in ops)
            sets = []
            for sd in seeds:
                S = {"x": wl.sparse_buffer(n, d, seed=wl.stream_seed(sd, 0), dtype=dtype, device=device),
                     "px": pk.alloc_pici(n, D, device)}
                pk.compress(S["x"], S["px"], ws)
                if "decompress" in ops:
                    S["out"] = torch.empty_like(S["x"])
                if merge:
                    S["y"] = wl.sparse_buffer(n, d, seed=wl.stream_seed(sd, 1), dtype=dtype, device=device)
                    S["py"], S["po"] = pk.alloc_pici(n, D, device), pk.alloc_pici(n, D, device)
                    pk.compress(S["y"], S["py"], ws)
                    pk.reduce_ss(S["px"], S["py"], S["po"], ws)
                sets.append(S)
            torch.cuda.synchronize()
            for S in sets:
                S["nx"] = S["px"].nnz_host()
                if merge:
                    S["ny"], S["no"] = S["py"].nnz_host(), S["po"].nnz_host()
            mean = lambda vals: sum(vals) / len(vals)

            def row(op, fns, nbytes, extra=None):
                ms, mn = graph_time(fns, launches)
                r = {"dtype": dtype, "sparsity": sp, "op": op, "ms": round(ms, 4), "ms_min": round(mn, 4),
                     "dense_equiv_gbs": round(n * s / ms / 1e6, 1), "alg_bytes": int(nbytes),
                     "bytes_moved_gbs": round(nbytes / ms / 1e6, 1), "frac": round(nbytes / ms / 1e6 / peak, 3),
                     "seeds": list(seeds), "launches_timed": launches * 5,
                     "l2": f"defeated: {len(seeds)} rotated buffer sets, {nbytes * (len(seeds) - 1) / L2_BYTES:.1f}x L2 between reuses"}
                if extra:
                    r.update(extra)
                rows.append(r)

            if "compress" in ops:
                row("compress", [lambda S=S: pk.compress(S["x"], S["px"], ws) for S in sets],
                    mean([bytes_compress(n, s, S["nx"]) for S in sets]))
            if "decompress" in ops:
                row("decompress", [lambda S=S: pk.decompress(S["px"], S["out"]) for S in sets],
                    mean([bytes_decompress(n, s, S["nx"]) for S in sets]))
            if merge and "reduce_ss" in ops:
                row("reduce_ss", [lambda S=S: pk.reduce_ss(S["px"], S["py"], S["po"], ws) for S in sets],
                    mean([bytes_reduce_ss(n, S["nx"], S["ny"], S["no"]) for S in sets]))
            if merge and "reduce_sd" in ops:
                sect = mean([touched_sectors_f32(S["x"]) for S in sets])
                elem = mean([meta_bytes(n) + 12 * S["nx"] for S in sets])      # S8(d): 0.126 + 12 d bytes per element
                # in place into the (dense) y buffer of the set: every launch adds x once more
                row("reduce_sd", [lambda S=S: pk.reduce_sd(S["px"], S["y"]) for S in sets],
                    mean([bytes_reduce_sd(n, S["nx"], sect) for S in sets]),
                    {"touched_sector_frac": round(sect / (n / 8), 4), "alg_bytes_element_level": int(elem)})
                if mean([S["nx"] for S in sets]) <= 224 * (n // TILE):
                    # read-modify-write regime: what the memory system gives for the bare access pattern - the same
                    # dense[i] += v on the same index sets, one thread per index, nothing else (pici_probe_random_rmw)
                    for S in sets:
                        S["idx"] = torch.nonzero(S["x"]).flatten().to(torch.int32)
                    pms, _ = graph_time([lambda S=S: pk.probe_random_rmw(S["idx"], S["y"]) for S in sets], launches)
                    rows[-1]["rmw_probe_ms"] = round(pms, 4)
                    rows[-1]["speed_vs_rmw_probe"] = round(pms / rows[-1]["ms"], 3)   # > 1: faster than the bare stream
            del sets
            torch.cuda.empty_cache()
    return rows


def run_coo_sweep(pk, n: int, peak: float, launches: int, device, sparsities=(0.9, 0.95, 0.96875, 0.99, 0.999, 0.9999),
                  seeds=(0, 1, 2)) -> list[dict]:
    """Pici against the paper's COO variant, kernel by kernel at
    N elements, fp32: same buffers, same rotation of seeded buffer sets as run_sweep.  A row gives both formats'
    time, algorithmic bytes and message size; `coo_over_pici` > 1 means Pici is faster.  There is no wire here, so
    this is the compute side of Fig. 3's crossover; the size side is `msg_bytes` (equal at 96.875 % sparsity but
    for Pici's I)."""
    from paper_2607_04676_b200 import coo as ck
    ck.lib()
    rows = []
    ws = pk.alloc_workspace(n, device)
    cws = ck.alloc_workspace(n, device)
    for sp in sparsities:
        d = 1.0 - sp
        sets = []
        for sd in seeds:
            S = {"x": wl.sparse_buffer(n, d, seed=wl.stream_seed(sd, 0), device=device),
                 "y": wl.sparse_buffer(n, d, seed=wl.stream_seed(sd, 1), device=device)}
            S["px"], S["py"], S["po"] = (pk.alloc_pici(n, pk.F32, device) for _ in range(3))
            S["cx"], S["cy"], S["co"] = (ck.alloc_coo(n, device) for _ in range(3))
            pk.compress(S["x"], S["px"], ws); pk.compress(S["y"], S["py"], ws)
            pk.reduce_ss(S["px"], S["py"], S["po"], ws)
            ck.compress(S["x"], S["cx"], cws); ck.compress(S["y"], S["cy"], cws)
            ck.reduce_ss(S["cx"], S["cy"], S["co"], cws)
            S["out"] = torch.empty_like(S["x"])
            sets.append(S)
        torch.cuda.synchronize()
        mean = lambda vals: sum(vals) / len(vals)
        nx = mean([S["cx"].nnz_host() for S in sets]); ny = mean([S["cy"].nnz_host() for S in sets])
        no = mean([S["co"].nnz_host() for S in sets])
        assert all(S["cx"].nnz_host() == S["px"].nnz_host() and S["co"].nnz_host() == S["po"].nnz_host() for S in sets)
        sect = mean([touched_sectors_f32(S["x"]) for S in sets])
        cases = {
            "compress": (lambda S: pk.compress(S["x"], S["px"], ws), lambda S: ck.compress(S["x"], S["cx"], cws),
                         bytes_compress(n, 4, nx), 4 * n + 8 * nx),
            "decompress": (lambda S: pk.decompress(S["px"], S["out"]), lambda S: ck.decompress(S["cx"], S["out"], cws),
                           bytes_decompress(n, 4, nx), 4 * n + 8 * nx),
            "reduce_ss": (lambda S: pk.reduce_ss(S["px"], S["py"], S["po"], ws), lambda S: ck.reduce_ss(S["cx"], S["cy"], S["co"], cws),
                          bytes_reduce_ss(n, nx, ny, no), 8 * (nx + ny + no)),
            "reduce_sd": (lambda S: pk.reduce_sd(S["px"], S["y"]), lambda S: ck.reduce_sd(S["cx"], S["y"]),
                          bytes_reduce_sd(n, nx, sect), 8 * nx + min(8 * n, 64 * sect)),
        }
        for op, (fp, fc, bp, bc) in cases.items():
            pms, _ = graph_time([lambda S=S: fp(S) for S in sets], launches)
            cms, _ = graph_time([lambda S=S: fc(S) for S in sets], launches)
            rows.append({"sparsity": sp, "op": op, "pici_ms": round(pms, 4), "coo_ms": round(cms, 4),
                         "coo_over_pici": round(cms / pms, 3), "pici_alg_bytes": int(bp), "coo_alg_bytes": int(bc),
                         "pici_frac": round(bp / pms / 1e6 / peak, 3), "coo_frac": round(bc / cms / 1e6 / peak, 3),
                         "msg_bytes": {"pici": int(meta_bytes(n) + 4 * nx), "coo": int(8 * nx), "dense": 4 * n},
                         "seeds": list(seeds), "launches_timed": launches * 5})
        del sets
        torch.cuda.empty_cache()
    return rows


def run_prune(pk, n: int, peak: float, launches: int, device, seeds=(0, 1, 2), leak: float = 0.9) -> dict:
    """The upstream workload step: sampled top-k pruning (sample 0.1 %, keep
    1 %) with leaky error feedback, fused with Pici compression in ONE pass over the gradient.  Synthetic gradients
    N(0, 0.02^2) (the paper's are GPT-2 XL / StarCoder2 gradients on WikiText-103, not in this container).  Algorithmic
    bytes of the fused pass: read g and e (8 N), write e (4 N), write the Pici object."""
    from paper_2607_04676_b200 import prune as pn
    pn.lib()
    sample = torch.arange(0, n, 1000, device=device, dtype=torch.int32)
    m = sample.numel()
    k = -(-m // 100)
    ws = pn.alloc_workspace(n, m, device)
    sets = []
    for sd in seeds:
        S = {"g": wl.values(n, seed=wl.stream_seed(sd, 0), scale=0.02, device=device),
             "e": wl.values(n, seed=wl.stream_seed(sd, 1), scale=0.01, device=device),
             "tau": torch.zeros(1, device=device), "p": pk.alloc_pici(n, pk.F32, device)}
        pn.threshold(S["g"], S["e"], leak, sample, k, S["tau"], ws)
        sets.append(S)
    tms, _ = graph_time([lambda S=S: pn.threshold(S["g"], S["e"], leak, sample, k, S["tau"], ws) for S in sets], launches)
    # the fused pass, launch by launch with CUDA events (0.5 ms each, far above the launch cost); the threshold is
    # recomputed (untimed) before every pass, as an iteration of the method does, so every message is ~99 % sparse
    ts, fr, sp = [], [], []
    for i in range(5 + launches):
        S = sets[i % len(sets)]
        pn.threshold(S["g"], S["e"], leak, sample, k, S["tau"], ws)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); pn.prune_compress(S["g"], S["e"], leak, S["tau"], S["p"], ws); b.record()
        torch.cuda.synchronize()
        if i >= 5:
            nnz = S["p"].nnz_host()
            ms = a.elapsed_time(b)
            ts.append(ms); sp.append(1.0 - nnz / n); fr.append((12 * n + meta_bytes(n) + 4 * nnz) / ms / 1e6)
    ts.sort(); fr.sort()
    fms, gbs = ts[len(ts) // 2], fr[len(fr) // 2]
    return {"n": n, "leak": leak, "sample": m, "k": k, "threshold_ms": round(tms, 4), "prune_compress_ms": round(fms, 4),
            "prune_compress_ms_min": round(ts[0], 4), "message_sparsity": round(sum(sp) / len(sp), 5),
            "alg_bytes_per_element": 12.0, "bytes_moved_gbs": round(gbs, 1), "frac": round(gbs / peak, 3),
            "unfused_bytes_per_element": 20.0, "launches_timed": len(ts), "seeds": list(seeds),
            "l2": "defeated: 3 rotated (g, e) sets of 2 GiB"}


def run_e2e(pk, n: int, density: float, steps: int, device, seed: int) -> dict:
    """HOST buffers in, HOST buffers out, through pici_compress_host / pici_decompress_host."""
    h_x = wl.sparse_buffer(n, density, seed=seed).pin_memory()
    h_back = torch.empty(n, dtype=torch.float32).pin_memory()
    h_p = pk.alloc_host_pici(n, pk.F32)
    d_dense = torch.empty(n, dtype=torch.float32, device=device)
    d_p = pk.alloc_pici(n, pk.F32, device)
    ws = pk.alloc_workspace(n, device)

    def step():
        pk.compress_host(h_x, h_p, d_dense, d_p, ws)
        pk.decompress_host(h_p, h_back, d_p, d_dense)

    step()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    ok = bool(torch.equal(h_back.view(torch.int32), h_x.view(torch.int32)))
    m = meta_bytes(n) + 4 * h_p.nnz
    return {"value": 2 * n * 4 * steps / dt / 1e9, "unit": UNIT, "h2d_bytes_per_step": n * 4 + m,
            "d2h_bytes_per_step": n * 4 + m, "ms_per_step": dt / steps * 1e3, "steps": steps, "round_trip_ok": ok,
            "path": "pici_compress_host + pici_decompress_host (pinned host buffers; 2 buffers of N*4 bytes per step)"}


class PinnedCore:
    """The oracle leg runs single-threaded on ONE host core (SURVEY.md S8(d) "Oracle timing": 1 thread, pinned as
    `taskset -c` would, nproc printed beside the result)."""

    def __enter__(self):
        self.saved, self.core = None, None
        try:
            self.saved = os.sched_getaffinity(0)
            self.core = max(self.saved)
            os.sched_setaffinity(0, {self.core})
        except Exception:
            self.saved = None
        return self

    def __exit__(self, *exc):
        if self.saved is not None:
            try:
                os.sched_setaffinity(0, self.saved)
            except Exception:
                pass

    def describe(self) -> dict:
        return {"pinned_core": self.core, "nproc": os.cpu_count()}


def oracle_step(po, np, x, y, n):
    px = po.compress(x.view(np.uint32), "f32")
    py = po.compress(y.view(np.uint32), "f32")
    pz = po.reduce_ss(px, py)
    po.nnz_pici(pz)
    dense = np.empty(n, np.uint32)
    po.maybe_densify(pz, 0, dense)
    po.reduce_sd(px, dense.view(np.float32))


def run_cpu_baseline(n: int, density: float) -> dict:
    import numpy as np
    from oracle import pici_oracle as po
    x = wl.sparse_buffer(n, density, seed=wl.stream_seed(0, 0)).numpy()
    y = wl.sparse_buffer(n, density, seed=wl.stream_seed(0, 1)).numpy()
    best = None
    with PinnedCore() as pin:
        for _ in range(3):                       # best of 3
            t0 = time.perf_counter()
            oracle_step(po, np, x, y, n)
            dt = time.perf_counter() - t0
            best = dt if best is None else min(best, dt)
        where = pin.describe()
    out = {"value": OPS_PER_STEP * n * 4 / best / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"same step on N=2^{n.bit_length() - 1} elements of the same recipe (fp32, same sparsity, seeds 0/1), "
                     f"best of 3; oracle/pici_oracle.c single thread pinned to one core, gcc -O2",
           "host_cores_available": os.cpu_count()}
    out.update(where)
    return out


def _timed_collective(fn, iters: int):
    """(median ms of eager enqueues, median ms of CUDA-graph replays of the same enqueues, result)"""
    fn()                                   # warm-up
    torch.cuda.synchronize()

    def med(run):
        ts = []
        for _ in range(iters):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); run(); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ts.sort()
        return ts[len(ts) // 2]

    eager = med(fn)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        res = fn()
    g.replay()
    torch.cuda.synchronize()
    graph_ms = med(g.replay)
    return eager, graph_ms, res


RING_CASES = {
    "config3": [("reduce_scatter", st, pm) for st in ("fused", "paper") for pm in (400, 80, 40, 20)],
    "config4": [("all_reduce", st, pm) for st in ("fused", "paper") for pm in (400, 200, 100)],
    "config5": [("all_gather", "fused", 900), ("all_reduce", "fused", 400), ("all_reduce", "paper", 400)],
}


def run_ring(pk, name: str, iters: int, device, cases=None) -> list[dict]:
    """Ring collectives of configs[2..4] on P logical ranks in one HBM: local-compute time of
    the whole collective - one C call, CUDA events around it; pointer hand-offs cost nothing - eager and as a
    CUDA-graph replay, the launches it enqueued and the step at which each chunk switched to dense."""
    from paper_2607_04676_b200 import ring
    cfg = {"config3": wl.config3, "config4": wl.config4, "config5": lambda: wl.config5(0)}[name]()
    X = cfg.buffers(device=device)
    P, n = cfg.ranks, cfg.chunk
    dense_bytes = P * P * n * 4
    rows = []
    for coll, strategy, permille in (cases or RING_CASES[name]):
        drv = ring.RingDriver(P, n, device=device, strategy=strategy)
        sw = wl.nnz_switch_from_permille(n, permille)
        if coll == "reduce_scatter":
            outs = [torch.empty(n, dtype=torch.float32, device=device) for _ in range(P)]
            ms, gms, res = _timed_collective(lambda: drv.reduce_scatter(X, sw, outputs=outs), iters)
        elif coll == "all_reduce":
            outs = [torch.empty(P * n, dtype=torch.float32, device=device) for _ in range(P)]
            ms, gms, res = _timed_collective(lambda: drv.all_reduce(X, sw, wl.nnz_switch_from_permille(n, 900), outputs=outs), iters)
        else:
            outs = [torch.empty(P * n, dtype=torch.float32, device=device) for _ in range(P)]
            shards = [X[r][r * n:(r + 1) * n] for r in range(P)]
            ms, gms, res = _timed_collective(lambda: drv.all_gather(shards, outputs=outs), iters)
        steps = res.switch_steps("rs") if coll != "all_gather" else {}
        rows.append({"config": name, "collective": coll, "strategy": strategy, "theta_permille": permille, "ranks": P,
                     "chunk": n, "ms_eager": round(ms, 3), "ms_cuda_graph": round(gms, 3), "launches": res.launches,
                     "dense_equiv_gbs": round(dense_bytes / gms / 1e6, 1),      # P ranks x N x 4 bytes / graph time
                     "switch_step_per_chunk": [steps.get(c) for c in range(P)] if steps else None})
        del drv, res, outs
        torch.cuda.empty_cache()
    return rows


def run_policy_sweep(pk, iters: int, device, density: float = 0.05, ranks_per_node: int = 2) -> list[dict]:
    """Fig. 2's analogue on logical ranks: reduce-scatter under the paper's policy, P = 8 ranks
    as 4 "nodes" of 2, N = 2^26 per rank, initial sparsity 95 % (density 0.337 after 8 contributions), every pair of
    intra_thresh x inter_thresh in 0.1 .. 0.9.  There is no link here, so the time is the LOCAL COMPUTE of the
    collective: it shows what each switching rule costs in kernels, not what it saves on a wire."""
    from paper_2607_04676_b200 import ring
    cfg = wl.config3(density)
    X = cfg.buffers(device=device)
    P, n = cfg.ranks, cfg.chunk
    outs = [torch.empty(n, dtype=torch.float32, device=device) for _ in range(P)]
    rows = []
    for strategy in ("fused", "paper"):
        for intra in range(1, 10):
            for inter in range(1, 10):
                drv = ring.RingDriver(P, n, device=device, strategy=strategy,
                                      policy=ring.Policy(intra / 10.0, inter / 10.0, 0.1, ranks_per_node))
                _, gms, res = _timed_collective(lambda: drv.reduce_scatter(X, outputs=outs), iters)
                f = res.formats()
                rows.append({"strategy": strategy, "intra_thresh": intra / 10.0, "inter_thresh": inter / 10.0,
                             "ms_cuda_graph": round(gms, 3), "dense_sends": sum(1 for v in f if v == "dense"), "sends": len(f)})
                del drv, res
    return rows


def run_dist_ring(args, rank: int, world: int, device) -> None:
    """`torchrun ... bench.py --gpus N --dist-ring`: the REAL ring (ring_dist.py, S8(f) f2) over N ranks, one process
    per GPU, NCCL point-to-point: all-reduce of config 3's recipe (N = 2^26 per rank, 99 % sparsity, independent
    supports), time = max over ranks (CUDA events, barrier on both sides).  One JSON line from rank 0."""
    import torch.distributed as dist
    from paper_2607_04676_b200 import replicas, ring_dist as rd
    n_per_rank = 1 << 26
    chunk = n_per_rank // world // (8 * TILE) * (8 * TILE)
    x = wl.sparse_buffer(world * chunk, 0.01, seed=wl.stream_seed(0, rank), device=device)
    out = torch.empty(world * chunk, dtype=torch.float32, device=device)
    ring = rd.DistRing(chunk, device, strategy="fused", segments=8)
    for _ in range(max(args.warmup, 3)):
        ring.all_reduce(x, out, None, None)
    dist.barrier(); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ring.log.sent.clear()
    a.record()
    for _ in range(args.steps):
        ring.all_reduce(x, out, None, None)
    b.record()
    dist.barrier(); torch.cuda.synchronize()
    ms = replicas.max_over_ranks(a.elapsed_time(b), device) / args.steps
    if rank == 0:
        print(json.dumps({"metric": "sparse ring all-reduce, dense-equivalent GB/s", "value": world * chunk * 4 / ms / 1e6,
                          "unit": "GB/s (dense-equivalent, per rank)", "n_gpus": world, "steps": args.steps, "ms_per_step": ms,
                          "config": {"workload": f"config3 recipe over {world} real ranks, chunk {chunk}, fused strategy, 8 segments",
                                     "transport": dist.get_backend()},
                          "wire_bytes_per_rank_per_step": ring.log.bytes_sent() // args.steps,
                          "dense_wire_bytes": 2 * (world - 1) * chunk * 4}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="pici", choices=["pici", "reference"])
    ap.add_argument("--sparsity", type=float, default=0.99)
    ap.add_argument("--log2n", type=int, default=28, help="elements per buffer (configs[1]: 2^28)")
    ap.add_argument("--ref-n", type=int, default=1 << 26, help="--impl reference: elements per step (bounded sample)")
    ap.add_argument("--cpu-n", type=int, default=1 << 26, help="cpu_baseline sample size")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sweep-iters", type=int, default=20, help="launches per timed CUDA graph (x5 replays)")
    ap.add_argument("--sweep-only", action="store_true",
                    help="time single kernels only (one JSON line per row); filters: --ops --dtypes --sparsities")
    ap.add_argument("--ops", default="compress,decompress,reduce_ss,reduce_sd")
    ap.add_argument("--dtypes", default="f32,bf16")
    ap.add_argument("--sparsities", default="")
    ap.add_argument("--ring", default="", choices=["", "config3", "config4", "config5"],
                    help="time the ring collectives of that config on P logical ranks (one JSON line per case)")
    ap.add_argument("--policy-sweep", action="store_true",
                    help="reduce-scatter under the paper's policy for every intra x inter threshold pair (Fig. 2 analogue)")
    ap.add_argument("--no-rings", action="store_true")
    ap.add_argument("--coo-sweep", action="store_true", help="Pici vs COO kernel by kernel (one JSON line per row)")
    ap.add_argument("--no-coo", action="store_true")
    ap.add_argument("--dist-ring", action="store_true", help="N > 1 under torchrun: the real ring over NCCL (ring_dist.py)")
    ap.add_argument("--prune", action="store_true", help="time the fused prune-and-compress step only (one JSON line)")
    ap.add_argument("--no-prune", action="store_true")
    ap.add_argument("--no-step-graph", action="store_true",
                    help="enqueue every step of the timed region eagerly with per-kernel events (no CUDA graph replay)")
    ap.add_argument("--no-graph", action="store_true", help="sweep rows: eager launches timed one by one (for ncu captures)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    global NO_GRAPH
    NO_GRAPH = args.no_graph
    if args.impl == "reference":
        return run_reference(args)

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the Pici path has no CPU fallback")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    from paper_2607_04676_b200 import pici as pk
    pk.lib()

    if args.dist_ring:
        if world < 2:
            raise SystemExit("bench.py --dist-ring needs torchrun with --gpus N >= 2 (one process per GPU)")
        run_dist_ring(args, rank, world, device)
        dist.barrier()
        dist.destroy_process_group()
        return
    n = 1 << args.log2n
    density = 1.0 - args.sparsity
    peak, peak_src = measured_peak()
    if args.ring:
        for r in run_ring(pk, args.ring, 7, device):
            print(json.dumps(r), flush=True)
        return
    if args.policy_sweep:
        for r in run_policy_sweep(pk, 5, device):
            print(json.dumps(r), flush=True)
        return
    if args.prune:
        print(json.dumps(run_prune(pk, n, peak, args.sweep_iters, device)), flush=True)
        return
    if args.coo_sweep:
        kw = {"sparsities": tuple(float(v) for v in args.sparsities.split(","))} if args.sparsities else {}
        for r in run_coo_sweep(pk, n, peak, args.sweep_iters, device, **kw):
            print(json.dumps(r), flush=True)
        return
    if args.sweep_only:   # kernel-by-kernel timing (also the program the single-kernel ncu captures run)
        sp = tuple(float(v) for v in args.sparsities.split(",")) if args.sparsities else None
        for r in run_sweep(pk, n, peak, args.sweep_iters, device, tuple(args.dtypes.split(",")), sp, tuple(args.ops.split(","))):
            print(json.dumps(r), flush=True)
        return
    from paper_2607_04676_b200 import replicas
    seed_x, seed_y = replicas.rank_seeds(0, rank, 2)
    hp = HotPath(pk, n, density, seed_x, seed_y, device)
    for _ in range(args.warmup):
        hp.step()
    nx, ny, no = hp.counts()

    # The step's 7 launches are captured into a CUDA graph (the calls only enqueue on the stream they are given) and
    # replayed.  Every EVENT_EVERY-th step of the timed region replays a graph of its own that carries a CUDA event
    # pair around each call (external event-record nodes) - the per-kernel durations `roofline` is computed from,
    # taken inside the timed region.  (Eager enqueues with an event pair around every call of every step cost 4.5 %
    # of the step: 0.734 ms, against 0.701 eager without events and 0.690 as a graph.)
    K = args.steps
    nops = len(HotPath.OPS)
    EVENT_EVERY = 1 if args.no_step_graph else 4
    evs = [[(torch.cuda.Event(enable_timing=True, external=not args.no_step_graph),
             torch.cuda.Event(enable_timing=True, external=not args.no_step_graph)) for _ in range(nops)]
           if k % EVENT_EVERY == 0 else None for k in range(K)]
    graphs, plain = [None] * K, None
    if not args.no_step_graph:
        side = torch.cuda.Stream(device=device)
        side.wait_stream(torch.cuda.current_stream())

        def capture(ev):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.stream(side):
                with torch.cuda.graph(g, stream=side):
                    hp.step(ev)
            return g
        plain = capture(None)
        graphs = [plain if evs[k] is None else capture(evs[k]) for k in range(K)]
        torch.cuda.current_stream().wait_stream(side)
        for g in (graphs[0], plain):
            g.replay()
        torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    w0 = time.time()
    e0.record()
    for k in range(K):
        if graphs[k] is not None:
            graphs[k].replay()
        else:
            hp.step(evs[k])
    e1.record()
    barrier()
    w1 = time.time()
    used_graph = graphs[0] is not None
    graphs = plain = None     # the graphs hold raw pointers into hp's buffers, some of which are freed below
    units_per_s, ms_total = replicas.whole_job_throughput(OPS_PER_STEP * n * 4 * K, e0.elapsed_time(e1), device)
    clocks = sampler.stop(w0, w1) if rank == 0 else None

    # per-kernel durations inside the timed region
    per_op = {}
    for i, name in enumerate(HotPath.OPS):
        per_op.setdefault(name, []).extend(evs[k][i][0].elapsed_time(evs[k][i][1]) for k in range(K) if evs[k] is not None)
    sect = touched_sectors_f32(hp.x)
    alg = {"compress": (bytes_compress(n, 4, nx) + bytes_compress(n, 4, ny)) / 2,
           "reduce_ss": bytes_reduce_ss(n, nx, ny, no),
           "maybe_densify": bytes_decompress(n, 4, no),
           "reduce_sd": bytes_reduce_sd(n, nx, sect),
           "nnz": 8}
    traffic = ncu_traffic()
    kernels = {}
    for name, ts in per_op.items():
        avg = sum(ts) / len(ts)
        n_ev = sum(1 for e in evs if e is not None)          # steps whose calls carried events
        kernels[name] = {"avg_ms": round(avg, 4), "launches": len(ts), "share": round(sum(ts) / n_ev * K / ms_total, 3),
                         "alg_bytes": int(alg[name]), "achieved_gbs": round(alg[name] / avg / 1e6, 1),
                         "frac": round(alg[name] / avg / 1e6 / peak, 3)}
    dom = max((k for k in kernels if k != "nnz"), key=lambda k: kernels[k]["avg_ms"] * kernels[k]["launches"])
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "traffic": traffic.get(dom), "peak_source": peak_src,
                "alg_bytes_per_launch": kernels[dom]["alg_bytes"], "avg_launch_ms": kernels[dom]["avg_ms"]}

    e2e = None
    if not args.no_e2e:
        del hp.dense
        torch.cuda.empty_cache()
        e2e = run_e2e(pk, n, density, max(2, min(K, 5)), device, seed_x)
        thr, ms = replicas.whole_job_throughput(2 * n * 4 * e2e["steps"], e2e["ms_per_step"] * e2e["steps"], device)
        e2e["value"], e2e["ms_per_step"] = thr / 1e9, ms / e2e["steps"]

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    value = units_per_s / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[1]: Pici hot path (2x compress, reduce_ss, nnz, maybe_densify->decompress, reduce_sd) "
                               f"on N=2^{args.log2n} fp32 buffers, Bernoulli sparsity {args.sparsity}, N(0,1), seeds 0/1",
                   "n": n, "sparsity": args.sparsity, "nnz": [nx, ny, no],
                   "l2": "inputs larger than L2 (1 GiB dense buffers, 126 MB L2); no explicit flush",
                   "step_launch": ("eager, a CUDA event pair around every call" if not used_graph else
                                   f"CUDA graph replay of the step's 7 launches; every {EVENT_EVERY}th step's graph carries a CUDA "
                                   "event pair around every call (the per-kernel times)"),
                   "parallelism": f"replicas x{world}, no data-path collective"},
        "gpu_launches": hp.launches_per_step * K,
        "kernels": kernels, "roofline": roofline, "clocks": clocks,
    }
    if e2e is not None:
        out["e2e"] = e2e
    if not args.no_sweep and world == 1:
        del hp
        torch.cuda.empty_cache()
        out["sweep"] = run_sweep(pk, n, peak, args.sweep_iters, device)
    if not args.no_rings and world == 1:    # configs[2..4]: the collectives' local-compute time (graph replay and eager)
        out["rings"] = (run_ring(pk, "config3", 5, device, [("reduce_scatter", "fused", 400), ("reduce_scatter", "fused", 40),
                                                             ("reduce_scatter", "paper", 400)]) +
                        run_ring(pk, "config4", 5, device, [("all_reduce", "fused", 400), ("all_reduce", "fused", 200)]) +
                        run_ring(pk, "config5", 5, device, [("all_gather", "fused", 900), ("all_reduce", "fused", 400)]))
    if not args.no_coo and world == 1:      # S8(f) f3: the second format, kernel by kernel against Pici
        out["coo"] = run_coo_sweep(pk, n, peak, args.sweep_iters, device)
    if not args.no_prune and world == 1:    # S8(f) f4: the upstream prune-and-compress step
        out["prune"] = run_prune(pk, n, peak, args.sweep_iters, device)
    if not args.no_cpu and world == 1:
        out["cpu_baseline"] = run_cpu_baseline(args.cpu_n, density)
    print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
