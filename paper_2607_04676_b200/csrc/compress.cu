// compress.cu - pici_compress: dense[n] -> (B, I, A) in one pass over the dense buffer.
//
// What it computes: Algorithm 1 of the paper: Phase 1 mask words + tile counts,
// Phase 2 exclusive scan of tile counts, Phase 3 compaction.  How it is laid out on B200 differs from
// the paper's A100 kernel:
//   * one warp owns one 64x64 tile; lane l owns the ADJACENT columns 2l and 2l+1 for all three phases
//     (the paper's Phase-3 mapping), so a row of the tile is one fully coalesced
//     256-byte (fp32, 64-bit per lane) or 128-byte (bf16, 32-bit per lane) request, all 64 row loads
//     of the tile are in flight at once, and the tile is read from HBM exactly ONCE: its values stay
//     in registers between Phase 1 and Phase 3;
//   * Phase 2, the device-wide exclusive scan of the tile counts (the paper scans block-locally per NCCLX segment,
//     PAPER.md:124), is a SERVICE: the compressing warps only publish their counts; CTA 0 scans them block by block
//     and writes I ("Phase 2 as a service" below); tiles are handed out by dynamic tickets from several counters,
//     and a tile's flush is deferred behind the next two tiles;
//   * Phase 3 compacts into a per-warp shared-memory stage (lane l's values are one contiguous run),
//     which is then written to A with coalesced stores.
#include <cuda_bf16.h>

#include <atomic>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

constexpr int kCompressWarps = 4;
#ifndef PICI_COMPRESS_DEFER
#define PICI_COMPRESS_DEFER 2
#endif
constexpr int kDefer = PICI_COMPRESS_DEFER;   // iterations a tile's flush lags behind its publish
#ifndef PICI_ROWSKIP_BF16
#define PICI_ROWSKIP_BF16 128
#endif

template <int DT>
struct CompressCfg;
template <>
struct CompressCfg<PICI_F32> {
    using Elem = uint32_t;
    static constexpr int kRegs = 128;       // 64 rows x 2 columns
    static constexpr int kMinBlocks = 3;    // 12 warps / SM, <= 168 registers
    static constexpr uint32_t kScanBlockLog = 8;
    static constexpr uint32_t kStageElems = kTile;          // 16 KB per warp
    static constexpr uint32_t kRowSkipNnz = 256;            // tiles with at most this many values skip empty rows in Phase 3
};
template <>
struct CompressCfg<PICI_BF16> {
    using Elem = uint16_t;
    static constexpr int kRegs = 64;        // 64 rows x (2 packed columns)
    // 3 CTAs / SM (with 5 the scan service fell behind: 0.141 ms at 99 %; 4: 0.128; 3: 0.122; 2: 0.168) and the same 16 KB
    // of stage per warp as fp32: three slots of 2730 values, so a tile at 50 % sparsity still fits a slot
    static constexpr int kMinBlocks = 3;
    static constexpr uint32_t kScanBlockLog = 9;
    static constexpr uint32_t kStageElems = 2 * kTile;
    // at 95 % sparsity (205 values per tile) only 4 % of the rows are empty and the row-skipping Phase 3 costs more than
    // it saves: limit 256 -> 128 took that point from 0.67 to 0.72 of the peak (99 %, 41 values per tile, still skips)
    static constexpr uint32_t kRowSkipNnz = PICI_ROWSKIP_BF16;
};

// (Phase 2 as a service: scan_service / service_prefix, pici_common.cuh)

// PRUNE (fp32 only): the tile that is compressed is not read but MADE while it is loaded - sampled top-k pruning with
// leaky error feedback fused into the same pass (include/pici_prune.h): acc = g + leak * e (two
// roundings), sent = |acc| >= tau ? acc : +0, e <- sent ? +0 : acc written back in place; Pici(sent) is what the
// three phases below then emit.  One pass over g and e instead of prune (read g, e; write sent, e) + compress (read
// sent): 12 instead of 20 bytes per element.
template <int DT, bool PRUNE>
__global__ void __launch_bounds__(kCompressWarps * 32, PRUNE ? 2 : CompressCfg<DT>::kMinBlocks)
compress_kernel(const Batch<CompressJob> batch) {
    static_assert(!PRUNE || DT == PICI_F32, "prune-and-compress is fp32");
    using Cfg = CompressCfg<DT>;
    using Elem = typename Cfg::Elem;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const CompressJob &job = batch.job[blockIdx.y];
    if (gate_closed(job.gate.ptr, job.gate.mask, job.gate.value)) return;
    const void *__restrict__ dense = job.dense;
    const uint64_t n = job.n;
    uint64_t *__restrict__ B = job.B;
    uint32_t *__restrict__ I = job.I;
    void *__restrict__ A = job.A;
    void *const ws = job.ws;
    uint64_t *const blk_acc = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(ws) + kWsHeaderBytes);
    uint64_t *const status = blk_acc + kWsAccWords;   // one tagged count per tile
    // [ticket, warps that have left] live behind the workspace header; the launch's last warp resets them and
    // advances the epoch, so no launch starts with a memset (status words carry the epoch, pici_common.cuh)
    uint32_t *const ticket = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + kWsCompressTicket);
    const uint32_t tag = launch_tag(ws);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    // tiles come from one of several ticket counters (pici_common.cuh "tile tickets from SEVERAL counters")
    const uint32_t T = (uint32_t)((n + kTile - 1) / kTile);
    const uint32_t worker_ctas = gridDim.x - 1u;            // CTA 0 of every job is the scan service
    if (blockIdx.x == 0) {
        __shared__ ScanShared scan_sh;
        if (threadIdx.x == 0) {
            scan_sh.seq = 0;
            scan_sh.base = 0;
        }
        __syncthreads();
        const uint32_t sbl = scan_block_log(worker_ctas * (uint32_t)kCompressWarps, Cfg::kScanBlockLog);
        scan_service(scan_sh, blk_acc, status, tag, T, sbl, I, nullptr, warp, kCompressWarps, lane);
        launch_exit(ws, ticket + 1, blk_acc, status, tag, T, sbl, gridDim.x * (uint32_t)kCompressWarps, lane);
        return;
    }
    const uint32_t cC = ticket_counters(worker_ctas * (uint32_t)kCompressWarps);
    const uint32_t cj = ((blockIdx.x - 1u) * (uint32_t)kCompressWarps + (uint32_t)warp) % cC;
    uint32_t *const tk = ticket_counter(ws, T, cj);
    Elem *stage = reinterpret_cast<Elem *>(smem_raw) + warp * Cfg::kStageElems;
    const uint32_t Tfull = (uint32_t)(n / kTile);
    Elem *Aout = reinterpret_cast<Elem *>(A);

    float *const resid = job.resid;
    float tau = 0.0f;
    if constexpr (PRUNE) tau = *job.d_tau;
    const float leak = job.leak;
    auto prune1 = [&](uint32_t gbits, uint32_t ebits, uint32_t &e_new) -> uint32_t {
        const float acc = __fadd_rn(__uint_as_float(gbits), __fmul_rn(leak, __uint_as_float(ebits)));
        const bool keep = fabsf(acc) >= tau;            // IEEE compare: a NaN is never sent
        e_new = keep ? 0u : __float_as_uint(acc);
        return keep ? __float_as_uint(acc) : 0u;
    };
    // Loads of a full tile: row r of the tile is one coalesced request; all 64 are issued back to back.
    auto load_full = [&](uint32_t tt, uint32_t (&v)[Cfg::kRegs]) {
        const size_t base = (size_t)tt * kTile;
        if constexpr (PRUNE) {
            const uint2 *pg = reinterpret_cast<const uint2 *>(reinterpret_cast<const uint32_t *>(dense) + base) + lane;
            uint2 *pe = reinterpret_cast<uint2 *>(reinterpret_cast<uint32_t *>(resid) + base) + lane;
            constexpr int kChunk = 16;                  // rows of g and e in flight together
#pragma unroll
            for (int c = 0; c < kSide / kChunk; ++c) {
                uint2 gg[kChunk], ee[kChunk];
#pragma unroll
                for (int j = 0; j < kChunk; ++j) {
                    gg[j] = ldg_stream_u2(pg + 32 * (kChunk * c + j));
                    ee[j] = ldg_stream_u2(pe + 32 * (kChunk * c + j));
                }
#pragma unroll
                for (int j = 0; j < kChunk; ++j) {
                    const int r = kChunk * c + j;
                    uint2 en;
                    v[2 * r] = prune1(gg[j].x, ee[j].x, en.x);
                    v[2 * r + 1] = prune1(gg[j].y, ee[j].y, en.y);
                    stg_stream_u2(pe + 32 * r, en);
                }
            }
        } else if constexpr (DT == PICI_F32) {
            const uint2 *p = reinterpret_cast<const uint2 *>(reinterpret_cast<const uint32_t *>(dense) + base) + lane;
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                uint2 x = ldg_stream_u2(p + 32 * r);
                v[2 * r] = x.x;
                v[2 * r + 1] = x.y;
            }
        } else {
            const uint32_t *p = reinterpret_cast<const uint32_t *>(reinterpret_cast<const uint16_t *>(dense) + base) + lane;
#pragma unroll
            for (int r = 0; r < kSide; ++r) v[r] = ldg_stream_u32(p + 32 * r);
        }
    };
    // Ragged last tile: elements >= n are virtual zeros (C9 #4); padded through the stage.
    auto load_ragged = [&](uint32_t tt, uint32_t (&v)[Cfg::kRegs]) {
        const size_t base = (size_t)tt * kTile;
        const Elem *p = reinterpret_cast<const Elem *>(dense);
        if constexpr (PRUNE) {
            uint32_t *pe = reinterpret_cast<uint32_t *>(resid);
            for (int i = lane; i < kTile; i += 32) {
                uint32_t s = 0;
                if (base + i < n) {
                    uint32_t en;
                    s = prune1(p[base + i], pe[base + i], en);
                    pe[base + i] = en;
                }
                stage[i] = s;
            }
        } else {
            for (int i = lane; i < kTile; i += 32) stage[i] = (base + i < n) ? p[base + i] : (Elem)0;
        }
        __syncwarp();
        if constexpr (DT == PICI_F32) {
            const uint2 *q = reinterpret_cast<const uint2 *>(stage) + lane;
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                uint2 x = q[32 * r];
                v[2 * r] = x.x;
                v[2 * r + 1] = x.y;
            }
        } else {
            const uint32_t *q = reinterpret_cast<const uint32_t *>(stage) + lane;
#pragma unroll
            for (int r = 0; r < kSide; ++r) v[r] = q[32 * r];
        }
        __syncwarp();
    };

    uint32_t v[Cfg::kRegs];
    uint32_t t = 0;
    if (lane == 0) t = ticket_tile(tk, cC, cj);
    t = __shfl_sync(kFull, t, 0);
    if (t < Tfull) load_full(t, v);
    else if (t < T) load_ragged(t, v);

    // Per-warp software pipeline.  A tile's count is published as soon as its data has arrived and Phase 1 is done; the
    // flush of its compacted values (which needs its prefix from the scan service) is deferred until kDefer later tiles
    // of this warp have published theirs, by which time the service has normally passed the tile's block.  The stage is
    // cut into kDefer + 1 slots for that; a tile with more values than a slot holds (denser than ~67 % sparsity) takes
    // the whole stage and everything pending is flushed first.
    constexpr uint32_t kSlot = Cfg::kStageElems / (kDefer + 1);
    uint32_t q_t[kDefer], q_n[kDefer], q_o[kDefer];   // pending tiles, oldest first: tile, count, stage offset
    bool q_on[kDefer];
#pragma unroll
    for (int i = 0; i < kDefer; ++i) q_on[i] = false;
    bool wide_pending = false;     // a pending tile lies across the slots
    uint32_t seq = 0;
    const uint32_t sb_log = scan_block_log(worker_ctas * (uint32_t)kCompressWarps, Cfg::kScanBlockLog);
    uint32_t held = 0xFFFFFFFFu;   // the tile this warp has claimed but not yet published (>= T: none)
    auto flush_one = [&](uint32_t pt, uint32_t pnnz, uint32_t off) {
        const uint32_t excl = service_prefix(blk_acc, status, I, tag, sb_log, pt, held, T, lane);
        Elem *dst = Aout + excl;
        const Elem *src = stage + off;
        for (uint32_t i = lane; i < pnnz; i += 32) dst[i] = src[i];
        __syncwarp();
    };
    auto flush_all = [&]() {       // oldest first
#pragma unroll
        for (int i = 0; i < kDefer; ++i) {
            if (q_on[i]) flush_one(q_t[i], q_n[i], q_o[i]);
            q_on[i] = false;
        }
        wide_pending = false;
    };
    auto push = [&](uint32_t pt, uint32_t pnnz, uint32_t off) {   // the oldest entry has been flushed: shift, append
#pragma unroll
        for (int i = 0; i + 1 < kDefer; ++i) {
            q_t[i] = q_t[i + 1]; q_n[i] = q_n[i + 1]; q_o[i] = q_o[i + 1]; q_on[i] = q_on[i + 1];
        }
        q_t[kDefer - 1] = pt; q_n[kDefer - 1] = pnnz; q_o[kDefer - 1] = off; q_on[kDefer - 1] = true;
    };

    uint32_t t_next = 0;  // next ticket (lane 0): requested right behind a tile's loads, it arrives while they do
    if (t < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
    while (t < T) {
        // ---- the next tile starts moving HBM -> L2 now, as ONE bulk prefetch of its 16 KB / 8 KB: the 64 row
        // loads issued at the end of this iteration then hit L2 ----
        const uint32_t tn = __shfl_sync(kFull, t_next, 0);
        held = tn;
        if (tn < Tfull && lane == 0) {
            const unsigned char *src = reinterpret_cast<const unsigned char *>(dense) + (size_t)tn * kTile * sizeof(Elem);
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"((uint32_t)(kTile * sizeof(Elem))) : "memory");
            if constexpr (PRUNE) {
                const unsigned char *se = reinterpret_cast<const unsigned char *>(resid) + (size_t)tn * kTile * sizeof(Elem);
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(se), "r"((uint32_t)(kTile * sizeof(Elem))) : "memory");
            }
        }

        // ---- Phase 1: column words (bit r <-> row r) and counts --------------------------------
        uint32_t w0lo = 0, w0hi = 0, w1lo = 0, w1hi = 0;
        if constexpr (DT == PICI_F32) {
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                if (nz32(v[2 * r])) w0lo |= 1u << r;
                if (nz32(v[2 * r + 1])) w1lo |= 1u << r;
                if (nz32(v[2 * r + 64])) w0hi |= 1u << r;
                if (nz32(v[2 * r + 65])) w1hi |= 1u << r;
            }
        } else {
            // both columns of a row in ONE compare: bf16x2 "unordered or not equal to 0" is the predicate C1 (x != 0:
            // +-0 false, NaN true, subnormals true - the compare does not flush) and returns 0xFFFF per true half;
            // 16 rows share an accumulator (bit r & 15: column 2l, bit 16 + (r & 15): column 2l + 1), four
            // accumulators are regrouped into the two 64-bit column words by byte permutes.  Two instructions per
            // row instead of four.
            uint32_t acc[4] = {0u, 0u, 0u, 0u};
            const __nv_bfloat162 zero2 = __float2bfloat162_rn(0.0f);
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                __nv_bfloat162 x;
                *reinterpret_cast<uint32_t *>(&x) = v[r];
                acc[r >> 4] |= __hneu2_mask(x, zero2) & (0x00010001u << (r & 15));
            }
            w0lo = __byte_perm(acc[0], acc[1], 0x5410);
            w1lo = __byte_perm(acc[0], acc[1], 0x7632);
            w0hi = __byte_perm(acc[2], acc[3], 0x5410);
            w1hi = __byte_perm(acc[2], acc[3], 0x7632);
        }
        const uint32_t cnt0 = __popc(w0lo) + __popc(w0hi);
        const uint32_t cnt1 = __popc(w1lo) + __popc(w1hi);
        const uint32_t incl = warp_incl_scan(cnt0 + cnt1, lane);
        const uint32_t tile_nnz = __shfl_sync(kFull, incl, 31);

        // ---- Phase 2: publish this tile's count for the scan service ----
        if (lane == 0) st_status(status + t, tag, tile_nnz);

        // B: lane l holds words 2l, 2l+1 -> one 16-byte store per lane, 512 contiguous bytes per warp
        {
            ulonglong2 w;
            w.x = ((uint64_t)w0hi << 32) | w0lo;
            w.y = ((uint64_t)w1hi << 32) | w1lo;
            reinterpret_cast<ulonglong2 *>(B + (size_t)t * kSide)[lane] = w;
        }

        // ---- Phase 3b of the tile kDefer iterations back: its prefix has had that long to arrive; a tile that does
        // not fit a slot, or follows one, needs the whole stage ----
        const bool wide = tile_nnz > kSlot;
        if (wide || wide_pending) flush_all();
        else if (q_on[0]) flush_one(q_t[0], q_n[0], q_o[0]);
        Elem *const stg = stage + (wide ? 0u : (seq % (kDefer + 1)) * kSlot);

        // ---- Phase 3a: compact into the warp's stage (tile-local offsets; order: column, row) ---
        if (tile_nnz <= Cfg::kRowSkipNnz) {
            // sparse tile: a row in which no lane holds a value (52 % of the rows at 99 % sparsity) costs one
            // uniform test instead of the bit tests of both columns; one pass, two cursors (column 2l, then 2l + 1)
            const uint32_t anylo = __reduce_or_sync(kFull, w0lo | w1lo), anyhi = __reduce_or_sync(kFull, w0hi | w1hi);
            uint32_t pos0 = incl - (cnt0 + cnt1), pos1 = pos0 + cnt0;
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                if (((r < 32 ? anylo : anyhi) >> (r & 31)) & 1u) {
                    if constexpr (DT == PICI_F32) {
                        if (nz32(v[2 * r])) stg[pos0++] = v[2 * r];
                        if (nz32(v[2 * r + 1])) stg[pos1++] = v[2 * r + 1];
                    } else {
                        if (nz16lo(v[r])) stg[pos0++] = (uint16_t)v[r];
                        if (nz16hi(v[r])) stg[pos1++] = (uint16_t)(v[r] >> 16);
                    }
                }
            }
        } else {
            uint32_t pos = incl - (cnt0 + cnt1);
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                if constexpr (DT == PICI_F32) {
                    if (nz32(v[2 * r])) stg[pos++] = v[2 * r];
                } else {
                    if (nz16lo(v[r])) stg[pos++] = (uint16_t)v[r];
                }
            }
#pragma unroll
            for (int r = 0; r < kSide; ++r) {
                if constexpr (DT == PICI_F32) {
                    if (nz32(v[2 * r + 1])) stg[pos++] = v[2 * r + 1];
                } else {
                    if (nz16hi(v[r])) stg[pos++] = (uint16_t)(v[r] >> 16);
                }
            }
        }
        __syncwarp();
        push(t, tile_nnz, (uint32_t)(stg - stage));
        wide_pending = wide;
        ++seq;

        if (tn < Tfull) {
            load_full(tn, v);
        } else if (tn < T) {  // the ragged tile is padded through the stage: flush first
            flush_all();
            load_ragged(tn, v);
        }
        t = tn;
        if (t < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
    }
    held = 0xFFFFFFFFu;
    flush_all();
    launch_exit(ws, ticket + 1, blk_acc, status, tag, T, sb_log, gridDim.x * (uint32_t)kCompressWarps, lane);
}

int num_sms() {
    static std::atomic<int> cached[64];
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    int v = cached[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        if (v <= 0) v = 148;
        cached[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

// Scratch for the scans (layout: pici_common.cuh): header, reduce_ss's accumulators, one word per tile.
uint64_t scan_workspace_bytes(uint64_t n) {
    const uint64_t T = (n + kTile - 1) / kTile;
#if PICI_TICKET_OLD
    return tile_words_end(T) + 1024;
#endif
    return tile_words_end(T);   // header (with the ticket counters), accumulators, per-tile words (multiple of 16)
}

template <int DT>
static cudaError_t launch_compress_t(const CompressJob *jobs, int count, cudaStream_t s) {
    using Cfg = CompressCfg<DT>;
    const size_t smem = (size_t)kCompressWarps * Cfg::kStageElems * sizeof(typename Cfg::Elem);
    static std::atomic<bool> configured_on[64];   // one-time setup per device; doing it twice is harmless
    std::atomic<bool> &configured = configured_on[current_device_slot()];
    if (!configured.load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(compress_kernel<DT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured.store(true, std::memory_order_release);
    }
    Batch<CompressJob> batch;
    uint64_t T = 0;
    for (int j = 0; j < count; ++j) {
        batch.job[j] = jobs[j];
        T = max(T, (jobs[j].n + kTile - 1) / kTile);
    }
    uint64_t blocks = (T + kCompressWarps - 1) / kCompressWarps + 1;   // + the scan service (CTA 0 of every job)
    const uint64_t cap = max((uint64_t)num_sms() * Cfg::kMinBlocks / count, (uint64_t)2);   // persistent: one resident wave
    if (blocks > cap) blocks = cap;
    compress_kernel<DT, false><<<dim3((unsigned)blocks, (unsigned)count), kCompressWarps * 32, smem, s>>>(batch);
    return cudaGetLastError();
}

cudaError_t launch_prune_compress(const CompressJob &job, cudaStream_t s) {
    const size_t smem = (size_t)kCompressWarps * kTile * sizeof(uint32_t);
    static std::atomic<bool> configured_on[64];
    std::atomic<bool> &configured = configured_on[current_device_slot()];
    if (!configured.load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(compress_kernel<PICI_F32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured.store(true, std::memory_order_release);
    }
    Batch<CompressJob> batch;
    batch.job[0] = job;
    const uint64_t T = (job.n + kTile - 1) / kTile;
    uint64_t blocks = (T + kCompressWarps - 1) / kCompressWarps + 1;   // + the scan service
    const uint64_t cap = (uint64_t)num_sms() * 2;
    if (blocks > cap) blocks = cap;
    compress_kernel<PICI_F32, true><<<dim3((unsigned)blocks, 1u), kCompressWarps * 32, smem, s>>>(batch);
    return cudaGetLastError();
}

// jobs with n == 0 are not supported here (the single entry point handles them)
cudaError_t launch_compress_batch(const CompressJob *jobs, int count, int dtype, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (count > kMaxBatch) return cudaErrorInvalidValue;
    return dtype == PICI_F32 ? launch_compress_t<PICI_F32>(jobs, count, s) : launch_compress_t<PICI_BF16>(jobs, count, s);
}

cudaError_t launch_compress(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                            void *ws, Gate g, cudaStream_t s) {
    if (n == 0) return launch_set_u32(I, 0u, g, s);
    const CompressJob job = {dense, n, B, I, A, ws, g, nullptr, nullptr, 0.0f};
    return launch_compress_batch(&job, 1, dtype, s);
}

}  // namespace pici
