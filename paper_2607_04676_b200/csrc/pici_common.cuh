// pici_common.cuh - device-side helpers shared by the Pici kernels (sm_100a).
//
// Format and predicate: include/pici.h.
// Nothing here is shared with oracle/ - the oracle is plain C and includes none of this.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace pici {

constexpr int kTile = 4096;           // k = 4096 elements per virtual tile
constexpr int kSide = 64;             // 64 x 64, row-major
constexpr unsigned kFull = 0xFFFFFFFFu;

template <int DT> struct ElemOf;
template <> struct ElemOf<0> { using type = uint32_t; };   // PICI_F32: raw fp32 bits
template <> struct ElemOf<1> { using type = uint16_t; };   // PICI_BF16: raw bf16 bits

// ---- nonzero predicate on raw bits (C1): IEEE x != 0 ------------------------------------------
__device__ __forceinline__ bool nz32(uint32_t u) { return (u & 0x7FFFFFFFu) != 0u; }
__device__ __forceinline__ bool nz16lo(uint32_t u) { return (u & 0x00007FFFu) != 0u; }
__device__ __forceinline__ bool nz16hi(uint32_t u) { return (u & 0x7FFF0000u) != 0u; }

// ---- bf16 arithmetic of the reductions (include/pici.h: add in fp32, round to nearest even) -----------------------
// A bf16 is the high half of an fp32, so widening is exact; the sum takes ONE fp32 rounding (__fadd_rn) and one
// rounding to bf16 (ties to even); a NaN sum stays a (quiet) NaN with the sum's sign and high payload bits.
__device__ __forceinline__ uint32_t bf16_add_bits(uint32_t a16, uint32_t b16) {   // operands and result in the low 16 bits
    const uint32_t u = __float_as_uint(__fadd_rn(__uint_as_float(a16 << 16), __uint_as_float(b16 << 16)));
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (u >> 16) | 0x0040u;
    return (u + 0x7FFFu + ((u >> 16) & 1u)) >> 16;
}

// ---- streaming global accesses ---------------------------------------------------------------
__device__ __forceinline__ uint2 ldg_stream_u2(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ uint32_t ldg_stream_u32(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ldg_stream_u4(const uint4 *p) {  // coherent (buffer may be written later)
    uint4 v;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ldg_nc_u4(const uint4 *p) {      // read-only for the whole kernel
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void stg_stream_u4(uint4 *p, uint4 v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void stg_stream_u2(uint2 *p, uint2 v) {
    asm volatile("st.global.cs.v2.u32 [%0], {%1, %2};" ::"l"(p), "r"(v.x), "r"(v.y) : "memory");
}
__device__ __forceinline__ void stg_stream_u32(uint32_t *p, uint32_t v) {
    asm volatile("st.global.cs.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- warp scans --------------------------------------------------------------------------------
// Inclusive prefix sum over the 32 lanes (Hillis-Steele with shuffles, as PAPER.md:191 Phase 3).
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t o = __shfl_up_sync(kFull, v, d);
        if (lane >= d) v += o;
    }
    return v;
}
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
    return v;
}

// ---- gate (include/pici.h "Gating") ------------------------------------------------------------
__device__ __forceinline__ bool gate_closed(const int32_t *gate, int32_t mask, int32_t value) {
    return gate != nullptr && (*reinterpret_cast<const volatile int32_t *>(gate) & mask) != value;
}

// ---- single-pass device-wide exclusive scan of per-tile counts (Phase 2) ------------------------
// Decoupled look-back at TILE granularity (one partition = one 64x64 tile = one warp's unit of work).
// One 64-bit status word per tile: high 32 bits = flag, low 32 bits = value; flag and value travel in
// ONE 64-bit access, so relaxed gpu-scope accesses suffice (nothing else is published through it).
//   aggregate : value = nnz of the tile               (published right after Phase 1)
//   prefix    : value = nnz of tiles 0..t inclusive   (published after the tile's look-back)
// A tile's look-back reads the 32 status words before it in one coalesced request (lane l <-> tile
// pos-1-l), takes everything up to the closest prefix, or - if the window holds aggregates only -
// adds all 32 and moves one window further back.  Aggregates do not depend on any other tile, so a
// look-back never waits on another look-back, only on Phase 1 of earlier tiles; tiles are handed out
// by a dynamic ticket, so every earlier tile is owned by a warp that is already running (forward
// progress without any residency assumption).  All sums are integers: the result does not depend on
// scheduling.
// Status words are tagged with the launch epoch kept in the workspace header (WsHeader below), so a workspace
// is never cleared between launches: high 32 bits = 1 (bit 31) | kind (bit 30: 0 aggregate, 1 prefix) | epoch tag
// (30 bits), low 32 bits = value.  A word of an earlier launch (or a zero word) never carries the current tag.
constexpr uint32_t kTagValid = 0x80000000u, kTagPrefix = 0x40000000u, kTagMask = 0x3FFFFFFFu;
// [0, 64): WsHeader; [64, 128): compress's exit counter; [128, 1152): the ticket counters (kTicketAreaBytes, below) - all
// at FIXED offsets: a workspace is shared by calls with different n, and what must be zero between launches may not
// lie where another call's per-tile words do
#ifndef PICI_TICKET_STRIDE
#define PICI_TICKET_STRIDE 128
#endif
constexpr int kWsHeaderBytes = 128 + 8 * PICI_TICKET_STRIDE;
constexpr int kWsCompressTicket = 64;
constexpr int kWsTicketArea = 128;
// Behind the header, at FIXED offsets (so that calls with different n can share a workspace): reduce_ss's
// accumulators - one word per 1024 tiles and one per 32 tiles, sized for the largest n (2^20 tiles), zero between
// launches - then one word per tile: compress's status words / reduce_ss's tagged tile counts.
constexpr uint32_t kWsBlkWords = 1024, kWsGrpWords = 32768, kWsAccWords = kWsBlkWords + kWsGrpWords;

struct WsHeader {             // first bytes of the workspace; persistent across launches (pici_workspace_init: 0)
    uint32_t epoch;           // tag of the last finished launch (compress and reduce_ss share it)
    uint32_t ticket;          // reduce_ss: next block
    uint32_t finished;        // reduce_ss: flusher warps that have left
    uint32_t high_words;      // the most per-tile words any launch on this workspace has used (for the wrap, below)
};
// Tag of the launch that starts now (read by every thread at kernel entry; 1 .. kTagMask).
__device__ __forceinline__ uint32_t launch_tag(const void *ws) {
    const uint32_t e = *reinterpret_cast<const volatile uint32_t *>(ws);
    return kTagValid | ((e + 1u) & kTagMask);
}
// The launch's last warp: every tagged word of an earlier launch is stale from now on.  When the 30-bit tag is
// about to wrap, the tagged words are cleared first (once per 2^30 launches), by the calling warp - all the words ANY
// launch on this workspace has used (the header keeps the high-water mark: calls with different n share a
// workspace, and a word a larger call tagged 2^30 launches ago must not meet its tag again).
__device__ __forceinline__ void finish_epoch(void *ws, uint32_t tag, uint64_t *tagged, uint64_t words, int lane) {
    WsHeader *h = reinterpret_cast<WsHeader *>(ws);
    uint32_t e = tag & kTagMask;
    const uint32_t high = max(*reinterpret_cast<volatile uint32_t *>(&h->high_words), (uint32_t)words);
    if (e == kTagMask) {
        for (uint64_t q = lane; q < high; q += 32) tagged[q] = 0;
        e = 0;
    }
    __syncwarp();
    if (lane == 0) {
        *reinterpret_cast<volatile uint32_t *>(&h->high_words) = high;
        __threadfence();
        *reinterpret_cast<volatile uint32_t *>(ws) = e;
    }
}

__device__ __forceinline__ uint64_t ld_status(const uint64_t *p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(uint64_t *p, uint64_t tag, uint32_t value) {
    uint64_t v = (tag << 32) | value;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Step 1 (warp-collective): make tile t's count visible.  Tile 0 has no predecessor: its aggregate
// is its inclusive prefix.
__device__ __forceinline__ void publish_count(uint64_t *status, uint32_t tag, uint32_t t, uint32_t count, int lane) {
    if (lane == 0) st_status(status + t, t == 0 ? (tag | kTagPrefix) : tag, count);
}

// Step 2 (warp-collective): exclusive prefix of tile t = sum of the counts of tiles 0..t-1; publishes
// the tile's inclusive prefix and writes I[t] (and I[T] from the last tile).
// `first` / `have_first`: the status words of the first window (lane l <-> tile t-1-l), loaded by the caller well
// ahead (lookback_peek) so that their L2 round trip is off the warp's critical path; a window that is not complete
// yet is simply loaded again.
__device__ __forceinline__ uint64_t lookback_peek(const uint64_t *status, uint32_t tag, uint32_t t, int lane) {
    const int64_t idx = (int64_t)t - 1 - lane;
    return idx >= 0 ? ld_status(status + idx) : ((uint64_t)(tag | kTagPrefix) << 32);
}
__device__ __forceinline__ uint32_t lookback_prefix(uint64_t *status, uint32_t tag, uint32_t t, uint32_t count, uint32_t T,
                                                    uint32_t *__restrict__ I, int lane, uint64_t first = 0,
                                                    bool have_first = false) {
    uint32_t excl = 0;
    int64_t pos = t;  // tiles [0, pos) are not yet accounted for
    while (pos > 0) {  // warp-uniform
        const int64_t idx = pos - 1 - lane;
        uint64_t s;
        unsigned pm, em;
        unsigned ns = 8;
        for (;;) {
            if (have_first) s = first;
            else s = idx >= 0 ? ld_status(status + idx) : ((uint64_t)(tag | kTagPrefix) << 32);
            const uint32_t hi = (uint32_t)(s >> 32);
            const bool valid = (hi & ~kTagPrefix) == tag;
            pm = __ballot_sync(kFull, valid && (hi & kTagPrefix) != 0u);
            em = __ballot_sync(kFull, !valid);
            // lanes that matter: up to and including the closest prefix (all 32 if there is none)
            const unsigned rel = pm ? ((pm & (0u - pm)) | ((pm & (0u - pm)) - 1u)) : kFull;
            if ((em & rel) == 0u) {
                const uint32_t v = ((1u << lane) & rel) ? (uint32_t)s : 0u;
                excl += warp_sum(v);
                have_first = false;
                break;
            }
            if (!have_first) {
                __nanosleep(ns);
                if (ns < 64) ns += ns;
            }
            have_first = false;
        }
        if (pm) break;
        pos -= 32;
    }
    if (lane == 0) {
        if (t != 0) st_status(status + t, tag | kTagPrefix, excl + count);
        I[t] = excl;
        if (t + 1 == T) I[T] = excl + count;
    }
    return excl;
}

constexpr uint64_t kOneAdd = 1ull << 48;
__device__ __forceinline__ void red_add_u64(uint64_t *p, uint64_t v) {
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---- store-only hierarchical exclusive scan of per-tile counts (reduce_ss, the COO merge) ---------------------------
// Three levels over tiles: one tagged word per tile, one accumulator per group of 32 tiles, one per block of 1024
// tiles, each accumulator (tiles << 48) + count, added to by 64-bit red.add and zero between launches (the launch's
// last warp clears them).  prefix(t0) = [complete 1024-blocks below, carried in E / E_blk from call to call: t0 must
// not decrease per warp] + [complete groups below inside the own block] + [tiles below inside the own group]: three
// independent sets of loads, each word says by itself whether it is complete, so a prefix only ever waits for COUNTS
// of lower tiles - never for another prefix - and there is no chain of look-backs however many tiles are in flight.
__device__ __forceinline__ bool tagged(uint64_t v, uint32_t tag) { return (uint32_t)(v >> 32) == tag; }
__device__ __forceinline__ void hier_publish(uint64_t *blk_acc, uint64_t *grp_acc, uint64_t *tile_word, uint32_t tag,
                                             uint32_t t, uint32_t count) {   // one lane
    st_status(tile_word + t, tag, count);
    const uint64_t v = kOneAdd + count;
    red_add_u64(grp_acc + (t >> 5), v);
    red_add_u64(blk_acc + (t >> 10), v);
}
__device__ __forceinline__ uint32_t hier_prefix(const uint64_t *blk_acc, const uint64_t *grp_acc, const uint64_t *tile_word,
                                                uint32_t tag, uint32_t t0, uint32_t &E, uint32_t &E_blk, int lane) {
    const uint32_t u = t0 & 31u, grp = (t0 >> 5) & 31u, blk = t0 >> 10, gbase = t0 & ~31u;
    uint64_t va, vg, vb = 0;
    unsigned ns = 8;
    for (;;) {
        va = (uint32_t)lane < u ? ld_status(tile_word + gbase + lane) : ((uint64_t)tag << 32);
        vg = (uint32_t)lane < grp ? ld_status(grp_acc + blk * 32u + lane) : (32ull << 48);
        const bool more = E_blk + (uint32_t)lane < blk;
        vb = more ? ld_status(blk_acc + E_blk + lane) : (1024ull << 48);
        if (__all_sync(kFull, tagged(va, tag) && (vg >> 48) == 32u && (vb >> 48) == 1024u)) break;
        __nanosleep(ns);
        if (ns < 128) ns += ns;
    }
    const uint32_t nb = min(32u, blk - E_blk);
    E += __reduce_add_sync(kFull, (uint32_t)lane < nb ? (uint32_t)vb : 0u);
    E_blk += nb;
    while (E_blk < blk) {   // more than 32 new blocks since this warp's last prefix (first call on a huge input)
        const uint32_t c = min(32u, blk - E_blk);
        uint64_t v;
        for (;;) {
            v = (uint32_t)lane < c ? ld_status(blk_acc + E_blk + lane) : (1024ull << 48);
            if (__all_sync(kFull, (v >> 48) == 1024u)) break;
            __nanosleep(64);
        }
        E += __reduce_add_sync(kFull, (uint32_t)lane < c ? (uint32_t)v : 0u);
        E_blk += c;
    }
    return E + __reduce_add_sync(kFull, (uint32_t)va + (uint32_t)vg);
}

// ---- Phase 2 as a service ---------------------------------------------------------------------------------------------
// The device-wide exclusive scan of the tile counts is not taken by the warps that compress (a decoupled look-back
// cost them 3.5 - 4.7 dependent L2 round trips per tile: the whole gap between 0.79 and 1.03 of the HBM peak) but by
// the warps of CTA 0: warp w takes the scan blocks b = w, w + nwarps, ...; it waits until the block's counts are
// all published (tickets hand tiles out in order, so that is when the front of the launch has passed it), scans them
// (32 coalesced 256-byte rows of status words, a warp scan per row), receives the block's base from the warp that
// scanned block b - 1 through shared memory, writes I for the block - I itself is the result -, turns every tile's
// status word into its exclusive prefix (flag kTagPrefix) and marks the block done (a tagged word that carries the
// prefix at the block's end).  A compressing warp flushes a tile two iterations after publishing its count; by then
// the service has normally passed and the flush costs ONE load - the tile's own word (done word, then I[t]: two
// dependent L2 round trips per tile, was 0.95 / 0.72 of the peak for fp32 at 50 % / bf16 at 99 %; one: 1.02 / 0.76).
struct ScanShared {
    volatile uint32_t seq;    // blocks whose base has been handed on
    volatile uint32_t base;   // exclusive prefix of block `seq`
};
// log2 of the scan block: 256 tiles (fp32) / 512 (bf16) for a full-size launch - measured at N = 2^28, 99 %: blocks of
// 256 / 512 / 1024 tiles give fp32 0.169 / 0.169 / 0.177 ms and bf16 0.180 / 0.137 / 0.156 (small blocks: the service's
// four warps, one L2 round trip per poll, fall behind bf16's tile rate; large blocks: a tile waits longer for the rest
// of its block, and at 50 % sparsity, where a tile is flushed one iteration after its publish, 512 / 1024 stall:
// fp32 0.270 / 0.519 / 0.628) - smaller when the launch has few warps, so that the tiles one warp takes one after the
// other (about `warps` apart) fall into different blocks (see service_prefix)
__device__ __forceinline__ uint32_t scan_block_log(uint32_t worker_warps, uint32_t max_log) {
    const uint32_t half = max(worker_warps / 2u, 32u);
    return min(31u - (uint32_t)__clz(half), max_log);
}
__device__ __forceinline__ void scan_service(ScanShared &sh, uint64_t *blk_done, uint64_t *status, uint32_t tag,
                                             uint32_t T, uint32_t sb_log, uint32_t *__restrict__ I, uint32_t *total_out, int warp, int nwarps,
                                             int lane) {
    const uint32_t sb = 1u << sb_log, rows = sb >> 5;
    const uint32_t nblk = (T + sb - 1u) >> sb_log;
    for (uint32_t b = (uint32_t)warp; b < nblk; b += (uint32_t)nwarps) {
        const uint32_t t0 = b << sb_log;
        uint32_t cnt[32];
        uint64_t w[32];
        // all rows are requested together (one L2 round trip for the block) and the whole block is read again until
        // every word carries the tag
        for (;;) {
            bool ok = true;
#pragma unroll
            for (int i = 0; i < 32; ++i) {      // row i: tiles t0 + 32 i + lane
                const uint32_t t = t0 + 32u * i + (uint32_t)lane;
                w[i] = ((uint32_t)i < rows && t < T) ? ld_status(status + t) : ((uint64_t)tag << 32);   // others count 0
            }
#pragma unroll
            for (int i = 0; i < 32; ++i) ok = ok && tagged(w[i], tag);
            if (__all_sync(kFull, ok)) break;
            __nanosleep(100);    // 100 / 500 / 2000 ns: fp32 0.266 / 0.272 / 0.312 ms at 50 % sparsity, no difference above
        }
#pragma unroll
        for (int i = 0; i < 32; ++i) cnt[i] = (uint32_t)w[i];
        uint32_t run = 0;                   // block-local exclusive prefixes, in place
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            if ((uint32_t)i < rows) {       // warp-uniform
                const uint32_t incl = warp_incl_scan(cnt[i], lane);
                const uint32_t tot = __shfl_sync(kFull, incl, 31);
                cnt[i] = run + incl - cnt[i];
                run += tot;
            }
        }
        uint32_t base = 0;
        if (lane == 0) {
            while (sh.seq != b) __nanosleep(32);
            base = sh.base;
            sh.base = base + run;           // hand the next block its base before the stores below
            __threadfence_block();
            sh.seq = b + 1u;
        }
        base = __shfl_sync(kFull, base, 0);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const uint32_t t = t0 + 32u * i + (uint32_t)lane;
            if ((uint32_t)i < rows && t < T) {
                I[t] = base + cnt[i];
                st_status(status + t, tag | kTagPrefix, base + cnt[i]);   // the tile's word now carries its prefix
            }
        }
        if (b + 1u == nblk && lane == 0) {
            I[T] = base + run;
            if (total_out != nullptr) *total_out = base + run;
        }
        // no fence: a flush takes its prefix from the tile's word and a self-scan the block's end from the done word -
        // each carries its value; I is read by later launches only
        if (lane == 0) st_status(blk_done + b, tag, base + run);   // done; the value is the prefix at the block's end
    }
}

// The worker's side: exclusive prefix of tile pt, which this warp published earlier.  `held` is the tile the warp has
// claimed but not yet published (>= T: none).  The scan service finishes a block only when EVERY tile of it has
// published its count - also the held one.  So the warp waits for the service only if that tile lies in a later block
// (blocks then resolve in increasing order: no cycle); otherwise - small launches, the tail of a launch - it takes the
// prefix itself: the end of the block below plus the counts of the tiles of its own block below pt (all of them lower
// than anything this warp holds).
__device__ __forceinline__ uint32_t service_wait_done(const uint64_t *blk_done, uint32_t tag, uint32_t b) {
    unsigned ns = 16;
    uint64_t v;
    while (!tagged(v = ld_status(blk_done + b), tag)) {
        __nanosleep(ns);
        if (ns < 128) ns += ns;
    }
    return (uint32_t)v;   // the prefix at the end of scan block b
}
__device__ __forceinline__ uint32_t service_prefix(const uint64_t *blk_done, const uint64_t *status, const uint32_t *I,
                                                   uint32_t tag, uint32_t sb_log, uint32_t pt, uint32_t held, uint32_t T,
                                                   int lane) {
    const uint32_t bq = pt >> sb_log;
    uint32_t excl;
    if (held >= T || bq < (held >> sb_log)) {
        unsigned ns = 16;
        uint64_t v;
        while ((uint32_t)((v = ld_status(status + pt)) >> 32) != (tag | kTagPrefix)) {   // ONE load when the service has passed
            __nanosleep(ns);
            if (ns < 128) ns += ns;
        }
        excl = (uint32_t)v;
    } else {
        excl = bq ? service_wait_done(blk_done, tag, bq - 1u) : 0u;
        uint32_t part = 0;
        for (uint32_t u0 = bq << sb_log; u0 < pt; u0 += 32u) {
            const uint32_t u = u0 + (uint32_t)lane;
            uint64_t v = (uint64_t)tag << 32;
            if (u < pt) {
                unsigned ns = 16;
                while (!tagged(v = ld_status(status + u), tag)) {
                    __nanosleep(ns);
                    if (ns < 128) ns += ns;
                }
            }
            part += (uint32_t)v;
        }
        excl += warp_sum(part);
    }
    return excl;
}

// ---- TMA 1-D bulk copy global -> shared, completion on an mbarrier (UBLKCP in SASS) -------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// dst (shared), src (global) 16-byte aligned, bytes a non-zero multiple of 16.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// Orders earlier generic-proxy accesses to shared memory before later async-proxy (TMA) ones.
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- tile tickets from SEVERAL counters ------------------------------------------------------------------------------
// One ticket per tile from ONE counter is what bounded every tile-per-warp kernel of this library: ~1800 resident warps
// each keep one atomic on the same address in flight, the L2 serves them at ~3 ns apiece under load, so a ticket takes
// ~5 us to return and 65 536 of them take 0.2 ms - exactly compress's run time at every sparsity from 95 % up.  (A bare
// kernel that only reads 1 GiB tile by tile: 5.2 TB/s with one counter, 7.2 TB/s with four or more.)  So there are
// kTicketCounters counters, 128 bytes apart, in the tail of the workspace header (zero between launches: the
// launch's last warp clears them again); warp w draws from counter w mod kTicketCounters,
// and ticket k of counter j is tile C * k + j (C = kTicketCounters, or the number of warps of the launch if that is smaller:
// every counter needs a warp).  Each counter's tiles increase, the counters advance at
// about the same pace, and the smallest unclaimed tile always belongs to a group whose warps only wait for claimed
// tiles - forward progress is as with one counter.
constexpr uint32_t kTicketCounters = 8;
constexpr uint32_t kTicketAreaBytes = kTicketCounters * (uint32_t)PICI_TICKET_STRIDE;
static_assert(kWsTicketArea + (int)kTicketAreaBytes == kWsHeaderBytes, "ticket counters fill the header's tail");
__host__ __device__ __forceinline__ uint64_t tile_words_end(uint64_t T) {   // bytes from the start of the workspace
    return (uint64_t)kWsHeaderBytes + ((uint64_t)kWsAccWords + ((T + 65) & ~1ull)) * 8;
}
__device__ __forceinline__ uint32_t *ticket_counter(void *ws, uint32_t T, uint32_t j) {
#if PICI_TICKET_OLD
    return reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + tile_words_end(T)) + 32u * j;
#else
    (void)T;
    return reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + kWsTicketArea) + (uint32_t)(PICI_TICKET_STRIDE / 4) * j;
#endif
}
__device__ __forceinline__ uint32_t ticket_counters(uint32_t warps_in_launch) { return min(kTicketCounters, warps_in_launch); }
__device__ __forceinline__ uint32_t ticket_tile(uint32_t *counter, uint32_t C, uint32_t j) {   // one lane
    return atomicAdd(counter, 1u) * C + j;
}
__device__ __forceinline__ void ticket_reset(void *ws, uint32_t T, int lane) {     // the launch's last warp
    if ((uint32_t)lane < kTicketCounters) *ticket_counter(ws, T, (uint32_t)lane) = 0u;
}

// Every warp of a tile-ticket launch - the compressing warps AND the warps of the scan service - leaves through here.
// The last one clears what must be zero between launches (ticket counters, the exit counter, the service's done words:
// that area is reduce_ss's accumulators) and advances the epoch.  The service's warps count too: a compressing warp
// can take its last prefix from a tile word and leave before the service has stored that block's done word, and a
// done word stored after the clear would stay behind.
#ifndef PICI_EXIT_INLINE
#define PICI_EXIT_INLINE __noinline__
#endif
static __device__ PICI_EXIT_INLINE void launch_exit(void *ws, uint32_t *exit_counter, uint64_t *blk_done, uint64_t *status, uint32_t tag,
                                            uint32_t T, uint32_t sb_log, uint32_t warps_in_launch, int lane) {
    uint32_t last = 0;
    if (lane == 0) {
        __threadfence();
        last = atomicAdd(exit_counter, 1u) + 1u == warps_in_launch;
    }
    if (__shfl_sync(kFull, last, 0)) {
        __threadfence();
        ticket_reset(ws, T, lane);
        if (lane == 0) *exit_counter = 0;
        for (uint32_t q = lane; q < ((T + (1u << sb_log) - 1u) >> sb_log); q += 32) blk_done[q] = 0;
        finish_epoch(ws, tag, status, T, lane);
    }
}

// Dynamic tile ticket (one atomic per tile, issued by lane 0 and broadcast).
__device__ __forceinline__ uint32_t next_ticket(uint32_t *ticket, int lane) {
    uint32_t t = 0;
    if (lane == 0) t = atomicAdd(ticket, 1u);
    return __shfl_sync(kFull, t, 0);
}

}  // namespace pici
