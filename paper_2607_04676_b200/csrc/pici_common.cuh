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
__device__ __forceinline__ bool gate_closed(const int32_t *gate, int32_t gate_value) {
    return gate != nullptr && *reinterpret_cast<const volatile int32_t *>(gate) != gate_value;
}

// ---- single-pass device-wide exclusive scan of per-tile counts (Phase 2) ------------------------
// Decoupled look-back at TILE granularity (one partition = one 64x64 tile = one warp's unit of work).
// One 64-bit status word per tile: high 32 bits = flag, low 32 bits = value; flag and value travel in
// ONE 64-bit access, so relaxed gpu-scope accesses suffice (nothing else is published through it).
//   kStAggregate : value = nnz of the tile               (published right after Phase 1)
//   kStPrefix    : value = nnz of tiles 0..t inclusive   (published after the tile's look-back)
// A tile's look-back reads the 32 status words before it in one coalesced request (lane l <-> tile
// pos-1-l), takes everything up to the closest kStPrefix, or - if the window holds aggregates only -
// adds all 32 and moves one window further back.  Aggregates do not depend on any other tile, so a
// look-back never waits on another look-back, only on Phase 1 of earlier tiles; tiles are handed out
// by a dynamic ticket, so every earlier tile is owned by a warp that is already running (forward
// progress without any residency assumption).  All sums are integers: the result does not depend on
// scheduling.
constexpr uint64_t kStEmpty = 0, kStAggregate = 1, kStPrefix = 2;
constexpr int kWsHeaderBytes = 128;       // [0, 64): reduce_ss's persistent header; [64, 128): compress's ticket
constexpr int kWsCompressTicket = 64;
// Behind the header, at FIXED offsets (so that calls with different n can share a workspace): reduce_ss's
// accumulators - one word per 1024 tiles and one per 32 tiles, sized for the largest n (2^20 tiles), zero between
// launches - then one word per tile: compress's status words / reduce_ss's tagged tile counts.
constexpr uint32_t kWsBlkWords = 1024, kWsGrpWords = 32768, kWsAccWords = kWsBlkWords + kWsGrpWords;

__device__ __forceinline__ uint64_t ld_status(const uint64_t *p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(uint64_t *p, uint64_t flag, uint32_t value) {
    uint64_t v = (flag << 32) | value;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Step 1 (warp-collective): make tile t's count visible.  Tile 0 has no predecessor: its aggregate
// is its inclusive prefix.
__device__ __forceinline__ void publish_count(uint64_t *status, uint32_t t, uint32_t count, int lane) {
    if (lane == 0) st_status(status + t, t == 0 ? kStPrefix : kStAggregate, count);
}

// Step 2 (warp-collective): exclusive prefix of tile t = sum of the counts of tiles 0..t-1; publishes
// the tile's inclusive prefix and writes I[t] (and I[T] from the last tile).
__device__ __forceinline__ uint32_t lookback_prefix(uint64_t *status, uint32_t t, uint32_t count, uint32_t T,
                                                    uint32_t *__restrict__ I, int lane) {
    uint32_t excl = 0;
    int64_t pos = t;  // tiles [0, pos) are not yet accounted for
    while (pos > 0) {  // warp-uniform
        const int64_t idx = pos - 1 - lane;
        uint64_t s;
        unsigned pm, em;
        unsigned ns = 8;
        for (;;) {
            s = idx >= 0 ? ld_status(status + idx) : (kStPrefix << 32);
            const uint32_t flag = (uint32_t)(s >> 32);
            pm = __ballot_sync(kFull, flag == (uint32_t)kStPrefix);
            em = __ballot_sync(kFull, flag == (uint32_t)kStEmpty);
            // lanes that matter: up to and including the closest prefix (all 32 if there is none)
            const unsigned rel = pm ? ((pm & (0u - pm)) | ((pm & (0u - pm)) - 1u)) : kFull;
            if ((em & rel) == 0u) {
                const uint32_t v = ((1u << lane) & rel) ? (uint32_t)s : 0u;
                excl += warp_sum(v);
                break;
            }
            __nanosleep(ns);
            if (ns < 64) ns += ns;
        }
        if (pm) break;
        pos -= 32;
    }
    if (lane == 0) {
        if (t != 0) st_status(status + t, kStPrefix, excl + count);
        I[t] = excl;
        if (t + 1 == T) I[T] = excl + count;
    }
    return excl;
}

// ---- round-robin scan: exclusive prefix of per-unit counts in ONE L2 round trip --------------------
// For persistent grids launched cooperatively (every worker resident) whose W workers take units
// round-robin: worker c handles units c, c + W, c + 2W, ...; "iteration" it covers units
// [it*W, (it+1)*W).  A worker publishes its unit's count as (a) a per-unit word (1 << 32 | count),
// (b) a 64-bit atomic add of (1 << 48) + count into the word of its group of 32 units and (c) into the
// word of its iteration; each word carries (number of adds, sum) in one 64-bit access, so relaxed
// gpu-scope accesses suffice.  prefix(it, c) = complete iterations below it + complete groups below
// c's + the units of c's own group below c: independent loads, 32 + 64 + 32 words at most.  The workers
// run nearly in lock-step, so a flat decoupled look-back would find no prefix among the W - 1 units
// of its own iteration and walk W / 32 dependent hops (measured in reduce_ss: ~8 us per iteration).
constexpr uint32_t kRoundRobinMaxUnits = 2048;   // W <= 2048: two group words per lane
struct RoundRobinScan {
    uint64_t *unit_word;   // [units]
    uint64_t *grp_word;    // [iterations][ngrp], ngrp = ceil(W / 32)
    uint64_t *iter_word;   // [iterations]
    uint32_t ngrp;
};
constexpr uint64_t kOneAdd = 1ull << 48;
__device__ __forceinline__ void red_add_u64(uint64_t *p, uint64_t v) {
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// One thread: publish the count of unit u = it * W + c.
__device__ __forceinline__ void rr_publish(const RoundRobinScan &sc, uint64_t u, uint32_t it, uint32_t c, uint32_t count) {
    st_status(sc.unit_word + u, 1u, count);
    red_add_u64(sc.grp_word + (size_t)it * sc.ngrp + (c >> 5), kOneAdd + count);
    red_add_u64(sc.iter_word + it, kOneAdd + count);
}
// One warp: sum of the counts of all units below (it, c).  E = running sum of the complete iterations
// [0, E_it), carried by the caller from call to call (up to 32 iteration words are added per call).
// All W units of an iteration below `it` exist, and so do all 32 units of a group below c's.
__device__ __forceinline__ uint32_t rr_lookback(const RoundRobinScan &sc, uint32_t W, uint32_t it, uint32_t c, uint32_t &E,
                                                uint32_t &E_it, int lane) {
    const uint32_t nfull = c >> 5, rem = c & 31u;
    const uint64_t *gw = sc.grp_word + (size_t)it * sc.ngrp;
    const uint64_t *uw = sc.unit_word + (size_t)it * W + (size_t)nfull * 32;
    while (E_it + 32 < it) {   // not taken when a worker sees consecutive iterations
        uint64_t v;
        do { v = ld_status(sc.iter_word + E_it); } while ((uint32_t)(v >> 48) != W);
        E += (uint32_t)v;
        ++E_it;
    }
    const uint32_t nit = it - E_it;
    uint64_t vi, vg, vh, vs;
    unsigned ns = 8;
    for (;;) {
        vi = (uint32_t)lane < nit ? ld_status(sc.iter_word + E_it + lane) : ((uint64_t)W << 48);
        vg = (uint32_t)lane < nfull ? ld_status(gw + lane) : (32ull << 48);
        vh = (uint32_t)lane + 32u < nfull ? ld_status(gw + 32 + lane) : (32ull << 48);
        vs = (uint32_t)lane < rem ? ld_status(uw + lane) : (1ull << 32);
        const bool ok = (uint32_t)(vi >> 48) == W && (uint32_t)(vg >> 48) == 32u && (uint32_t)(vh >> 48) == 32u &&
                        (uint32_t)(vs >> 32) != 0u;
        if (__all_sync(kFull, ok)) break;
        __nanosleep(ns);
        if (ns < 128) ns += ns;
    }
    E += warp_sum((uint32_t)vi);
    E_it = it;
    return E + warp_sum((uint32_t)vg + (uint32_t)vh + (uint32_t)vs);
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

// Dynamic tile ticket (one atomic per tile, issued by lane 0 and broadcast).
__device__ __forceinline__ uint32_t next_ticket(uint32_t *ticket, int lane) {
    uint32_t t = 0;
    if (lane == 0) t = atomicAdd(ticket, 1u);
    return __shfl_sync(kFull, t, 0);
}

}  // namespace pici
