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

// ---- single-pass device-wide exclusive scan of per-tile counts: decoupled look-back ------------
// One 64-bit status word per tile: high 32 bits = flag, low 32 bits = value.  Flag and value travel
// in ONE 64-bit access, so relaxed gpu-scope accesses are sufficient (no other data is published
// through the flag).  Workspace header word 0 is the dynamic tile ticket: a warp only ever waits on
// tiles with a SMALLER ticket, all of which are already owned by running warps, so forward progress
// does not depend on how many CTAs are co-resident.
constexpr uint64_t kStEmpty = 0, kStAggregate = 1, kStPrefix = 2;
constexpr int kWsHeaderBytes = 128;

__device__ __forceinline__ uint64_t ld_status(const uint64_t *p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(uint64_t *p, uint64_t flag, uint32_t value) {
    uint64_t v = (flag << 32) | value;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Warp-collective, step 1: make tile t's count visible to its successors as early as possible
// (tile 0 publishes its inclusive prefix straight away).
__device__ __forceinline__ void publish_aggregate(uint64_t *status, uint32_t t, uint32_t count, int lane) {
    if (lane == 0) st_status(status + t, t == 0 ? kStPrefix : kStAggregate, count);
}

// Warp-collective, step 2 (after publish_aggregate): returns the exclusive prefix (sum of the counts
// of tiles 0..t-1) and publishes tile t's inclusive prefix.  All 32 lanes call it with the same
// arguments.
__device__ __forceinline__ uint32_t lookback_exclusive(uint64_t *status, uint32_t t, uint32_t count,
                                                       int lane) {
    if (t == 0) return 0;
    uint32_t excl = 0;
    int64_t pos = (int64_t)t - 1;  // nearest predecessor examined by lane 0
    for (;;) {
        const int64_t idx = pos - lane;
        uint32_t sum = 0;
        bool found_prefix = false;
        for (;;) {
            uint64_t s = (idx >= 0) ? ld_status(status + idx) : (kStPrefix << 32);
            const uint32_t flag = (uint32_t)(s >> 32);
            const unsigned ready = __ballot_sync(kFull, flag != (uint32_t)kStEmpty);
            const unsigned pref = __ballot_sync(kFull, flag == (uint32_t)kStPrefix);
            if (pref != 0) {
                const int first = __ffs(pref) - 1;  // nearest predecessor that carries a prefix
                const unsigned need = (first == 31) ? kFull : ((2u << first) - 1u);
                if ((ready & need) == need) {
                    sum = warp_sum(lane <= first ? (uint32_t)s : 0u);
                    found_prefix = true;
                    break;
                }
            } else if (ready == kFull) {
                sum = warp_sum((uint32_t)s);
                break;
            }
            __nanosleep(32);
        }
        excl += sum;
        if (found_prefix) break;
        pos -= 32;
    }
    if (lane == 0) st_status(status + t, kStPrefix, excl + count);
    return excl;
}

// Dynamic tile ticket (one atomic per tile, issued by lane 0 and broadcast).
__device__ __forceinline__ uint32_t next_ticket(uint32_t *ticket, int lane) {
    uint32_t t = 0;
    if (lane == 0) t = atomicAdd(ticket, 1u);
    return __shfl_sync(kFull, t, 0);
}

}  // namespace pici
