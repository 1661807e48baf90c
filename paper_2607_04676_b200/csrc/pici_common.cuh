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
// One 64-bit status word per tile: high 32 bits = flag, low 32 bits = value; flag and value travel in
// ONE 64-bit access, so relaxed gpu-scope accesses suffice (nothing else is published through it).
//
// Decoupled look-back, with the look-back itself decoupled from the workers: every worker warp only
// PUBLISHES its tile count (flag kStCount) and later waits on its OWN word; one dedicated scanner warp
// (block 0) walks the status array in tile order, kScanRows*32 words per round, and replaces each
// count by the tile's exclusive prefix (flag kStPrefix), writing I[] as it goes.  The scan is
// ~T additions in total, so one warp keeps up with tiles retiring at HBM speed, and the polling
// traffic is one word per waiting warp instead of a 32-word window per warp.
// Tiles are handed out by a dynamic ticket, so every tile below the highest ticket is owned by a
// resident warp; the scanner block is block 0 of a grid that is sized to be fully resident.
constexpr uint64_t kStEmpty = 0, kStCount = 1, kStPrefix = 2;
constexpr int kWsHeaderBytes = 128;
#ifndef PICI_SCAN_ROWS
#define PICI_SCAN_ROWS 4
#endif
constexpr int kScanRows = PICI_SCAN_ROWS;

__device__ __forceinline__ uint64_t ld_status(const uint64_t *p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(uint64_t *p, uint64_t flag, uint32_t value) {
    uint64_t v = (flag << 32) | value;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Worker, step 1 (warp-collective): make tile t's count visible to the scanner.
__device__ __forceinline__ void publish_count(uint64_t *status, uint32_t t, uint32_t count, int lane) {
    if (lane == 0) st_status(status + t, kStCount, count);
}

// Worker, step 2 (warp-collective): the exclusive prefix of tile t (sum of the counts of tiles 0..t-1).
__device__ __forceinline__ uint32_t wait_prefix(const uint64_t *status, uint32_t t, int lane) {
    uint32_t excl = 0;
    if (lane == 0) {
        uint64_t s = ld_status(status + t);
        unsigned ns = 20;
        while ((uint32_t)(s >> 32) != (uint32_t)kStPrefix) {
            __nanosleep(ns);
            if (ns < 160) ns += ns;
            s = ld_status(status + t);
        }
        excl = (uint32_t)s;
    }
    return __shfl_sync(kFull, excl, 0);
}

// The scanner warp.  Writes I[0..T] (I[T] = total nnz).
__device__ __forceinline__ void scanner_warp(uint64_t *status, uint32_t T, uint32_t *__restrict__ I, int lane) {
    uint32_t pos = 0, run = 0;
    unsigned ns = 20;
    while (pos < T) {
        uint64_t st[kScanRows];
#pragma unroll
        for (int j = 0; j < kScanRows; ++j) {
            const uint32_t idx = pos + 32 * j + lane;
            st[j] = idx < T ? ld_status(status + idx) : 0ull;
        }
        uint32_t nready = 0;
        bool open = true;
#pragma unroll
        for (int j = 0; j < kScanRows; ++j) {
            const unsigned m = __ballot_sync(kFull, (uint32_t)(st[j] >> 32) == (uint32_t)kStCount);
            if (open) {
                const uint32_t lead = (m == kFull) ? 32u : (uint32_t)(__ffs(~m) - 1);
                nready += lead;
                open = (lead == 32u);
            }
        }
        if (nready == 0) {
            __nanosleep(ns);
            if (ns < 80) ns += ns;
            continue;
        }
        ns = 20;
#pragma unroll
        for (int j = 0; j < kScanRows; ++j) {
            if (32u * j < nready) {  // warp-uniform
                const uint32_t k = 32 * j + lane;
                const uint32_t c = k < nready ? (uint32_t)st[j] : 0u;
                const uint32_t incl = warp_incl_scan(c, lane);
                if (k < nready) {
                    const uint32_t excl = run + incl - c;
                    st_status(status + pos + k, kStPrefix, excl);
                    I[pos + k] = excl;
                }
                run += __shfl_sync(kFull, incl, 31);
            }
        }
        pos += nready;
    }
    if (lane == 0) I[T] = run;
}

// Dynamic tile ticket (one atomic per tile, issued by lane 0 and broadcast).
__device__ __forceinline__ uint32_t next_ticket(uint32_t *ticket, int lane) {
    uint32_t t = 0;
    if (lane == 0) t = atomicAdd(ticket, 1u);
    return __shfl_sync(kFull, t, 0);
}

}  // namespace pici
