// coo.cu - the COO variant (include/pici_coo.h): flat 32-bit index + fp32 value per
// nonzero, ascending index, structure of arrays, nnz in a device word.
//
// Layout of the work on B200.  The unit is the same 4096-element block Pici calls a tile (here just a contiguous
// index range [4096 t, 4096 t + 4096)), one warp per block:
//   * compress: the block sits in 128 registers per lane (32 rows of 128 elements, lane l holds elements
//     128 i + 4 l .. + 3 of row i: every row is one coalesced 512-byte request, all 32 in flight at once).  The
//     output order of COO is the input order, so the compaction offset inside a block is a running, warp-uniform
//     row base plus a popcount of four ballots: count and compaction are ONE pass into a shared-memory stage
//     (idx, val).  The block's count is published right after it; the device-wide exclusive scan is the same
//     single-pass decoupled look-back as pici_compress (pici_common.cuh), deferred behind the next block (two
//     stage buffers per warp), and the flush is coalesced.  A block with more entries than the stage holds (density
//     above 25 %, not a COO regime) takes its look-back at once and writes from registers;
//   * decompress / merge find a block's index range in `off` (off[t] = first entry with idx >= 4096 t), built by a
//     streaming pre-pass over idx (what Pici's I gives for free); decompress assembles the block in shared memory and
//     writes every dense byte once; the merge keeps two presence bitmaps per warp in shared memory, reads the values
//     from the lists at popcount-prefix cursors, re-applies the predicate to the sums and emits survivors in
//     ascending order behind a deferred look-back;
//   * reduce_sd is the bare read-modify-write of the touched elements.
#include <atomic>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"
#include "../../include/pici_coo.h"

namespace pici {

constexpr int kCooWarps = 4;
constexpr uint32_t kCooStage = 640;                  // entries a stage buffer holds before a block goes direct
constexpr int kCooBufs = 3;                          // stage buffers per warp: the block in hand + two whose flush is deferred
constexpr uint32_t kCooStageWords = kCooStage + 128; // + one row of slack (the check is per row)

struct CooWs {            // views into the caller's workspace (layout: coo_workspace_bytes)
    void *hdr;            // WsHeader + ticket / exit counter (pici_common.cuh)
    uint64_t *blk_acc, *grp_acc;   // the merge's accumulators (hier_prefix, pici_common.cuh), zero between launches
    uint64_t *status;     // [T] tagged look-back words (compress) / tagged counts (merge)
    uint32_t *excl;       // [T + 1] exclusive prefix per block (scratch the look-back writes)
    uint32_t *offx, *offy;// [T + 1] each
};

static uint64_t round16(uint64_t b) { return (b + 15) & ~15ull; }
uint64_t coo_workspace_bytes(uint64_t n) {
    const uint64_t T = (n + kTile - 1) / kTile;
    return scan_workspace_bytes(n) + 3 * round16((T + 1) * 4);
}
// The three scratch arrays lie at the END of the caller's buffer, not behind this call's tile words: a workspace is
// shared by calls with different n, and scratch data must not land where a larger call keeps tagged words.
static CooWs coo_ws(void *ws, uint64_t ws_bytes, uint64_t n) {
    const uint64_t T = (n + kTile - 1) / kTile;
    unsigned char *b = reinterpret_cast<unsigned char *>(ws);
    CooWs w;
    w.hdr = ws;
    w.blk_acc = reinterpret_cast<uint64_t *>(b + kWsHeaderBytes);
    w.grp_acc = w.blk_acc + kWsBlkWords;
    w.status = w.blk_acc + kWsAccWords;
    unsigned char *tail = b + ((ws_bytes & ~15ull) - 3 * round16((T + 1) * 4));
    w.excl = reinterpret_cast<uint32_t *>(tail);
    w.offx = reinterpret_cast<uint32_t *>(tail + round16((T + 1) * 4));
    w.offy = reinterpret_cast<uint32_t *>(tail + 2 * round16((T + 1) * 4));
    return w;
}

// ================================================ compress ================================================
struct CooCompressArgs {
    const uint32_t *dense;
    uint64_t n;
    uint32_t *idx, *val, *d_nnz;
    CooWs ws;
};

__global__ void __launch_bounds__(kCooWarps * 32, 3) coo_compress_kernel(const CooCompressArgs a) {
    extern __shared__ __align__(16) uint32_t coo_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // per warp: kCooBufs buffers of (idx[kCooStageWords], val[kCooStageWords])
    uint32_t *const stage = coo_smem + (size_t)warp * kCooBufs * 2 * kCooStageWords;
    uint32_t *const ticket = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(a.ws.hdr) + kWsCompressTicket);
    const uint32_t tag = launch_tag(a.ws.hdr);
    const uint64_t n = a.n;
    const uint32_t T = (uint32_t)((n + kTile - 1) / kTile), Tfull = (uint32_t)(n / kTile);
    const uint32_t lt = (1u << lane) - 1u;
    // Phase 2 is a service, as in pici_compress (pici_common.cuh): CTA 0 scans the published counts block by block and
    // writes the exclusive prefixes into ws.excl (and the total into *d_nnz); the other CTAs compress
    const uint32_t worker_ctas = gridDim.x - 1u;
    const uint32_t sb_log = scan_block_log(worker_ctas * (uint32_t)kCooWarps, 8u);
    if (blockIdx.x == 0) {
        __shared__ ScanShared scan_sh;
        if (threadIdx.x == 0) {
            scan_sh.seq = 0;
            scan_sh.base = 0;
        }
        __syncthreads();
        scan_service(scan_sh, a.ws.blk_acc, a.ws.status, tag, T, sb_log, a.ws.excl, a.d_nnz, warp, kCooWarps, lane);
        launch_exit(a.ws.hdr, ticket + 1, a.ws.blk_acc, a.ws.status, tag, T, sb_log, gridDim.x * (uint32_t)kCooWarps, lane);
        return;
    }
    const uint32_t cC = ticket_counters(worker_ctas * (uint32_t)kCooWarps);
    const uint32_t cj = ((blockIdx.x - 1u) * (uint32_t)kCooWarps + (uint32_t)warp) % cC;
    uint32_t *const tk = ticket_counter(a.ws.hdr, T, cj);

    uint4 v[32];
    auto load_block = [&](uint32_t tt) {
        const uint32_t *base = a.dense + (size_t)tt * kTile + 4 * lane;
        if (tt < Tfull) {
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = ldg_nc_u4(reinterpret_cast<const uint4 *>(base + 128 * i));
        } else {   // ragged last block: elements >= n are zeros
            const uint64_t e0 = (uint64_t)tt * kTile + 4 * lane;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                const uint64_t e = e0 + 128 * i;
                uint4 x = make_uint4(0u, 0u, 0u, 0u);
                if (e + 3 < n) x = ldg_nc_u4(reinterpret_cast<const uint4 *>(base + 128 * i));
                else {
                    if (e < n) x.x = base[128 * i];
                    if (e + 1 < n) x.y = base[128 * i + 1];
                    if (e + 2 < n) x.z = base[128 * i + 2];
                }
                v[i] = x;
            }
        }
    };
    // rows of the block in registers -> (idx, val) at dst_i / dst_v + running base (shared or global memory);
    // returns the block's count.  bounded: stop storing (keep counting) once the stage is full.
    bool stored_all = true;     // compact(bounded): every entry of the block fitted the stage
    auto compact = [&](uint32_t tt, uint32_t *dst_i, uint32_t *dst_v, bool bounded) -> uint32_t {
        uint32_t base = 0;
        bool on = true;
        const uint32_t e0 = tt * (uint32_t)kTile + 4u * (uint32_t)lane;
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const bool m0 = nz32(v[i].x), m1 = nz32(v[i].y), m2 = nz32(v[i].z), m3 = nz32(v[i].w);
            const unsigned b0 = __ballot_sync(kFull, m0), b1 = __ballot_sync(kFull, m1), b2 = __ballot_sync(kFull, m2),
                           b3 = __ballot_sync(kFull, m3);
            if ((b0 | b1 | b2 | b3) != 0u) {
                if (bounded && base > kCooStage) on = false;     // warp-uniform: the rest of the block only counts
                if (on) {
                    uint32_t pos = base + __popc(b0 & lt) + __popc(b1 & lt) + __popc(b2 & lt) + __popc(b3 & lt);
                    const uint32_t e = e0 + 128u * (uint32_t)i;
                    if (m0) { dst_i[pos] = e; dst_v[pos] = v[i].x; ++pos; }
                    if (m1) { dst_i[pos] = e + 1u; dst_v[pos] = v[i].y; ++pos; }
                    if (m2) { dst_i[pos] = e + 2u; dst_v[pos] = v[i].z; ++pos; }
                    if (m3) { dst_i[pos] = e + 3u; dst_v[pos] = v[i].w; }
                }
                base += __popc(b0) + __popc(b1) + __popc(b2) + __popc(b3);
            }
        }
        stored_all = on;
        return base;
    };

    // two deferred blocks (oldest first) + the block in hand: three stage buffers
    uint32_t q_t[2], q_n[2], q_b[2];
    bool q_on[2] = {false, false};
    uint32_t cur = 0;
    uint32_t held = 0xFFFFFFFFu;   // the block this warp has claimed but not yet published (>= T: none)
    auto flush_one = [&](uint32_t pt, uint32_t pcnt, uint32_t pbuf) {
        const uint32_t excl = service_prefix(a.ws.blk_acc, a.ws.status, a.ws.excl, tag, sb_log, pt, held, T, lane);
        const uint32_t *si = stage + (size_t)pbuf * 2 * kCooStageWords, *sv = si + kCooStageWords;
        for (uint32_t i = lane; i < pcnt; i += 32) {
            a.idx[excl + i] = si[i];
            a.val[excl + i] = sv[i];
        }
        __syncwarp();
    };
    auto flush_all = [&]() {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            if (q_on[i]) flush_one(q_t[i], q_n[i], q_b[i]);
            q_on[i] = false;
        }
    };

    uint32_t t = 0;
    if (lane == 0) t = ticket_tile(tk, cC, cj);
    t = __shfl_sync(kFull, t, 0);
    if (t < T) load_block(t);
    uint32_t t_next = 0;
    if (t < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
    while (t < T) {
        const uint32_t tn = __shfl_sync(kFull, t_next, 0);
        held = tn;
        if (tn < Tfull && lane == 0) {   // the next block starts moving HBM -> L2 now (one bulk prefetch)
            const unsigned char *src = reinterpret_cast<const unsigned char *>(a.dense) + (size_t)tn * kTile * 4;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"((uint32_t)(kTile * 4)) : "memory");
        }
        uint32_t *si = stage + (size_t)cur * 2 * kCooStageWords;
        const uint32_t cnt = compact(t, si, si + kCooStageWords, true);
        __syncwarp();
        if (lane == 0) st_status(a.ws.status + t, tag, cnt);      // for the scan service
        if (q_on[0]) flush_one(q_t[0], q_n[0], q_b[0]);           // the block two iterations back
        q_t[0] = q_t[1]; q_n[0] = q_n[1]; q_b[0] = q_b[1]; q_on[0] = q_on[1];
        if (stored_all) {
            q_t[1] = t; q_n[1] = cnt; q_b[1] = cur; q_on[1] = true;
            cur = cur == (uint32_t)kCooBufs - 1u ? 0u : cur + 1u;
        } else {                                // dense block: its prefix now, write from the registers
            q_on[1] = false;
            const uint32_t excl = service_prefix(a.ws.blk_acc, a.ws.status, a.ws.excl, tag, sb_log, t, held, T, lane);
            compact(t, a.idx + excl, a.val + excl, false);
        }
        if (tn < T) load_block(tn);
        t = tn;
        if (t < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
    }
    held = 0xFFFFFFFFu;
    flush_all();
    launch_exit(a.ws.hdr, ticket + 1, a.ws.blk_acc, a.ws.status, tag, T, sb_log, gridDim.x * (uint32_t)kCooWarps, lane);
}

// ============================================ block offsets (pre-pass) ============================================
// off[t] = number of entries with idx < 4096 t, t = 0 .. T: entry k (and the end sentinel k = nnz) writes the
// offsets of every block boundary that lies between its predecessor and itself.  One streaming pass over idx.
struct CooOffsetsArgs {
    const uint32_t *idx[2];
    const uint32_t *d_nnz[2];
    uint32_t *off[2];
    uint32_t T;
};
__global__ void __launch_bounds__(256) coo_offsets_kernel(const CooOffsetsArgs a) {
    const uint32_t *__restrict__ idx = a.idx[blockIdx.y];
    uint32_t *__restrict__ off = a.off[blockIdx.y];
    const uint32_t nnz = *a.d_nnz[blockIdx.y], T = a.T;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k <= nnz; k += stride) {
        const uint32_t lo = k == 0 ? 0u : (idx[k - 1] >> 12) + 1u;       // first block that starts behind entry k - 1
        const uint32_t hi = k == nnz ? T : (idx[k] >> 12);               // last block that starts at or before entry k
        for (uint32_t t = lo; t <= hi; ++t) off[t] = (uint32_t)k;
    }
}

// =============================================== decompress ===============================================
struct CooExpandArgs {
    const uint32_t *idx, *val, *off;
    uint32_t *dense;
    uint64_t n;
};
__global__ void __launch_bounds__(kCooWarps * 32, 3) coo_decompress_kernel(const CooExpandArgs a) {
    extern __shared__ __align__(16) uint32_t coo_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *const blk = coo_smem + (size_t)warp * kTile;
    const uint32_t T = (uint32_t)((a.n + kTile - 1) / kTile), Tfull = (uint32_t)(a.n / kTile);
    const uint32_t nwarps = gridDim.x * kCooWarps;
    for (uint32_t t = blockIdx.x * kCooWarps + warp; t < T; t += nwarps) {
        const uint32_t k0 = a.off[t], k1 = a.off[t + 1];
        uint4 *b4 = reinterpret_cast<uint4 *>(blk);
        uint4 *d4 = reinterpret_cast<uint4 *>(a.dense + (size_t)t * kTile);
        if (k0 == k1 && t < Tfull) {                 // empty block: a 16 KB zero fill
#pragma unroll 8
            for (int i = 0; i < 32; ++i) stg_stream_u4(d4 + 32 * i + lane, make_uint4(0u, 0u, 0u, 0u));
            continue;
        }
#pragma unroll 8
        for (int i = 0; i < 32; ++i) b4[32 * i + lane] = make_uint4(0u, 0u, 0u, 0u);
        __syncwarp();
        for (uint32_t k = k0 + lane; k < k1; k += 32) blk[a.idx[k] & (kTile - 1)] = a.val[k];
        __syncwarp();
        if (t < Tfull) {
#pragma unroll 8
            for (int i = 0; i < 32; ++i) stg_stream_u4(d4 + 32 * i + lane, b4[32 * i + lane]);
        } else {
            const uint32_t rem = (uint32_t)(a.n - (uint64_t)t * kTile);
            for (uint32_t i = lane; i < rem; i += 32) a.dense[(size_t)t * kTile + i] = blk[i];
        }
        __syncwarp();
    }
}

// ================================================ reduce_sd ================================================
__global__ void __launch_bounds__(256) coo_scatter_add_kernel(const uint32_t *__restrict__ idx, const uint32_t *__restrict__ val,
                                                              const uint32_t *d_nnz, uint32_t *dense) {
    const uint32_t nnz = *d_nnz;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nnz; k += stride) {
        uint32_t *p = dense + idx[k];
        uint32_t d;
        asm volatile("ld.global.L2::64B.u32 %0, [%1];" : "=r"(d) : "l"(p) : "memory");
        *p = __float_as_uint(__fadd_rn(__uint_as_float(d), __uint_as_float(val[k])));
    }
}

// ============================================== reduce_ss (merge) ==============================================
struct CooMergeArgs {
    const uint32_t *ix, *vx, *iy, *vy;
    uint32_t *io, *vo, *d_no;
    uint64_t n;
    CooWs ws;
};
constexpr uint32_t kBmWords = kTile / 32;   // presence bitmap of one operand in one block
constexpr int kMergeWarps = 8;
#ifndef PICI_COO_MERGE_UNROLL
#define PICI_COO_MERGE_UNROLL 4
#endif
static __device__ __forceinline__ uint32_t popc4(uint4 v) { return __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }
constexpr int kU = PICI_COO_MERGE_UNROLL;   // entries per lane whose loads are issued together
#ifndef PICI_COO_MERGE_BLOCKS
#define PICI_COO_MERGE_BLOCKS 4
#endif

// One warp per block.  The entries' indices are scattered into presence bitmaps of X and Y (two 512-byte bitmaps in
// shared memory); with a per-word table of the candidates (x | y) and of the Y entries before each word, every entry
// of a list then knows by itself where its sum goes in the output (the candidate rank of its bit) and where its partner
// in the other list is (entry k of a block is its k-th set bit: the lists ascend).  So all three passes - build the
// bitmaps, test the sums where both lists have an entry (the only place a sum can vanish), emit - read the lists
// COALESCED with kU independent loads per lane in flight.  A block in which a sum did cancel (rare) takes the first
// version's path instead: lane l owns positions 128 l .. 128 l + 127 and walks the set bits of x | y one by one, once
// to count the survivors and once to emit them.  That walk used to be the only path: one dependent global load per
// candidate and lane, twice - 0.88 ms at 90 % sparsity against 0.45 now (95 %: 0.377 -> 0.234, 99 %: 0.133 -> 0.104;
// 99.9 / 99.99 %: 0.078 / 0.072 -> 0.084 / 0.080, the price of the larger kernel where blocks are almost empty).
// The bitmaps and tables stay in one of three slots per warp until the block is emitted two iterations later, with its
// prefix from the scan service (pici_common.cuh), as in pici_compress; the next ticket and the next block's offsets
// are requested one block ahead.  Measured: kU = 2 / 4 / 8 at 90 %: 0.566 / 0.450 / 0.517 ms (8 spills); 3 CTAs per SM:
// 0.481; no prefix wait for blocks without survivors: 0.233 instead of 0.080 ms at 99.99 % (the waits pace the warps).
// An almost empty block costs a ticket, four offsets and a prefix and nothing else: the kernel is latency-bound there.
__global__ void __launch_bounds__(kMergeWarps * 32, PICI_COO_MERGE_BLOCKS) coo_merge_kernel(const CooMergeArgs a) {
    constexpr uint32_t kSlotWords = 3 * kBmWords;           // bitmaps of X and Y, two tables of 128 u16
    __shared__ __align__(16) uint32_t bms[kMergeWarps][3 * kSlotWords];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *const slots = bms[warp];
    uint32_t *const ticket = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(a.ws.hdr) + kWsCompressTicket);
    const uint32_t tag = launch_tag(a.ws.hdr);
    const uint32_t T = (uint32_t)((a.n + kTile - 1) / kTile);
    const uint32_t *__restrict__ ix = a.ix, *__restrict__ iy = a.iy, *__restrict__ vx = a.vx, *__restrict__ vy = a.vy;
    // the device-wide scan of the survivor counts is a service (CTA 0; pici_common.cuh), as in the compress kernels
    const uint32_t worker_ctas = gridDim.x - 1u;
    const uint32_t sb_log = scan_block_log(worker_ctas * (uint32_t)kMergeWarps, 9u);
    if (blockIdx.x == 0) {
        __shared__ ScanShared scan_sh;
        if (threadIdx.x == 0) {
            scan_sh.seq = 0;
            scan_sh.base = 0;
        }
        __syncthreads();
        scan_service(scan_sh, a.ws.blk_acc, a.ws.status, tag, T, sb_log, a.ws.excl, a.d_no, warp, kMergeWarps, lane);
        launch_exit(a.ws.hdr, ticket + 1, a.ws.blk_acc, a.ws.status, tag, T, sb_log, gridDim.x * (uint32_t)kMergeWarps, lane);
        return;
    }
    const uint32_t cC = ticket_counters(worker_ctas * (uint32_t)kMergeWarps);
    const uint32_t cj = ((blockIdx.x - 1u) * (uint32_t)kMergeWarps + (uint32_t)warp) % cC;
    uint32_t *const tk = ticket_counter(a.ws.hdr, T, cj);

    // lane 0 .. 3 hold offx[t], offx[t + 1], offy[t], offy[t + 1] of the block in hand / the next block
    auto load_off = [&](uint32_t tt) -> uint32_t {
        uint32_t v = 0;
        if (tt < T && lane < 4) v = (lane < 2 ? a.ws.offx : a.ws.offy)[tt + (lane & 1)];
        return v;
    };
    // A block's tables live in one of the warp's three shared-memory slots from its count to its emission two
    // iterations later (behind the prefix): the presence bitmaps of X and Y (128 words each) and, per word, the
    // number of candidates (x | y) and of Y entries of the block before it (u16).  Entry k of a list is its k-th set
    // bit (the lists ascend), so with these an entry finds its place in the output, and its partner in the other
    // list, by itself: all passes read the lists coalesced, kU loads per lane in flight.
    struct Blk {          // warp-uniform
        uint32_t x0, y0, nx, ny, t, total, slot;
        bool fast;        // no candidate of the block cancelled: survivor k IS candidate k
    };
    auto bmx_of = [&](uint32_t slot) -> uint32_t * { return slots + slot * kSlotWords; };
    // the sequential walk over the lane's candidates (only for a block in which a sum cancelled): emit = false counts
    // the lane's survivors, true stores them from `o` on
    auto walk = [&](const Blk &B, bool emit, uint32_t o) -> uint32_t {
        const uint32_t *bx = bmx_of(B.slot), *by = bx + kBmWords;
        const uint4 X = reinterpret_cast<const uint4 *>(bx)[lane], Y = reinterpret_cast<const uint4 *>(by)[lane];
        const uint32_t wx[4] = {X.x, X.y, X.z, X.w}, wy[4] = {Y.x, Y.y, Y.z, Y.w};
        const uint32_t v = popc4(X) | (popc4(Y) << 16);       // <= 4096 each
        const uint32_t sc = warp_incl_scan(v, lane) - v;
        uint32_t px = B.x0 + (sc & 0xFFFFu), py = B.y0 + (sc >> 16), cnt = 0;
        const uint32_t e0 = B.t * (uint32_t)kTile + 128u * (uint32_t)lane;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t u = wx[q] | wy[q];
            while (u) {
                const uint32_t bit = u & (0u - u);
                u ^= bit;
                const bool hx = (wx[q] & bit) != 0u, hy = (wy[q] & bit) != 0u;
                const float x = hx ? __uint_as_float(vx[px]) : 0.0f;
                const float y = hy ? __uint_as_float(vy[py]) : 0.0f;
                px += hx ? 1u : 0u;
                py += hy ? 1u : 0u;
                const uint32_t sum = __float_as_uint(__fadd_rn(x, y));      // received + local, an absent operand is +0
                if (nz32(sum)) {
                    if (emit) {
                        a.io[o + cnt] = e0 + 32u * q + (uint32_t)__ffs(bit) - 1u;
                        a.vo[o + cnt] = sum;
                    }
                    ++cnt;
                }
            }
        }
        return cnt;
    };
    Blk P0, P1;                                              // blocks whose emission is deferred, oldest first
    bool on0 = false, on1 = false;
    uint32_t held = 0xFFFFFFFFu;                              // claimed, not yet published (>= T: none)
    auto emit = [&](const Blk &P) {
        const uint32_t excl = service_prefix(a.ws.blk_acc, a.ws.status, a.ws.excl, tag, sb_log, P.t, held, T, lane);
        if (P.total == 0u) return;
        if (!P.fast) {
            const uint32_t cnt = walk(P, false, 0u);
            walk(P, true, excl + warp_incl_scan(cnt, lane) - cnt);
            return;
        }
        const uint32_t *bmx = bmx_of(P.slot), *bmy = bmx + kBmWords;
        const uint16_t *up16 = reinterpret_cast<const uint16_t *>(bmy + kBmWords), *yp16 = up16 + kBmWords;
        const uint32_t nx = P.nx, ny = P.ny;
        for (uint32_t k0 = lane; k0 < nx; k0 += 32 * kU) {    // the X entries, with their Y partner where there is one
            uint32_t pos[kU], xv[kU], r[kU], yi[kU];
            bool hy[kU];
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                const uint32_t k = k0 + 32 * j;
                pos[j] = k < nx ? ix[P.x0 + k] : 0u;
                xv[j] = k < nx ? vx[P.x0 + k] : 0u;
            }
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                const uint32_t w = (pos[j] & (kTile - 1)) >> 5, below = (1u << (pos[j] & 31)) - 1u;
                const uint32_t by = bmy[w];
                r[j] = up16[w] + __popc((bmx[w] | by) & below);
                hy[j] = ((by >> (pos[j] & 31)) & 1u) != 0u && k0 + 32 * j < nx;
                yi[j] = P.y0 + yp16[w] + __popc(by & below);
            }
            uint32_t yv[kU];
#pragma unroll
            for (int j = 0; j < kU; ++j) yv[j] = hy[j] ? vy[yi[j]] : 0u;
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                if (k0 + 32 * j < nx) {
                    a.io[excl + r[j]] = pos[j];
                    a.vo[excl + r[j]] = __float_as_uint(__fadd_rn(__uint_as_float(xv[j]), __uint_as_float(yv[j])));
                }
            }
        }
        for (uint32_t k0 = lane; k0 < ny; k0 += 32 * kU) {    // the Y entries without a partner
            uint32_t pos[kU], yv[kU];
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                const uint32_t k = k0 + 32 * j;
                pos[j] = k < ny ? iy[P.y0 + k] : 0u;
                yv[j] = k < ny ? vy[P.y0 + k] : 0u;
            }
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                const uint32_t w = (pos[j] & (kTile - 1)) >> 5, below = (1u << (pos[j] & 31)) - 1u;
                const uint32_t bx = bmx[w];
                if (k0 + 32 * j < ny && ((bx >> (pos[j] & 31)) & 1u) == 0u) {
                    const uint32_t r = up16[w] + __popc((bx | bmy[w]) & below);
                    a.io[excl + r] = pos[j];
                    a.vo[excl + r] = __float_as_uint(__fadd_rn(0.0f, __uint_as_float(yv[j])));
                }
            }
        }
    };

    uint32_t t = 0;
    if (lane == 0) t = ticket_tile(tk, cC, cj);
    t = __shfl_sync(kFull, t, 0);
    uint32_t off = load_off(t);
    uint32_t t_next = 0;
    if (t < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
    uint32_t seq = 0;                                         // blocks with entries so far: slot = seq mod 3
    while (t < T) {
        const uint32_t x0 = __shfl_sync(kFull, off, 0), x1 = __shfl_sync(kFull, off, 1), y0 = __shfl_sync(kFull, off, 2),
                       y1 = __shfl_sync(kFull, off, 3);
        const uint32_t tn = __shfl_sync(kFull, t_next, 0);
        held = tn;
        off = load_off(tn);                                   // arrives while this block is merged
        if (tn < T && lane == 0) t_next = ticket_tile(tk, cC, cj);
        Blk C;
        C.x0 = x0; C.y0 = y0; C.nx = x1 - x0; C.ny = y1 - y0; C.t = t; C.fast = true; C.total = 0; C.slot = seq % 3u;
        if (C.nx != 0u || C.ny != 0u) {
            // the slot's previous block (three blocks with entries back) was emitted at least one iteration ago
            ++seq;
            uint32_t *bmx = bmx_of(C.slot), *bmy = bmx + kBmWords;
            __syncwarp();
            reinterpret_cast<uint4 *>(bmx)[lane] = make_uint4(0u, 0u, 0u, 0u);
            reinterpret_cast<uint4 *>(bmy)[lane] = make_uint4(0u, 0u, 0u, 0u);
            __syncwarp();
            const uint32_t nx = C.nx, ny = C.ny;
            for (uint32_t k0 = lane; k0 < max(nx, ny); k0 += 32 * kU) {
                uint32_t px[kU], py[kU];
#pragma unroll
                for (int j = 0; j < kU; ++j) {
                    const uint32_t k = k0 + 32 * j;
                    px[j] = k < nx ? ix[x0 + k] : 0u;
                    py[j] = k < ny ? iy[y0 + k] : 0u;
                }
#pragma unroll
                for (int j = 0; j < kU; ++j) {
                    const uint32_t k = k0 + 32 * j;
                    if (k < nx) atomicOr(&bmx[(px[j] & (kTile - 1)) >> 5], 1u << (px[j] & 31));
                    if (k < ny) atomicOr(&bmy[(py[j] & (kTile - 1)) >> 5], 1u << (py[j] & 31));
                }
            }
            __syncwarp();
            const uint4 X = reinterpret_cast<const uint4 *>(bmx)[lane], Y = reinterpret_cast<const uint4 *>(bmy)[lane];
            // the tables: candidates / Y entries of the block before each of the lane's four words
            {
                const uint32_t cu = __popc(X.x | Y.x) + __popc(X.y | Y.y) + __popc(X.z | Y.z) + __popc(X.w | Y.w);
                const uint32_t v = cu | (popc4(Y) << 16);
                const uint32_t incl = warp_incl_scan(v, lane);
                C.total = __shfl_sync(kFull, incl, 31) & 0xFFFFu;
                const uint32_t e = incl - v;
                const uint32_t u0 = e & 0xFFFFu, u1 = u0 + __popc(X.x | Y.x), u2 = u1 + __popc(X.y | Y.y), u3 = u2 + __popc(X.z | Y.z);
                const uint32_t q0 = e >> 16, q1 = q0 + __popc(Y.x), q2 = q1 + __popc(Y.y), q3 = q2 + __popc(Y.z);
                reinterpret_cast<uint2 *>(bmy + kBmWords)[lane] = make_uint2(u0 | (u1 << 16), u2 | (u3 << 16));
                reinterpret_cast<uint2 *>(bmy + kBmWords + kBmWords / 2)[lane] = make_uint2(q0 | (q1 << 16), q2 | (q3 << 16));
            }
            __syncwarp();
            // a sum can only vanish where both lists have an entry: test those (the predicate re-applied to x + y)
            if (__any_sync(kFull, ((X.x & Y.x) | (X.y & Y.y) | (X.z & Y.z) | (X.w & Y.w)) != 0u)) {
                const uint16_t *yp16 = reinterpret_cast<const uint16_t *>(bmy + kBmWords) + kBmWords;
                bool cancelled = false;
                for (uint32_t k0 = lane; k0 < nx; k0 += 32 * kU) {
                    uint32_t pos[kU], xv[kU], yv[kU];
                    bool hy[kU];
#pragma unroll
                    for (int j = 0; j < kU; ++j) pos[j] = k0 + 32 * j < nx ? ix[x0 + k0 + 32 * j] : 0u;
#pragma unroll
                    for (int j = 0; j < kU; ++j) {
                        const uint32_t w = (pos[j] & (kTile - 1)) >> 5, by = bmy[w];
                        hy[j] = k0 + 32 * j < nx && ((by >> (pos[j] & 31)) & 1u) != 0u;
                        xv[j] = yv[j] = 0x3F800000u;         // 1 + 1: no cancellation
                        if (hy[j]) {
                            xv[j] = vx[x0 + k0 + 32 * j];
                            yv[j] = vy[y0 + yp16[w] + __popc(by & ((1u << (pos[j] & 31)) - 1u))];
                        }
                    }
#pragma unroll
                    for (int j = 0; j < kU; ++j)
                        cancelled |= hy[j] && !nz32(__float_as_uint(__fadd_rn(__uint_as_float(xv[j]), __uint_as_float(yv[j]))));
                }
                if (__any_sync(kFull, cancelled)) {           // rare: count (and later emit) lane by lane
                    C.fast = false;
                    C.total = warp_sum(walk(C, false, 0u));
                }
            }
        }
        if (lane == 0) st_status(a.ws.status + t, tag, C.total);   // for the scan service
        if (on0) emit(P0);                                    // the block two iterations back
        P0 = P1; on0 = on1;
        P1 = C; on1 = true;
        t = tn;
    }
    held = 0xFFFFFFFFu;
    if (on0) emit(P0);
    if (on1) emit(P1);
    launch_exit(a.ws.hdr, ticket + 1, a.ws.blk_acc, a.ws.status, tag, T, sb_log, gridDim.x * (uint32_t)kMergeWarps, lane);
}

// ================================================= launchers =================================================
template <class K>
static cudaError_t allow_smem(K kernel, size_t smem, std::atomic<bool> (&done)[64]) {   // one-time per device
    std::atomic<bool> &flag = done[current_device_slot()];
    if (!flag.load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        flag.store(true, std::memory_order_release);
    }
    return cudaSuccess;
}
static unsigned persistent_grid(uint64_t T, uint64_t waves = 1) {   // waves > 1: the block scheduler balances the SMs
    uint64_t blocks = (T + kCooWarps - 1) / kCooWarps;
    const uint64_t cap = (uint64_t)num_sms() * 3 * waves;
    return (unsigned)(blocks > cap ? cap : (blocks ? blocks : 1));
}

static cudaError_t launch_coo_compress(const void *dense, uint64_t n, uint32_t *idx, void *val, uint32_t *d_nnz, void *ws,
                                       uint64_t ws_bytes, cudaStream_t s) {
    if (n == 0) return launch_set_u32(d_nnz, 0u, Gate{nullptr, 0, 0}, s);
    static std::atomic<bool> done[64];
    const size_t smem = (size_t)kCooWarps * kCooBufs * 2 * kCooStageWords * sizeof(uint32_t);
    cudaError_t e = allow_smem(coo_compress_kernel, smem, done);
    if (e != cudaSuccess) return e;
    const CooCompressArgs a = {reinterpret_cast<const uint32_t *>(dense), n, idx, reinterpret_cast<uint32_t *>(val), d_nnz,
                               coo_ws(ws, ws_bytes, n)};
    // + CTA 0, the scan service; all CTAs resident (one wave)
    const uint64_t T = (n + kTile - 1) / kTile;
    uint64_t blocks = (T + kCooWarps - 1) / kCooWarps + 1;
    if (blocks > (uint64_t)num_sms() * 3) blocks = (uint64_t)num_sms() * 3;
    coo_compress_kernel<<<(unsigned)blocks, kCooWarps * 32, smem, s>>>(a);
    return cudaGetLastError();
}

static cudaError_t launch_coo_offsets(const uint32_t *ix, const uint32_t *d_nx, uint32_t *offx, const uint32_t *iy,
                                      const uint32_t *d_ny, uint32_t *offy, uint64_t n, cudaStream_t s) {
    CooOffsetsArgs a;
    a.idx[0] = ix; a.d_nnz[0] = d_nx; a.off[0] = offx;
    a.idx[1] = iy; a.d_nnz[1] = d_ny; a.off[1] = offy;
    a.T = (uint32_t)((n + kTile - 1) / kTile);
    coo_offsets_kernel<<<dim3((unsigned)num_sms() * 8, iy ? 2 : 1), 256, 0, s>>>(a);
    return cudaGetLastError();
}

static cudaError_t launch_coo_decompress(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n, void *dense,
                                         void *ws, uint64_t ws_bytes, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    static std::atomic<bool> done[64];
    const size_t smem = (size_t)kCooWarps * kTile * sizeof(uint32_t);
    cudaError_t e = allow_smem(coo_decompress_kernel, smem, done);
    if (e != cudaSuccess) return e;
    const CooWs w = coo_ws(ws, ws_bytes, n);
    e = launch_coo_offsets(idx, d_nnz, w.offx, nullptr, nullptr, nullptr, n, s);
    if (e != cudaSuccess) return e;
    const CooExpandArgs a = {idx, reinterpret_cast<const uint32_t *>(val), w.offx, reinterpret_cast<uint32_t *>(dense), n};
    coo_decompress_kernel<<<persistent_grid((n + kTile - 1) / kTile, 12), kCooWarps * 32, smem, s>>>(a);   // write-bound: see expand.cu
    return cudaGetLastError();
}

static cudaError_t launch_coo_reduce_sd(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n, void *dense,
                                        cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    coo_scatter_add_kernel<<<(unsigned)num_sms() * 8, 256, 0, s>>>(idx, reinterpret_cast<const uint32_t *>(val), d_nnz,
                                                                   reinterpret_cast<uint32_t *>(dense));
    return cudaGetLastError();
}

static cudaError_t launch_coo_merge(const uint32_t *ix, const void *vx, const uint32_t *d_nx, const uint32_t *iy, const void *vy,
                                    const uint32_t *d_ny, uint64_t n, uint32_t *io, void *vo, uint32_t *d_no, void *ws,
                                    uint64_t ws_bytes, cudaStream_t s) {
    if (n == 0) return launch_set_u32(d_no, 0u, Gate{nullptr, 0, 0}, s);
    const CooWs w = coo_ws(ws, ws_bytes, n);
    cudaError_t e = launch_coo_offsets(ix, d_nx, w.offx, iy, d_ny, w.offy, n, s);
    if (e != cudaSuccess) return e;
    const CooMergeArgs a = {ix, reinterpret_cast<const uint32_t *>(vx), iy, reinterpret_cast<const uint32_t *>(vy), io,
                            reinterpret_cast<uint32_t *>(vo), d_no, n, w};
    const uint64_t T = (n + kTile - 1) / kTile;
    uint64_t blocks = (T + kMergeWarps - 1) / kMergeWarps + 1;   // + CTA 0, the scan service
    const uint64_t cap = (uint64_t)num_sms() * PICI_COO_MERGE_BLOCKS;
    if (blocks > cap) blocks = cap;
    coo_merge_kernel<<<(unsigned)blocks, kMergeWarps * 32, 0, s>>>(a);
    return cudaGetLastError();
}

}  // namespace pici

// =================================================== C ABI ===================================================
using namespace pici;
namespace {
inline bool al(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }
inline int rc_of(cudaError_t e) { return e == cudaSuccess ? PICI_OK : PICI_ERR_CUDA; }
constexpr uint64_t kCooMaxN = 1ull << 32;
int check_coo(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n) {
    if (n >= kCooMaxN || d_nnz == nullptr) return PICI_ERR_INVALID_ARG;
    if (n != 0 && (idx == nullptr || val == nullptr)) return PICI_ERR_INVALID_ARG;
    if (!al(idx, 16) || !al(val, 16) || !al(d_nnz, 4)) return PICI_ERR_ALIGN;
    return PICI_OK;
}
int check_ws(void *ws, uint64_t ws_bytes, uint64_t n) {
    if (!al(ws, 16)) return PICI_ERR_ALIGN;
    if (n != 0 && (ws == nullptr || ws_bytes < coo_workspace_bytes(n))) return PICI_ERR_WORKSPACE;
    return PICI_OK;
}
}  // namespace

extern "C" {

int pici_coo_sizes(uint64_t n, uint64_t *capacity, uint64_t *workspace_bytes) {
    if (n >= kCooMaxN) return PICI_ERR_INVALID_ARG;
    if (capacity) *capacity = n;
    if (workspace_bytes) *workspace_bytes = coo_workspace_bytes(n);
    return PICI_OK;
}

int pici_coo_compress(const void *dense, uint64_t n, uint32_t *idx, void *val, uint64_t capacity, uint32_t *d_nnz,
                      void *ws, uint64_t ws_bytes, void *stream) {
    int rc = check_coo(idx, val, d_nnz, n);
    if (rc != PICI_OK) return rc;
    if (n != 0 && dense == nullptr) return PICI_ERR_INVALID_ARG;
    if (!al(dense, 16)) return PICI_ERR_ALIGN;
    if (capacity < n) return PICI_ERR_CAPACITY;
    if ((rc = check_ws(ws, ws_bytes, n)) != PICI_OK) return rc;
    return rc_of(launch_coo_compress(dense, n, idx, val, d_nnz, ws, ws_bytes, static_cast<cudaStream_t>(stream)));
}

int pici_coo_decompress(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n, void *dense_out,
                        void *ws, uint64_t ws_bytes, void *stream) {
    int rc = check_coo(idx, val, d_nnz, n);
    if (rc != PICI_OK) return rc;
    if (n != 0 && dense_out == nullptr) return PICI_ERR_INVALID_ARG;
    if (!al(dense_out, 16)) return PICI_ERR_ALIGN;
    if ((rc = check_ws(ws, ws_bytes, n)) != PICI_OK) return rc;
    return rc_of(launch_coo_decompress(idx, val, d_nnz, n, dense_out, ws, ws_bytes, static_cast<cudaStream_t>(stream)));
}

int pici_coo_reduce_sd(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n, void *dense_inout,
                       void *stream) {
    int rc = check_coo(idx, val, d_nnz, n);
    if (rc != PICI_OK) return rc;
    if (n != 0 && dense_inout == nullptr) return PICI_ERR_INVALID_ARG;
    if (!al(dense_inout, 16)) return PICI_ERR_ALIGN;
    return rc_of(launch_coo_reduce_sd(idx, val, d_nnz, n, dense_inout, static_cast<cudaStream_t>(stream)));
}

int pici_coo_reduce_ss(const uint32_t *ix, const void *vx, const uint32_t *d_nx, const uint32_t *iy, const void *vy,
                       const uint32_t *d_ny, uint64_t n, uint32_t *io, void *vo, uint64_t capacity, uint32_t *d_no,
                       void *ws, uint64_t ws_bytes, void *stream) {
    int rc = check_coo(ix, vx, d_nx, n);
    if (rc == PICI_OK) rc = check_coo(iy, vy, d_ny, n);
    if (rc == PICI_OK) rc = check_coo(io, vo, d_no, n);
    if (rc != PICI_OK) return rc;
    if (capacity < n) return PICI_ERR_CAPACITY;
    if ((rc = check_ws(ws, ws_bytes, n)) != PICI_OK) return rc;
    if (n != 0 && (io == ix || io == iy || vo == vx || vo == vy || d_no == d_nx || d_no == d_ny)) return PICI_ERR_INVALID_ARG;
    return rc_of(launch_coo_merge(ix, vx, d_nx, iy, vy, d_ny, n, io, vo, d_no, ws, ws_bytes, static_cast<cudaStream_t>(stream)));
}

}  // extern "C"
