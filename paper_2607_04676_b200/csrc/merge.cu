// merge.cu - pici_reduce_ss: O = compress(decompress(X) + decompress(Y)) without the dense buffer.
//
// This is the fused form of the paper's reduce-scatter step "accumulate into a dense buffer using
// our Pici scatter-add kernel ... this accumulated dense buffer must be recompressed";
// the sparse+sparse merge itself is not in the paper.  Semantics (S8(c) C5):
// o_i = x_i + y_i wherever X or Y has its bit set (an absent operand reads as +0.0, one fp32 add in
// the order "received + local" = x + y), the nonzero predicate is RE-APPLIED to the sum, so an exact
// cancellation is dropped from the output mask.
//
// Because A is ordered tile -> column -> row and B[64t+c] is column c with bit r = row r, the words of
// B read as ONE little-endian bit string ARE the order of A.  The merge therefore never needs a dense
// position: it is a 1-D merge of two (bit string, value stream) pairs, and I[t] is the number of
// survivors before bit 4096*t.  The kernel works on SPANS of that string:
//   * a span is m = 16, 8, 4, 2 or 1 consecutive tiles, the same m for the whole launch: the largest
//     whose AVERAGE contents fit one shared-memory stage and whose expected union of the two supports fits
//     the output region (read on the device from Ix[T], Iy[T]), halved while the launch has fewer than
//     two spans per CTA;
//   * the launch is COOPERATIVE with G CTAs (two per SM, all co-resident); CTA c takes spans c, c + G,
//     c + 2G, ...  A CTA is 16 WALKER warps plus one SERVICE warp per stage (576 threads).  The service
//     warp of stage s starts the four 1-D TMA bulk copies of a span - its Bx / By words (contiguous) and
//     its X / Y value runs (contiguous in Ax / Ay), one mbarrier - two spans ahead, index entries loaded
//     one span before that, so the walkers find the stage filled when they get to it;
//   * walkers: thread j owns the 8m-bit piece j of the span; x's and y's cursors come from the
//     block-wide popc prefix of their own pieces, the candidate cursor from the popc prefix of the OR;
//     every thread walks the set bits of its piece, adds, tests the predicate and packs its surviving
//     sums into its own run of the stage's output region (runs start at the OR-prefix, so they never
//     overlap); they publish the span's count and go on - they never wait for a look-back;
//   * Phase 2 (exclusive scan of the counts) is the round-robin scan of pici_common.cuh:
//     per-span / per-32-spans / per-iteration words, prefix = three independent loads (a flat decoupled
//     look-back walks up to G/32 dependent hops here because the CTAs run in lock-step; a block-wide flat
//     read hot-spots a few L2 lines - both measured).  The service warp takes the prefix once the count
//     is out, writes the span's index entries and copies the output region to Ao (packed; if a
//     cancellation left gaps, run by run from what the walkers recorded), then releases the region;
//   * a span whose values do not fit the stage, or whose exact candidate count exceeds the output region
//     (the span length is chosen from an estimate), is processed tile by tile in two sweeps (count, then
//     emit) by the walkers themselves - one tile always fits.
// The kernel is bound by the issue of its per-span bookkeeping, not by HBM (S5).
#include <type_traits>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

#ifdef PICI_MERGE_TRACE   // debug only: per-CTA, per-iteration %globaltimer stamps
__device__ uint64_t *g_merge_trace;
#define PICI_TR(it, k)                                                                      \
    do {                                                                                    \
        if (threadIdx.x == 0 && (it) < 16u) {                                               \
            uint64_t t_;                                                                    \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                          \
            g_merge_trace[((size_t)blockIdx.x * 16 + (it)) * 8 + (k)] = t_;                 \
        }                                                                                   \
    } while (0)
#else
#define PICI_TR(it, k) do { } while (0)
#endif

constexpr int kMergeWarps = 16;
constexpr int kMergeThreads = kMergeWarps * 32;
constexpr int kMaxSpan = 16;                            // tiles per span: 16, 8, 4, 2 or 1
constexpr uint32_t kTileWords = 2 * kSide;              // u32 words of B per tile
// stage = [Bx words of the span][By words][X window][Y window]; one full tile always fits
constexpr uint32_t kStageWords = 2 * kTileWords + 2 * kTile + 16;
constexpr uint32_t kOutWords = kTile;                   // candidates (bits of x | y) of a span
constexpr uint32_t kPoolWords = 2 * kStageWords + 2 * kOutWords;   // two stages, two output regions
constexpr int kMergeMinBlocks = 2;
constexpr uint32_t kMaxGrid = kRoundRobinMaxUnits;       // units per iteration the round-robin scan supports

// What the staging warp tells the walkers about the span in a stage.
struct SpanInfo {
    uint32_t fits;      // 0: the span takes the slow path (nothing was copied)
    uint32_t Xb, Yb;    // stage word of the first x / y value
    uint32_t xs, ys;    // Ix[ts], Iy[ts]
};
struct MergeShared {
    uint64_t full[2];         // mbarrier: the copies of the span in stage s have landed
    uint64_t stage_free[2];   // mbarrier: the walkers are done with stage s
    uint64_t counts[2];       // mbarrier: out region s, tcs[s], tot[s] are written, the count is published
    uint64_t lb_done[2];      // mbarrier: excl[s] is written
    uint64_t flushed[2];      // mbarrier: out region s has been written to Ao
    uint64_t slow_bar;        // mbarrier: copies of the slow path
    SpanInfo info[2];
    uint32_t excl[2];                 // survivors before the span (from the look-back)
    uint32_t tot[2], cand[2];         // survivors / candidates of the span; cand == ~0u: the walkers flush it
    uint32_t tcs[2][kMaxSpan];        // per-tile survivors of the span
    uint32_t wxy[kMergeWarps];        // per-warp totals: popc(x piece) | popc(y piece) << 16
    uint32_t wu[kMergeWarps];         // per-warp totals: popc(x | y)
    uint32_t ws[kMergeWarps];         // per-warp totals: survivors
    uint16_t run_at[2][kMergeThreads];   // per-thread runs of a span that had cancellations: first word,
    uint16_t run_k[2][kMergeThreads];    // survivors
};
// Barrier of the 16 walker warps (the staging warp never joins it).
__device__ __forceinline__ void walkers_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kMergeThreads) : "memory"); }
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

struct MergeArgs {
    const uint64_t *Bx, *By;
    const uint32_t *Ix, *Iy, *Ax, *Ay;
    uint64_t *Bo;
    uint32_t *Io, *Ao;
    RoundRobinScan scan;   // per-span / per-group / per-iteration words (pici_common.cuh)
    uint32_t T;
    uint64_t a_limit;      // bytes of Ax / Ay that may be read: (n * 4) & ~15 (capacity >= n elements)
};

// ---- staging ------------------------------------------------------------------------------------
// The values A[beg .. beg+cnt) are copied as ONE bulk copy of the 16-byte aligned window around them
// (up to 12 bytes before and after belong to neighbouring spans of the same buffer; the window never
// passes a_limit, so nothing outside the caller's capacity is read).  Only a run that ends in the last
// < 16 bytes of a completely full buffer keeps a tail, moved by plain loads.
struct Window {
    uint64_t g_beg;    // byte offset in A of the window start
    uint32_t bulk;     // bytes of the bulk copy (multiple of 16, may be 0)
    uint32_t words;    // window length in words, multiple of 4 (what the stage reserves)
    uint32_t first;    // word index inside the window of element 0
    uint32_t tail_beg; // element index (relative to beg) where the plain-load tail starts; == cnt if none
};
__device__ __forceinline__ Window window_of(uint32_t beg, uint32_t cnt, uint64_t a_limit) {
    Window w;
    const uint64_t a_beg = (uint64_t)beg * 4, a_end = a_beg + (uint64_t)cnt * 4;
    w.g_beg = a_beg & ~15ull;
    const uint64_t end_up = (a_end + 15ull) & ~15ull;
    const uint64_t end_bulk = cnt == 0 ? w.g_beg : (end_up <= a_limit ? end_up : (a_end & ~15ull));
    w.bulk = end_bulk > w.g_beg ? (uint32_t)(end_bulk - w.g_beg) : 0u;
    w.words = (uint32_t)((end_up - w.g_beg) / 4);
    w.first = (uint32_t)(a_beg - w.g_beg) / 4;
    const uint64_t covered = w.g_beg + w.bulk;   // bytes below this are in the bulk copy
    w.tail_beg = covered >= a_end ? cnt : (covered > a_beg ? (uint32_t)((covered - a_beg) / 4) : 0u);
    return w;
}

// Layout of a span inside a stage (m tiles per span).
struct SpanLayout {
    uint32_t By0;      // word of the span's By words (Bx words start at 0)
    uint32_t Xb, Yb;   // word of the first x / y value
    uint32_t tx;       // bytes the bulk copies signal on the mbarrier
};
__device__ __forceinline__ bool span_fits(uint32_t m, uint32_t nx, uint32_t ny, uint32_t mt) {
    (void)mt;   // the output region is checked on the exact candidate count, after the popc scan (walk_span)
    return 2u * m * kTileWords + nx + ny + 16u <= kStageWords;
}

// Warp 0: start the copies of the span of mt tiles at tile ts (m tiles per span) into `stage`; returns
// its layout.  Other callers pass issue = false to get the layout only.
__device__ __forceinline__ SpanLayout span_stage(const MergeArgs &a, uint32_t *stage, uint32_t bar, uint32_t ts, uint32_t m,
                                                 uint32_t mt, uint32_t xs, uint32_t nx, uint32_t ys, uint32_t ny,
                                                 bool issue, int lane) {
    const Window wx = window_of(xs, nx, a.a_limit), wy = window_of(ys, ny, a.a_limit);
    SpanLayout L;
    L.By0 = m * kTileWords;
    const uint32_t V = 2u * m * kTileWords;
    L.Xb = V + wx.first;
    L.Yb = V + wx.words + wy.first;
    const uint32_t bbytes = mt * kTileWords * 4u;
    L.tx = 2u * bbytes + wx.bulk + wy.bulk;
    if (issue) {
        // tail elements first (plain stores, < 4 per operand), so that lane 0's arrive on the mbarrier - the
        // release the walkers' wait acquires - is ordered behind every lane's stores
        if (wx.tail_beg + lane < nx) stage[L.Xb + wx.tail_beg + lane] = a.Ax[xs + wx.tail_beg + lane];
        if (wy.tail_beg + lane < ny) stage[L.Yb + wy.tail_beg + lane] = a.Ay[ys + wy.tail_beg + lane];
        __syncwarp();
        if (lane == 0) {
            fence_proxy_async_smem();
            mbar_expect_tx(bar, L.tx);
            bulk_g2s(smem_u32(stage), a.Bx + (size_t)ts * kSide, bbytes, bar);
            bulk_g2s(smem_u32(stage + L.By0), a.By + (size_t)ts * kSide, bbytes, bar);
            if (wx.bulk) bulk_g2s(smem_u32(stage + V), reinterpret_cast<const unsigned char *>(a.Ax) + wx.g_beg, wx.bulk, bar);
            if (wy.bulk)
                bulk_g2s(smem_u32(stage + V + wx.words), reinterpret_cast<const unsigned char *>(a.Ay) + wy.g_beg, wy.bulk, bar);
        }
    }
    return L;
}

// This thread's 8*m-bit piece of the staged Bx / By words.  Pieces past the span's last tile are 0.
__device__ __forceinline__ void read_piece(const uint32_t *stage, uint32_t By0, uint32_t m, uint32_t mt, int tid,
                                           uint32_t (&ax)[4], uint32_t (&ay)[4]) {
    ax[0] = ax[1] = ax[2] = ax[3] = 0u;
    ay[0] = ay[1] = ay[2] = ay[3] = 0u;
    if ((uint32_t)tid * m >= (uint32_t)kMergeThreads * mt) return;
    const uint32_t *bx = stage, *by = stage + By0;
    if (m == 16) {
        const uint4 p = reinterpret_cast<const uint4 *>(bx)[tid], q = reinterpret_cast<const uint4 *>(by)[tid];
        ax[0] = p.x; ax[1] = p.y; ax[2] = p.z; ax[3] = p.w;
        ay[0] = q.x; ay[1] = q.y; ay[2] = q.z; ay[3] = q.w;
    } else if (m == 8) {
        const uint2 p = reinterpret_cast<const uint2 *>(bx)[tid], q = reinterpret_cast<const uint2 *>(by)[tid];
        ax[0] = p.x; ax[1] = p.y;
        ay[0] = q.x; ay[1] = q.y;
    } else if (m == 4) {
        ax[0] = bx[tid];
        ay[0] = by[tid];
    } else if (m == 2) {
        ax[0] = reinterpret_cast<const uint16_t *>(bx)[tid];
        ay[0] = reinterpret_cast<const uint16_t *>(by)[tid];
    } else {
        ax[0] = reinterpret_cast<const uint8_t *>(bx)[tid];
        ay[0] = reinterpret_cast<const uint8_t *>(by)[tid];
    }
}
__device__ __forceinline__ void store_piece(const MergeArgs &a, uint32_t ts, uint32_t m, uint32_t mt, int tid,
                                            const uint32_t (&ao)[4]) {
    if ((uint32_t)tid * m >= (uint32_t)kMergeThreads * mt) return;
    const size_t wbase = (size_t)ts * kSide;
    if (m == 16) reinterpret_cast<uint4 *>(a.Bo + wbase)[tid] = make_uint4(ao[0], ao[1], ao[2], ao[3]);
    else if (m == 8) reinterpret_cast<uint2 *>(a.Bo + wbase)[tid] = make_uint2(ao[0], ao[1]);
    else if (m == 4) reinterpret_cast<uint32_t *>(a.Bo + wbase)[tid] = ao[0];
    else if (m == 2) reinterpret_cast<uint16_t *>(a.Bo + wbase)[tid] = (uint16_t)ao[0];
    else reinterpret_cast<uint8_t *>(a.Bo + wbase)[tid] = (uint8_t)ao[0];
}

// What a thread keeps from one walk of a span.
struct WalkOut {
    uint32_t k;            // this thread's survivors
    uint32_t ko0;          // word of this thread's run in the output region
    uint32_t sk;           // inclusive warp scan of k
    uint32_t cand_total;   // candidates (bits of x | y) in the span
};

// Read this thread's piece of the staged span, block-wide popc prefixes, then the walk of the piece's
// set bits: add, re-test, pack.  The caller has waited for the span's copies.  With EMIT the surviving
// sums go to `out` and ao[] receives the piece of Bo; without it the survivors are only counted.
// Contains two walkers_sync(); on return sh.ws[] holds the per-warp survivor totals and nobody reads
// the stage any more.
template <bool EMIT>
__device__ __forceinline__ WalkOut walk_span(const uint32_t *stage, uint32_t *out, MergeShared &sh, uint32_t By0, uint32_t Xb,
                                             uint32_t Yb, uint32_t m, uint32_t mt, uint32_t (&ao)[4], int tid,
                                             uint16_t *run_at = nullptr, uint16_t *run_k = nullptr, uint32_t trace_it = 99u) {
    const int lane = tid & 31, warp = tid >> 5;
    uint32_t ax[4], ay[4];
    read_piece(stage, By0, m, mt, tid, ax, ay);
    const uint32_t cx = __popc(ax[0]) + __popc(ax[1]) + __popc(ax[2]) + __popc(ax[3]);
    const uint32_t cy = __popc(ay[0]) + __popc(ay[1]) + __popc(ay[2]) + __popc(ay[3]);
    const uint32_t cu = __popc(ax[0] | ay[0]) + __popc(ax[1] | ay[1]) + __popc(ax[2] | ay[2]) + __popc(ax[3] | ay[3]);
    const uint32_t sxy = warp_incl_scan(cx | (cy << 16), lane);
    const uint32_t su = warp_incl_scan(cu, lane);
    if (lane == 31) {
        sh.wxy[warp] = sxy;
        sh.wu[warp] = su;
    }
    walkers_sync();  // #1: warp totals are visible
    PICI_TR(trace_it, 2);
    // prefix over the 16 warp totals: lanes 0..15 of every warp scan them with shuffles (an unrolled loop over
    // the 16 shared-memory words costs ~80 instructions per thread; the kernel is issue-bound on exactly this
    // kind of per-span bookkeeping: 60 % issue activity with almost no values to add at 99.99 % sparsity)
    uint32_t pw = lane < kMergeWarps ? sh.wxy[lane] : 0u, uw = lane < kMergeWarps ? sh.wu[lane] : 0u;
#pragma unroll
    for (int d = 1; d < kMergeWarps; d <<= 1) {
        const uint32_t o1 = __shfl_up_sync(kFull, pw, d), o2 = __shfl_up_sync(kFull, uw, d);
        if (lane >= d) {
            pw += o1;
            uw += o2;
        }
    }
    const uint32_t cand_total = __shfl_sync(kFull, uw, kMergeWarps - 1);
    const uint32_t bxy = warp > 0 ? __shfl_sync(kFull, pw, (warp + 31) & 31) : 0u;   // inclusive prefix of warp - 1
    const uint32_t bu = warp > 0 ? __shfl_sync(kFull, uw, (warp + 31) & 31) : 0u;
    if (EMIT && cand_total > kOutWords) {   // uniform: more candidates than the output region holds
        WalkOut none = {0u, 0u, 0u, cand_total};
        return none;                        // the caller takes the tile-by-tile path (only one barrier passed)
    }
    uint32_t kx = Xb + (bxy & 0xFFFFu) + (sxy & 0xFFFFu) - cx;
    uint32_t ky = Yb + (bxy >> 16) + (sxy >> 16) - cy;
    const uint32_t ko0 = bu + su - cu;
    uint32_t ko = ko0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        uint32_t u = ax[q] | ay[q], o = 0;
        while (u) {
            const uint32_t bit = u & (0u - u);
            u ^= bit;
            float x = 0.0f, y = 0.0f;
            if (ax[q] & bit) x = __uint_as_float(stage[kx++]);
            if (ay[q] & bit) y = __uint_as_float(stage[ky++]);
            const uint32_t sum = __float_as_uint(__fadd_rn(x, y));   // received + local (C9 #7)
            if (nz32(sum)) {
                o |= bit;
                if (EMIT) out[ko] = sum;
                ++ko;
            }
        }
        ao[q] = o;
    }
    WalkOut r;
    r.k = ko - ko0;
    r.ko0 = ko0;
    r.sk = warp_incl_scan(r.k, lane);
    r.cand_total = cand_total;
    if (lane == 31) sh.ws[warp] = r.sk;
    if (run_at != nullptr) {   // where this thread's survivors sit: only read if the span had a cancellation
        run_at[tid] = (uint16_t)ko0;
        run_k[tid] = (uint16_t)r.k;
    }
    walkers_sync();  // #2: survivor totals and the output region are visible; the stage is no longer read
    PICI_TR(trace_it, 4);
    return r;
}

// ---- Phase 2: counts -> exclusive prefix: the round-robin scan of pici_common.cuh ----------------------
__device__ __forceinline__ void publish_span(const MergeArgs &a, uint32_t g, uint32_t it, uint32_t c, uint32_t total) {
    rr_publish(a.scan, g, it, c, total);
}
__device__ __forceinline__ uint32_t iter_lookback(const MergeArgs &a, uint32_t G, uint32_t it, uint32_t c, uint32_t &E,
                                                  uint32_t &E_it, int lane) {
    return rr_lookback(a.scan, G, it, c, E, E_it, lane);
}

// Io for the mt tiles of a span (one warp; lane i < mt holds tc = survivors of tile ts + i).
__device__ __forceinline__ void write_index(const MergeArgs &a, uint32_t ts, uint32_t mt, uint32_t tc, uint32_t excl, int lane) {
    const uint32_t tincl = warp_incl_scan((uint32_t)lane < mt ? tc : 0u, lane);
    if ((uint32_t)lane < mt) {
        a.Io[ts + lane] = excl + tincl - tc;
        if (ts + lane + 1 == a.T) a.Io[a.T] = excl + tincl;
    }
}

// One warp writes a walked span's output region to Ao + off.  Packed (no cancellation): the region is
// contiguous.  Otherwise the walkers left their runs (first word, survivors) in shared memory: lane l
// moves the runs of threads 32q + l, q = 0..15, offsets from a running warp scan.
__device__ __forceinline__ void warp_flush(uint32_t *__restrict__ Ao, const uint32_t *out, uint32_t off, uint32_t surv_total,
                                           uint32_t cand_total, const uint16_t *run_at, const uint16_t *run_k, int lane) {
    uint32_t *dst = Ao + off;
    if (surv_total == cand_total) {
        for (uint32_t i = lane; i < surv_total; i += 32) dst[i] = out[i];
        return;
    }
    uint32_t base = 0;
    for (int q = 0; q < kMergeWarps; ++q) {
        const uint32_t k = run_k[32 * q + lane], at = run_at[32 * q + lane];
        const uint32_t incl = warp_incl_scan(k, lane);
        for (uint32_t i = 0; i < k; ++i) dst[base + incl - k + i] = out[at + i];
        base += __shfl_sync(kFull, incl, 31);
    }
}

// Write a walked span's output region to Ao + off.  Packed (no cancellation happened): the region is
// contiguous; otherwise every thread moves its own run (before = survivors of earlier threads).
__device__ __forceinline__ void span_flush(uint32_t *__restrict__ Ao, const uint32_t *out, const WalkOut &r, uint32_t off,
                                           uint32_t surv_total, uint32_t before, int tid) {
    uint32_t *dst = Ao + off;
    if (surv_total == r.cand_total) {
        for (uint32_t i = tid; i < surv_total; i += kMergeThreads) dst[i] = out[i];
    } else {
        for (uint32_t i = 0; i < r.k; ++i) dst[before + i] = out[r.ko0 + i];
    }
}

// Survivors of earlier warps / of the whole block, from sh.ws[] (after walk_span's last barrier).
__device__ __forceinline__ void survivor_sums(const MergeShared &sh, int warp, uint32_t &before, uint32_t &total) {
    before = 0;
    total = 0;
#pragma unroll
    for (int q = 0; q < kMergeWarps; ++q) {
        const uint32_t v = sh.ws[q];
        if (q < warp) before += v;
        total += v;
    }
}

// One tile (a span of m = 1) end to end, copies included (walker warp 0 issues them on slow_bar): the
// slow path of a span that does not fit.  Starts with a walkers_sync() (the stage may still be read).
template <bool EMIT>
__device__ __forceinline__ WalkOut tile_pass(const MergeArgs &a, uint32_t *stage, uint32_t *out, MergeShared &sh,
                                             uint32_t t, uint32_t x0, uint32_t x1, uint32_t y0, uint32_t y1, uint32_t bar,
                                             uint32_t &parity, int tid) {
    walkers_sync();
    const SpanLayout L = span_stage(a, stage, bar, t, 1u, 1u, x0, x1 - x0, y0, y1 - y0, tid < 32, tid & 31);
    mbar_wait(bar, parity);
    parity ^= 1u;
    uint32_t ao[4];
    const WalkOut r = walk_span<EMIT>(stage, out, sh, L.By0, L.Xb, L.Yb, 1u, 1u, ao, tid);
    if (EMIT) store_piece(a, t, 1u, 1u, tid, ao);
    return r;
}


constexpr int kMergeLaunchThreads = kMergeThreads + 64;   // 16 walker warps + one service warp per stage

__global__ void __launch_bounds__(kMergeLaunchThreads, kMergeMinBlocks)
reduce_ss_kernel(MergeArgs a, const int32_t *gate, int32_t gate_value) {
    extern __shared__ __align__(128) uint32_t pool[];
    __shared__ MergeShared sh;
    if (gate_closed(gate, gate_value)) return;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t T = a.T;
    const uint32_t G = gridDim.x;

    // ---- span length of this launch: the largest m whose AVERAGE span (plus 1/16 margin) fits a stage
    // and the output region, from the totals Ix[T], Iy[T]; halved while the launch has fewer than two
    // spans per CTA (ring chunks are a few thousand tiles).
    uint32_t m = 1;
    {
        const uint64_t nx = __ldg(a.Ix + T), ny = __ldg(a.Iy + T);
        const uint64_t avg = (nx + ny + T - 1) / T;   // values per tile, X and Y together
        // candidates per tile: the union of two INDEPENDENT supports of these densities (a span whose
        // union is larger than the output region takes the slow path, so this is an estimate, not a bound)
        const uint64_t both = (nx / T) * (ny / T) / kTile;
        const uint64_t uni = min(avg - min(both, avg), (uint64_t)kTile);
#pragma unroll
        for (uint32_t mm = kMaxSpan; mm >= 2; mm /= 2) {
            const uint64_t vals = avg * mm + 16, cand = uni * mm;
            if (m == 1 && 2u * mm * kTileWords + vals + vals / 16 <= kStageWords && cand + cand / 16 <= kOutWords) m = mm;
        }
        while (m > 1 && (T + m - 1) / m < 2u * G) m /= 2;
    }
    const uint32_t spans = (T + m - 1) / m;
    uint32_t *const out = pool + 2 * kStageWords;
    const uint32_t full0 = smem_u32(&sh.full[0]), free0 = smem_u32(&sh.stage_free[0]);
    const uint32_t cnt0 = smem_u32(&sh.counts[0]), lbd0 = smem_u32(&sh.lb_done[0]), fl0 = smem_u32(&sh.flushed[0]);
    const uint32_t slow_bar = smem_u32(&sh.slow_bar);
    if (tid == 0) {
#pragma unroll
        for (uint32_t s = 0; s < 2; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(free0 + 8 * s, 1);
            mbar_init(cnt0 + 8 * s, 1);
            mbar_init(lbd0 + 8 * s, 1);
            mbar_init(fl0 + 8 * s, 1);
        }
        mbar_init(slow_bar, 1);
    }
    __syncthreads();
    // Spans are dealt round-robin: CTA c takes spans c, c + G, c + 2G, ...; j counts this CTA's spans,
    // span j lives in stage / output region s = j & 1.  The launch is cooperative (all G CTAs are
    // co-resident), so every span a look-back waits on belongs to a running CTA, and span j of a CTA
    // only depends on spans <= j of the others.
    const uint32_t c = blockIdx.x;

    if (warp >= kMergeWarps) {
        // ============================ service warp of stage s ============================
        // For this CTA's spans j = s, s + 2, ...: start the copies of span j (stage s is free once the
        // walkers have left span j - 2); once span j's count is published take its prefix, write its
        // index entries, write its output region to Ao and release the region.  The walkers never wait
        // for a look-back: they only need stage s filled and region s released two spans later.
        const uint32_t s = (uint32_t)warp - kMergeWarps;
        uint32_t *const stage = pool + s * kStageWords;
        const uint32_t *const out_s = out + s * kOutWords;
        auto load_index = [&](uint32_t gg, uint32_t &ixl, uint32_t &iyl) {   // lanes 0..mt hold I[ts .. ts+mt]
            ixl = 0;
            iyl = 0;
            if (gg < spans) {
                const uint32_t ts = gg * m, jj = min((uint32_t)lane, min(m, T - ts));
                ixl = __ldg(a.Ix + ts + jj);
                iyl = __ldg(a.Iy + ts + jj);
            }
        };
        auto prepare = [&](uint32_t gg, uint32_t ixl, uint32_t iyl) {
            if (gg >= spans) return;
            const uint32_t ts = gg * m, mt = min(m, T - ts);
            const uint32_t xs = __shfl_sync(kFull, ixl, 0), xe = __shfl_sync(kFull, ixl, mt);
            const uint32_t ys = __shfl_sync(kFull, iyl, 0), ye = __shfl_sync(kFull, iyl, mt);
            const bool fits = span_fits(m, xe - xs, ye - ys, mt);
            const SpanLayout L = span_stage(a, stage, full0 + 8 * s, ts, m, mt, xs, xe - xs, ys, ye - ys, false, lane);
            if (lane == 0) {
                sh.info[s].fits = fits ? 1u : 0u;
                sh.info[s].Xb = L.Xb;
                sh.info[s].Yb = L.Yb;
                sh.info[s].xs = xs;
                sh.info[s].ys = ys;
            }
            __syncwarp();
            if (fits) span_stage(a, stage, full0 + 8 * s, ts, m, mt, xs, xe - xs, ys, ye - ys, true, lane);
            else if (lane == 0) mbar_arrive(full0 + 8 * s);   // nothing to copy: the walkers stage tile by tile
        };
        uint32_t ixa, iya;
        load_index(c + s * G, ixa, iya);
        prepare(c + s * G, ixa, iya);
        load_index(c + (s + 2) * G, ixa, iya);   // entries of the next span to prepare, one ahead
        uint32_t E = 0, E_it = 0;                // survivors of the complete iterations [0, E_it)
        for (uint32_t j = s; c + j * G < spans; j += 2) {
            const uint32_t ph = (j >> 1) & 1u;
            const uint32_t ts = (c + j * G) * m, mt = min(m, T - ts);
            // Copies first when the stage is already free (they are what the walkers wait for two spans
            // later); a span on the slow path frees its stage only after its look-back, so poll both.
            bool prepared = false;
            for (;;) {
                if (!prepared && mbar_test(free0 + 8 * s, ph)) {
                    prepare(c + (j + 2) * G, ixa, iya);
                    load_index(c + (j + 4) * G, ixa, iya);
                    prepared = true;
                }
                if (mbar_test(cnt0 + 8 * s, ph)) break;
            }
            const uint32_t excl = iter_lookback(a, G, j, c, E, E_it, lane);
            write_index(a, ts, mt, (uint32_t)lane < mt ? sh.tcs[s][lane] : 0u, excl, lane);
            const uint32_t tot = sh.tot[s], cand = sh.cand[s];
            if (lane == 0) {
                sh.excl[s] = excl;
                mbar_arrive(lbd0 + 8 * s);
            }
            if (!prepared) {
                mbar_wait(free0 + 8 * s, ph);
                prepare(c + (j + 2) * G, ixa, iya);
                load_index(c + (j + 4) * G, ixa, iya);
            }
            if (cand != ~0u) warp_flush(a.Ao, out_s, excl, tot, cand, sh.run_at[s], sh.run_k[s], lane);
            __syncwarp();
            if (lane == 0) mbar_arrive(fl0 + 8 * s);
        }
        return;
    }

    // ======================================= walker warps =======================================
    // The loop is instantiated once per span length, so the piece width, the tile / warp ratio and the empty
    // words of narrow pieces are compile-time facts (the kernel is bound by exactly these instructions).
    uint32_t slow_par = 0;
    auto walkers = [&](auto span_len) {
        constexpr uint32_t M = decltype(span_len)::value;
        for (uint32_t j = 0; c + j * G < spans; ++j) {
            const uint32_t s = j & 1u, ph = (j >> 1) & 1u;
            const uint32_t g = c + j * G, ts = g * M, mt = min(M, T - ts);
            uint32_t *const stage = pool + s * kStageWords;
            uint32_t *const out_s = out + s * kOutWords;
            PICI_TR(j, 0);
            // span j - 2 must have left output region s before anything is written to it; warp 0 waits for all (the
            // first write comes behind the walkers' barrier #1, which warp 0 joins afterwards): 15 warps fewer polling
            if (j >= 2 && warp == 0) mbar_wait(fl0 + 8 * s, ph ^ 1u);
            mbar_wait(full0 + 8 * s, ph);
            PICI_TR(j, 1);
            const SpanInfo info = sh.info[s];

            bool slow = info.fits == 0u;
            if (!slow) {
                // ---- walk, publish the count; the service warp of stage s does the rest ---------------------
                uint32_t ao[4];
                const WalkOut r = walk_span<true>(stage, out_s, sh, M * kTileWords, info.Xb, info.Yb, M, mt, ao, tid,
                                                  sh.run_at[s], sh.run_k[s], j);
                slow = r.cand_total > kOutWords;   // uniform; nothing was written
                if (!slow) {
                    if (warp == 0) {   // the other 15 warps go straight on to their piece of Bo and the next span
                        const uint32_t surv_total = warp_sum(lane < kMergeWarps ? sh.ws[lane] : 0u);
                        const uint32_t wpt = (uint32_t)kMergeWarps / M;   // a tile is covered by 16/m consecutive warps
                        uint32_t tc = 0;
                        if ((uint32_t)lane < mt)
                            for (uint32_t q = 0; q < wpt; ++q) tc += sh.ws[lane * wpt + q];
                        if (lane < kMaxSpan) sh.tcs[s][lane] = tc;
                        if (lane == 0) {
                            sh.tot[s] = surv_total;
                            sh.cand[s] = r.cand_total;
                            publish_span(a, g, j, c, surv_total);
                            mbar_arrive(free0 + 8 * s);           // every walker is past barrier #2
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(cnt0 + 8 * s);
                    }
                    store_piece(a, ts, M, mt, tid, ao);
                    PICI_TR(j, 6);
                }
            }
            if (slow) {
                // ---- the span does not fit: tile by tile (one tile always fits), two sweeps -----------------
                // Sweep 1 counts the survivors of every tile so that the span's count is published before
                // anything waits (no other CTA ever waits on a half-processed span); sweep 2 emits and the
                // walkers write Ao themselves (cand = ~0 tells the service warp not to).
                for (uint32_t i = 0; i < mt; ++i) {
                    const uint32_t x0 = __ldg(a.Ix + ts + i), x1 = __ldg(a.Ix + ts + i + 1);
                    const uint32_t y0 = __ldg(a.Iy + ts + i), y1 = __ldg(a.Iy + ts + i + 1);
                    tile_pass<false>(a, stage, out_s, sh, ts + i, x0, x1, y0, y1, slow_bar, slow_par, tid);
                    if (tid == 0) {
                        uint32_t cnt = 0;
                        for (int q = 0; q < kMergeWarps; ++q) cnt += sh.ws[q];
                        sh.tcs[s][i] = cnt;
                    }
                }
                walkers_sync();
                if (tid == 0) {
                    uint32_t span_total = 0;
                    for (uint32_t i = 0; i < mt; ++i) span_total += sh.tcs[s][i];
                    sh.tot[s] = span_total;
                    sh.cand[s] = ~0u;
                    publish_span(a, g, j, c, span_total);
                    mbar_arrive(cnt0 + 8 * s);
                }
                mbar_wait(lbd0 + 8 * s, ph);
                uint32_t off = sh.excl[s];
                for (uint32_t i = 0; i < mt; ++i) {
                    const uint32_t x0 = __ldg(a.Ix + ts + i), x1 = __ldg(a.Ix + ts + i + 1);
                    const uint32_t y0 = __ldg(a.Iy + ts + i), y1 = __ldg(a.Iy + ts + i + 1);
                    const WalkOut r = tile_pass<true>(a, stage, out_s, sh, ts + i, x0, x1, y0, y1, slow_bar, slow_par, tid);
                    uint32_t before, surv_total;
                    survivor_sums(sh, warp, before, surv_total);
                    span_flush(a.Ao, out_s, r, off, surv_total, before + r.sk - r.k, tid);
                    off += surv_total;
                }
                walkers_sync();
                if (tid == 0) mbar_arrive(free0 + 8 * s);
            }
        }
    };
    switch (m) {
        case 16: walkers(std::integral_constant<uint32_t, 16>{}); break;
        case 8: walkers(std::integral_constant<uint32_t, 8>{}); break;
        case 4: walkers(std::integral_constant<uint32_t, 4>{}); break;
        case 2: walkers(std::integral_constant<uint32_t, 2>{}); break;
        default: walkers(std::integral_constant<uint32_t, 1>{}); break;
    }
}

cudaError_t launch_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                             const uint32_t *Iy, const void *Ay, uint64_t n, uint64_t *Bo, uint32_t *Io,
                             void *Ao, void *ws, Gate g, cudaStream_t s) {
    if (n == 0) return launch_set_u32(Io, 0u, g, s);
    const uint64_t T = (n + kTile - 1) / kTile;
    const size_t smem = (size_t)kPoolWords * sizeof(uint32_t);
    static bool configured_on[64] = {false};
    static int per_sm_on[64] = {0};
    bool &configured = configured_on[current_device_slot()];
    int &per_sm = per_sm_on[current_device_slot()];
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(reduce_ss_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int v = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, reduce_ss_kernel, kMergeLaunchThreads, smem);
        if (e != cudaSuccess) return e;
        per_sm = v > 0 ? v : 1;
        configured = true;
    }
    // the span length is chosen on the device.  A chunk of a few thousand tiles does not need the whole GPU:
    // one CTA per 16 tiles leaves room for the other logical ranks' launches of the same ring step
    uint64_t blocks = (T + 15) / 16;
    uint64_t cap = (uint64_t)num_sms() * per_sm;   // cooperative: exactly one co-resident wave
    if (cap > kMaxGrid) cap = kMaxGrid;
    if (blocks > cap) blocks = cap;
    // workspace: [header][span words: T][iteration words: iters][group words: iters * ngrp], all zero
    const uint64_t iters = (T + blocks - 1) / blocks, ngrp = (blocks + 31) / 32;
    const uint64_t words = T + iters * (1 + ngrp);
    if ((uint64_t)kWsHeaderBytes + words * 8 > scan_workspace_bytes(n)) return cudaErrorInvalidValue;   // cannot happen
    cudaError_t e = cudaMemsetAsync(ws, 0, (size_t)kWsHeaderBytes + words * 8, s);
    if (e != cudaSuccess) return e;
    uint64_t *base = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(ws) + kWsHeaderBytes);
    MergeArgs a;
    a.Bx = Bx; a.By = By; a.Ix = Ix; a.Iy = Iy;
    a.Ax = reinterpret_cast<const uint32_t *>(Ax); a.Ay = reinterpret_cast<const uint32_t *>(Ay);
    a.Bo = Bo; a.Io = Io; a.Ao = reinterpret_cast<uint32_t *>(Ao);
    a.scan.unit_word = base; a.scan.iter_word = base + T; a.scan.grp_word = base + T + iters;
    a.scan.ngrp = (uint32_t)ngrp;
    a.T = (uint32_t)T;
    a.a_limit = (n * 4) & ~15ull;
#ifdef PICI_MERGE_TRACE
    {
        uint64_t *tr = base + words;   // needs a workspace with 296 * 16 * 8 spare words
        cudaMemcpyToSymbolAsync(g_merge_trace, &tr, sizeof(tr), 0, cudaMemcpyHostToDevice, s);
    }
#endif
    const int32_t *gate_ptr = g.ptr;
    int32_t gate_value = g.value;
    void *params[] = {&a, &gate_ptr, &gate_value};
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(reduce_ss_kernel), dim3((unsigned)blocks),
                                       dim3(kMergeLaunchThreads), params, smem, s);
}

}  // namespace pici
