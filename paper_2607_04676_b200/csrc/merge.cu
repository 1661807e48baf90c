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
//   * a CTA of 256 threads takes a group of 8 consecutive tiles by dynamic ticket and cuts it into
//     spans of m = 8, 4, 2 or 1 tiles - the largest m whose X values, Y values and worst-case output
//     all fit the CTA's shared-memory pool (read from Ix, Iy; one tile always fits).  Sparse inputs
//     run 8 tiles per span (many tiles in flight, one look-back per 8 tiles), dense ones 1 tile per
//     span with all 256 threads on it;
//   * thread j owns the 16m-bit piece j of the span (128 / 64 / 32 / 16 bits: one coalesced load of
//     consecutive pieces); the span's X and Y values are contiguous in Ax / Ay and are staged in the
//     pool by two 1-D TMA bulk copies (16-byte aligned window, < 16-byte tail by plain loads);
//   * x's and y's cursors come from the block-wide popc prefix of their own pieces, the candidate
//     cursor from the popc prefix of the OR; every thread walks the set bits of its piece, adds, tests
//     the predicate and packs its surviving sums into its own run of the pool's output region (runs
//     start at the OR-prefix, so they never overlap);
//   * the span's per-tile survivor counts go through the same per-tile decoupled look-back as compress
//     (Phase 2), and the output region is written to Ao with coalesced stores.  Only spans that
//     actually had a cancellation take the thread-by-thread copy.
#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

constexpr int kMergeWarps = 8;
constexpr int kMergeThreads = kMergeWarps * 32;
constexpr int kMaxSpan = 8;                             // tiles per ticket: 8, 4, 2 or 1
constexpr uint32_t kPoolWords = 3 * kTile + 16;         // X window + Y window + output region of ONE tile
constexpr int kMergeMinBlocks = 4;

struct MergeShared {
    uint64_t mbar;
    uint32_t ticket;
    uint32_t span_excl;               // exclusive prefix (survivors before the span) from the look-back
    uint32_t wxy[kMergeWarps];        // per-warp totals: popc(x piece) | popc(y piece) << 16
    uint32_t wu[kMergeWarps];         // per-warp totals: popc(x | y)
    uint32_t ws[kMergeWarps];         // per-warp totals: survivors
    uint32_t tc[kMaxSpan];            // per-tile survivors of a span walked tile by tile
};

// Stage A[beg .. beg+cnt) (4-byte elements) at pool word `dstw` (a multiple of 4): element i lands at
// pool[dstw + (beg & 3) + i].  Called by one warp; lane 0 issues the bulk copy (the caller has posted
// the expected byte count), lanes 0..2 move the tail.
__device__ __forceinline__ uint32_t bulk_bytes_of(uint32_t beg, uint32_t cnt) {
    const uint64_t a_beg = (uint64_t)beg * 4, a_end = a_beg + (uint64_t)cnt * 4;
    const uint64_t start_al = a_beg & ~15ull, end_dn = a_end & ~15ull;
    return end_dn > start_al ? (uint32_t)(end_dn - start_al) : 0u;
}
__device__ __forceinline__ void stage_values(uint32_t *pool, uint32_t dstw, const uint32_t *__restrict__ A,
                                             uint32_t beg, uint32_t cnt, uint32_t bar, int lane) {
    if (cnt == 0) return;
    const uint64_t a_beg = (uint64_t)beg * 4, a_end = a_beg + (uint64_t)cnt * 4;
    const uint64_t start_al = a_beg & ~15ull, end_dn = a_end & ~15ull;
    const uint32_t bulk = end_dn > start_al ? (uint32_t)(end_dn - start_al) : 0u;
    if (bulk != 0 && lane == 0)
        bulk_g2s(smem_u32(pool + dstw), reinterpret_cast<const unsigned char *>(A) + start_al, bulk, bar);
    const uint64_t tail_beg = bulk != 0 ? end_dn : a_beg;
    const uint32_t tail_cnt = (uint32_t)(a_end - tail_beg) / 4;
    if ((uint32_t)lane < tail_cnt) pool[dstw + (uint32_t)(tail_beg - start_al) / 4 + lane] = A[tail_beg / 4 + lane];
}


struct MergeArgs {
    const uint64_t *Bx, *By;
    const uint32_t *Ix, *Iy, *Ax, *Ay;
    uint64_t *Bo;
    uint32_t *Io, *Ao;
    uint64_t *status;
    uint32_t T;
};

// What a thread keeps from one walk of a span.
struct WalkOut {
    uint32_t k;            // this thread's survivors
    uint32_t ko0;          // pool word of this thread's run in the output region
    uint32_t sk;           // inclusive warp scan of k
    uint32_t Ob;           // pool word where the span's output region starts
    uint32_t cand_total;   // candidates (bits of x | y) in the span
};

// One pass over the span of mt (<= m) tiles that starts at tile ts: stage the span's X and Y values,
// load this thread's 16*m-bit piece of Bx / By, block-wide popc prefixes, walk the set bits.  With
// EMIT the surviving sums are packed into the pool's output region and the piece of Bo is written;
// without it only the survivors are counted (first sweep of a span that does not fit the pool).
// On return sh.ws[] holds the per-warp survivor totals (after a __syncthreads()).
template <bool EMIT>
__device__ __forceinline__ WalkOut span_walk(const MergeArgs &a, uint32_t *pool, MergeShared &sh, uint32_t ts,
                                             uint32_t m, uint32_t mt, uint32_t xs, uint32_t xe, uint32_t ys,
                                             uint32_t ye, uint32_t bar, uint32_t &parity, int tid) {
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t nx = xe - xs, ny = ye - ys;
    const uint32_t xw = ((xs & 3u) + nx + 3u) & ~3u;              // X window (words)
    const uint32_t yw = ((ys & 3u) + ny + 3u) & ~3u;              // Y window (words)
    const uint32_t Xb = (xs & 3u), Yb = xw + (ys & 3u), Ob = xw + yw;   // first x / y / output word
    const uint32_t tx = bulk_bytes_of(xs, nx) + bulk_bytes_of(ys, ny);

    if (warp == 0) {
        if (lane == 0 && tx != 0) {
            fence_proxy_async_smem();
            mbar_expect_tx(bar, tx);
        }
        stage_values(pool, 0, a.Ax, xs, nx, bar, lane);
        stage_values(pool, xw, a.Ay, ys, ny, bar, lane);
    }

    // ---- this thread's piece of the span: 16*m bits of Bx, By ---------------------------------------
    uint32_t ax[4] = {0, 0, 0, 0}, ay[4] = {0, 0, 0, 0};
    const bool valid = (uint32_t)tid * m < (uint32_t)kMergeThreads * mt;   // piece inside the span's tiles
    const size_t wbase = (size_t)ts * kSide;
    if (valid) {
        if (m == 8) {
            const uint4 p = __ldg(reinterpret_cast<const uint4 *>(a.Bx + wbase) + tid);
            const uint4 q = __ldg(reinterpret_cast<const uint4 *>(a.By + wbase) + tid);
            ax[0] = p.x; ax[1] = p.y; ax[2] = p.z; ax[3] = p.w;
            ay[0] = q.x; ay[1] = q.y; ay[2] = q.z; ay[3] = q.w;
        } else if (m == 4) {
            const uint2 p = __ldg(reinterpret_cast<const uint2 *>(a.Bx + wbase) + tid);
            const uint2 q = __ldg(reinterpret_cast<const uint2 *>(a.By + wbase) + tid);
            ax[0] = p.x; ax[1] = p.y;
            ay[0] = q.x; ay[1] = q.y;
        } else if (m == 2) {
            ax[0] = __ldg(reinterpret_cast<const uint32_t *>(a.Bx + wbase) + tid);
            ay[0] = __ldg(reinterpret_cast<const uint32_t *>(a.By + wbase) + tid);
        } else {
            ax[0] = __ldg(reinterpret_cast<const uint16_t *>(a.Bx + wbase) + tid);
            ay[0] = __ldg(reinterpret_cast<const uint16_t *>(a.By + wbase) + tid);
        }
    }
    const uint32_t cx = __popc(ax[0]) + __popc(ax[1]) + __popc(ax[2]) + __popc(ax[3]);
    const uint32_t cy = __popc(ay[0]) + __popc(ay[1]) + __popc(ay[2]) + __popc(ay[3]);
    const uint32_t cu = __popc(ax[0] | ay[0]) + __popc(ax[1] | ay[1]) + __popc(ax[2] | ay[2]) + __popc(ax[3] | ay[3]);
    const uint32_t sxy = warp_incl_scan(cx | (cy << 16), lane);
    const uint32_t su = warp_incl_scan(cu, lane);
    if (lane == 31) {
        sh.wxy[warp] = sxy;
        sh.wu[warp] = su;
    }
    __syncthreads();  // #1: warp totals and the tail words of the staged values are visible
    uint32_t bxy = 0, bu = 0, cand_total = 0;
#pragma unroll
    for (int w = 0; w < kMergeWarps; ++w) {
        const uint32_t p = sh.wxy[w], q = sh.wu[w];
        if (w < warp) {
            bxy += p;
            bu += q;
        }
        cand_total += q;
    }
    uint32_t kx = Xb + (bxy & 0xFFFFu) + (sxy & 0xFFFFu) - cx;
    uint32_t ky = Yb + (bxy >> 16) + (sxy >> 16) - cy;
    const uint32_t ko0 = Ob + bu + su - cu;
    uint32_t ko = ko0;
    if (tx != 0) {
        mbar_wait(bar, parity);
        parity ^= 1u;
    }

    // ---- walk the set bits of the piece: add, re-test, pack ------------------------------------------
    uint32_t ao[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        uint32_t u = ax[q] | ay[q], o = 0;
        while (u) {
            const uint32_t bit = u & (0u - u);
            u ^= bit;
            float x = 0.0f, y = 0.0f;
            if (ax[q] & bit) x = __uint_as_float(pool[kx++]);
            if (ay[q] & bit) y = __uint_as_float(pool[ky++]);
            const uint32_t sum = __float_as_uint(__fadd_rn(x, y));   // received + local (C9 #7)
            if (nz32(sum)) {
                o |= bit;
                if (EMIT) pool[ko] = sum;
                ++ko;
            }
        }
        ao[q] = o;
    }
    if (EMIT && valid) {
        if (m == 8) reinterpret_cast<uint4 *>(a.Bo + wbase)[tid] = make_uint4(ao[0], ao[1], ao[2], ao[3]);
        else if (m == 4) reinterpret_cast<uint2 *>(a.Bo + wbase)[tid] = make_uint2(ao[0], ao[1]);
        else if (m == 2) reinterpret_cast<uint32_t *>(a.Bo + wbase)[tid] = ao[0];
        else reinterpret_cast<uint16_t *>(a.Bo + wbase)[tid] = (uint16_t)ao[0];
    }
    WalkOut r;
    r.k = ko - ko0;
    r.ko0 = ko0;
    r.sk = warp_incl_scan(r.k, lane);
    r.Ob = Ob;
    r.cand_total = cand_total;
    if (lane == 31) sh.ws[warp] = r.sk;
    __syncthreads();  // #2: survivor totals and the output region are visible
    return r;
}

// Phase 2 for a span (one warp; lane i < mt holds tc = survivors of tile ts + i).  ONE status word per
// SPAN (index g): the aggregate is the span's survivor total, so a 32-entry look-back window covers
// 32 * m tiles and the chain of hops a look-back has to walk is m times shorter than with per-tile
// words (profiles/r1b: 49 % of reduce_ss's stall samples sat behind this look-back).  Publishes the
// aggregate, looks back from span g, publishes the inclusive prefix, writes Io for the span's tiles.
// Returns the number of survivors before tile ts.
__device__ __forceinline__ uint32_t span_lookback(const MergeArgs &a, uint32_t g, uint32_t ts, uint32_t mt, uint32_t tc,
                                                  int lane) {
    const uint32_t tincl = warp_incl_scan((uint32_t)lane < mt ? tc : 0u, lane);
    const uint32_t total = __shfl_sync(kFull, tincl, 31);
    if (lane == 0) st_status(a.status + g, g == 0 ? kStPrefix : kStAggregate, total);
    uint32_t excl = 0;
    int64_t pos = g;
    while (pos > 0) {
        const int64_t idx = pos - 1 - lane;
        uint64_t st;
        unsigned pm, em, ns = 8;
        for (;;) {
            st = idx >= 0 ? ld_status(a.status + idx) : (kStPrefix << 32);
            const uint32_t flag = (uint32_t)(st >> 32);
            pm = __ballot_sync(kFull, flag == (uint32_t)kStPrefix);
            em = __ballot_sync(kFull, flag == (uint32_t)kStEmpty);
            const unsigned rel = pm ? ((pm & (0u - pm)) | ((pm & (0u - pm)) - 1u)) : kFull;
            if ((em & rel) == 0u) {
                excl += warp_sum(((1u << lane) & rel) ? (uint32_t)st : 0u);
                break;
            }
            __nanosleep(ns);
            if (ns < 64) ns += ns;
        }
        if (pm) break;
        pos -= 32;
    }
    if (lane == 0 && g != 0) st_status(a.status + g, kStPrefix, excl + total);
    if ((uint32_t)lane < mt) {
        a.Io[ts + lane] = excl + tincl - tc;
        if (ts + lane + 1 == a.T) a.Io[a.T] = excl + tincl;
    }
    return excl;
}

// Write a walked span's output region to Ao + off.  packed: no cancellation happened, the region is
// contiguous; otherwise every thread moves its own run (before = survivors of earlier threads).
__device__ __forceinline__ void span_flush(uint32_t *__restrict__ Ao, const uint32_t *pool, const WalkOut &r,
                                           uint32_t off, uint32_t surv_total, uint32_t before, int tid) {
    uint32_t *dst = Ao + off;
    if (surv_total == r.cand_total) {
        for (uint32_t i = tid; i < surv_total; i += kMergeThreads) dst[i] = pool[r.Ob + i];
    } else {
        for (uint32_t i = 0; i < r.k; ++i) dst[before + i] = pool[r.ko0 + i];
    }
}

__global__ void __launch_bounds__(kMergeThreads, kMergeMinBlocks)
reduce_ss_kernel(MergeArgs a, uint32_t *ticket, const int32_t *gate, int32_t gate_value) {
    extern __shared__ __align__(128) uint32_t pool[];
    __shared__ MergeShared sh;
    if (gate_closed(gate, gate_value)) return;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    const uint32_t T = a.T;

    // ---- span length of this launch: the largest m in {8, 4, 2, 1} whose AVERAGE span (plus 1/16
    // margin) fits the pool; read from the totals Ix[T], Iy[T].  A span that still does not fit is
    // processed tile by tile in two sweeps (count, then emit), see below.
    uint32_t m = 1;
    {
        const uint64_t tot = (uint64_t)a.Ix[T] + (uint64_t)a.Iy[T];
        const uint64_t avg = (tot + T - 1) / T;   // values per tile, X and Y together
#pragma unroll
        for (uint32_t mm = 8; mm >= 2; mm /= 2) {
            const uint64_t need = avg * mm + min(avg, (uint64_t)kTile) * mm + 8;   // values + worst-case output
            if (m == 1 && need + need / 16 <= kPoolWords) m = mm;
        }
    }
    const uint32_t spans = (T + m - 1) / m;
    const uint32_t bar = smem_u32(&sh.mbar);
    if (tid == 0) {
        mbar_init(bar, 1);
        sh.ticket = atomicAdd(ticket, 1u);
    }
    __syncthreads();
    uint32_t parity = 0;

    for (;;) {
        const uint32_t g = sh.ticket;
        if (g >= spans) break;
        uint32_t next_ticket = 0;
        if (tid == 0) next_ticket = atomicAdd(ticket, 1u);   // its latency hides behind this span

        const uint32_t ts = g * m;
        const uint32_t mt = min(m, T - ts);
        // lanes 0..mt of every warp hold the span's index entries
        const uint32_t ixl = a.Ix[ts + min((uint32_t)lane, mt)];
        const uint32_t iyl = a.Iy[ts + min((uint32_t)lane, mt)];
        const uint32_t xs = __shfl_sync(kFull, ixl, 0), xe = __shfl_sync(kFull, ixl, mt);
        const uint32_t ys = __shfl_sync(kFull, iyl, 0), ye = __shfl_sync(kFull, iyl, mt);
        const uint32_t nxy = (xe - xs) + (ye - ys);
        const bool fits = nxy + min(nxy, (uint32_t)kTile * mt) + 8u <= kPoolWords;   // uniform over the CTA

        if (fits) {
            // ---- one sweep: walk, Phase 2, flush ---------------------------------------------------------
            const WalkOut r = span_walk<true>(a, pool, sh, ts, m, mt, xs, xe, ys, ye, bar, parity, tid);
            uint32_t before = 0, surv_total = 0;
#pragma unroll
            for (int w = 0; w < kMergeWarps; ++w) {
                const uint32_t v = sh.ws[w];
                if (w < warp) before += v;
                surv_total += v;
            }
            if (warp == 0) {
                const uint32_t wpt = (uint32_t)kMergeWarps / m;   // a tile is covered by 8/m consecutive warps
                uint32_t tc = 0;
                if ((uint32_t)lane < mt)
                    for (uint32_t w = 0; w < wpt; ++w) tc += sh.ws[lane * wpt + w];
                const uint32_t excl = span_lookback(a, g, ts, mt, tc, lane);
                if (lane == 0) sh.span_excl = excl;
            }
            if (tid == 0) sh.ticket = next_ticket;
            __syncthreads();  // #3: the span's offset in Ao is known
            span_flush(a.Ao, pool, r, sh.span_excl, surv_total, before + r.sk - r.k, tid);
            __syncthreads();  // #4: the pool may be reused
        } else {
            // ---- the span does not fit: tile by tile (one tile always fits), two sweeps -----------------
            // Sweep 1 counts the survivors of every tile so that all aggregates are published before
            // anything waits (no other CTA ever waits on a half-processed span); sweep 2 emits.
            for (uint32_t i = 0; i < mt; ++i) {
                const uint32_t x0 = __shfl_sync(kFull, ixl, i), x1 = __shfl_sync(kFull, ixl, i + 1);
                const uint32_t y0 = __shfl_sync(kFull, iyl, i), y1 = __shfl_sync(kFull, iyl, i + 1);
                span_walk<false>(a, pool, sh, ts + i, 1u, 1u, x0, x1, y0, y1, bar, parity, tid);
                if (tid == 0) {
                    uint32_t c = 0;
                    for (int w = 0; w < kMergeWarps; ++w) c += sh.ws[w];
                    sh.tc[i] = c;
                }
                __syncthreads();
            }
            if (warp == 0) {
                const uint32_t tc = (uint32_t)lane < mt ? sh.tc[lane] : 0u;
                const uint32_t excl = span_lookback(a, g, ts, mt, tc, lane);
                if (lane == 0) sh.span_excl = excl;
            }
            if (tid == 0) sh.ticket = next_ticket;
            __syncthreads();
            uint32_t off = sh.span_excl;
            for (uint32_t i = 0; i < mt; ++i) {
                const uint32_t x0 = __shfl_sync(kFull, ixl, i), x1 = __shfl_sync(kFull, ixl, i + 1);
                const uint32_t y0 = __shfl_sync(kFull, iyl, i), y1 = __shfl_sync(kFull, iyl, i + 1);
                const WalkOut r = span_walk<true>(a, pool, sh, ts + i, 1u, 1u, x0, x1, y0, y1, bar, parity, tid);
                uint32_t before = 0, surv_total = 0;
#pragma unroll
                for (int w = 0; w < kMergeWarps; ++w) {
                    const uint32_t v = sh.ws[w];
                    if (w < warp) before += v;
                    surv_total += v;
                }
                span_flush(a.Ao, pool, r, off, surv_total, before + r.sk - r.k, tid);
                off += surv_total;
                __syncthreads();
            }
        }
    }
}

cudaError_t launch_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                             const uint32_t *Iy, const void *Ay, uint64_t n, uint64_t *Bo, uint32_t *Io,
                             void *Ao, void *ws, Gate g, cudaStream_t s) {
    if (n == 0) return launch_set_u32(Io, 0u, g, s);
    const uint64_t T = (n + kTile - 1) / kTile;
    const size_t smem = (size_t)kPoolWords * sizeof(uint32_t);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(reduce_ss_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    cudaError_t e = cudaMemsetAsync(ws, 0, scan_workspace_bytes(n), s);
    if (e != cudaSuccess) return e;
    uint64_t blocks = T;   // the span length is chosen on the device; surplus CTAs find no ticket and exit
    const uint64_t cap = (uint64_t)num_sms() * kMergeMinBlocks;   // persistent: one resident wave
    if (blocks > cap) blocks = cap;
    uint32_t *ticket = reinterpret_cast<uint32_t *>(ws);
    uint64_t *status = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(ws) + kWsHeaderBytes);
    MergeArgs a;
    a.Bx = Bx; a.By = By; a.Ix = Ix; a.Iy = Iy;
    a.Ax = reinterpret_cast<const uint32_t *>(Ax); a.Ay = reinterpret_cast<const uint32_t *>(Ay);
    a.Bo = Bo; a.Io = Io; a.Ao = reinterpret_cast<uint32_t *>(Ao);
    a.status = status; a.T = (uint32_t)T;
    reduce_ss_kernel<<<(unsigned)blocks, kMergeThreads, smem, s>>>(a, ticket, g.ptr, g.value);
    return cudaGetLastError();
}

}  // namespace pici
