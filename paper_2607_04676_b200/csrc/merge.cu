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
// survivors before bit 4096*t.
//
// Structure (one persistent CTA per SM, NOT cooperative, no per-launch memset):
//   * work is handed out in BLOCKS of m consecutive tiles (m = 32 ... 1, the same for the whole launch,
//     chosen on the device from Ix[T] + Iy[T]) by a dynamic ticket; a block whose data does not fit the
//     CTA's shared-memory rings is cut into sub-spans of whole tiles (one tile always fits), so there is
//     no separate slow path: every sub-span is an ordinary item of the pipeline;
//   * the PRODUCER warp takes tickets two blocks ahead, loads the blocks' index entries one block ahead,
//     allocates an item's input bytes (its Bx / By words - contiguous - and its X / Y value runs -
//     contiguous in Ax / Ay) in the INPUT ring and its worst-case output words in the OUTPUT ring, and
//     starts the four 1-D TMA bulk copies on the item's `full` mbarrier;
//   * 16 WORKER warps, each on its own: an item is cut into pieces of 32 * LB bits (LB = bits per lane,
//     128 ... 8 with the density), piece p of the item goes to worker (base + p) mod 16.  A worker finds
//     its x / y cursors by itself - I[t] of its tile plus the popcount of the tile's words before its
//     piece (two REDUX) plus a warp scan of its own lanes - walks the set bits of x | y (add, re-test,
//     pack into the tile's region of the output ring at the candidate prefix), writes its piece of Bo and
//     leaves (start, survivors) of the piece in the item's descriptor.  No block-wide barrier or scan
//     exists; a worker never waits for a look-back;
//   * 4 FLUSHER warps (blocks are dealt to them round-robin): once an item's 16 workers have arrived on
//     `done`, the flusher publishes the item's per-tile survivor counts, takes the exclusive prefix of
//     the item's first tile (Phase 2, below), writes the item's index entries and copies
//     the pieces' survivors from the output ring to Ao, then releases the output words (`flushed`).
//     The input bytes are released as soon as the workers are done;
//   * Phase 2, the device-wide exclusive scan of the tile counts, is a three-level STORE-ONLY hierarchy
//     over tiles: one word per tile, one per group of 32 tiles, one per 1024 tiles, each (tag | value)
//     in one 64-bit word where tag = launch epoch.  prefix(t0) = [1024-blocks below] + [groups below in
//     the own block] + [tiles below in the own group]: independent loads, no chain of look-backs.  The
//     flusher whose item ends a group has just read the group's other tiles for its own prefix, so it
//     stores the group word for free (likewise the 1024-block word).  A prefix only ever waits for
//     COUNTS of earlier tiles, which are published before their owners wait for anything, and earlier
//     tiles belong to tickets taken earlier, i.e. to running CTAs: forward progress needs no
//     co-residency;
//   * the epoch lives in the workspace header and is advanced by the last flusher warp of the launch to
//     finish, which also resets the ticket: stale words of earlier launches never match the tag, so
//     nothing has to be cleared between launches (the workspace must have been zeroed ONCE,
//     pici_workspace_init).
#include <atomic>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

#ifndef PICI_MERGE_CTAS
#define PICI_MERGE_CTAS 1
#endif
constexpr int kCtasPerSm = PICI_MERGE_CTAS;
constexpr int kWorkers = 16 / kCtasPerSm;                    // worker warps per CTA
#ifndef PICI_MERGE_FLUSHERS
#define PICI_MERGE_FLUSHERS 4
#endif
constexpr int kFlushers = PICI_MERGE_FLUSHERS / kCtasPerSm;  // flusher warps per CTA
constexpr int kMergeThreads = 32 * (kWorkers + 3 + kFlushers);   // + the planner, the issuer and the publisher warp
constexpr int kDesc = 8;                                     // items in flight per CTA
constexpr uint32_t kTileWords = 2 * kSide;                   // u32 words of B per tile
constexpr uint32_t kMaxBlockTiles = 32;                      // m <= 32: one producer / flusher lane per tile
constexpr uint32_t kEnd = 0xFFFFFFFFu;
// One tile with every bit set in both operands: 2 x 128 words of B, 2 x 4096 values (+ window slack).
constexpr uint32_t kMaxTileIn = 2 * kTileWords + 2 * kTile + 16;
constexpr uint32_t kMaxTileOut = 2 * kTile + 4;        // candidates are bounded by |x| + |y| (cheap to prefix)
constexpr uint32_t kPoolWords = kCtasPerSm == 2 ? 26624 : 55296;   // 104 KB (two CTAs per SM) or 216 KB of dynamic shared memory
static_assert(kMaxTileIn + kMaxTileOut <= kPoolWords, "pool too small for one worst-case tile");

using MergeHeader = WsHeader;   // epoch, ticket, flusher warps that have left (pici_common.cuh)

struct ItemDesc {
    uint32_t t0;                       // first tile, kEnd = no more items
    uint32_t k;                        // tiles
    uint32_t npieces;                  // k * (128 / LB)
    uint32_t bx, by;                   // pool word of the item's Bx / By words
    uint32_t flusher;                  // which flusher warp owns the item
    uint32_t piece_base;               // pieces handed out before this item, mod kWorkers
    uint32_t tile_x[kMaxBlockTiles];   // pool word of tile i's first x value
    uint32_t tile_y[kMaxBlockTiles];
    uint32_t tile_out[kMaxBlockTiles]; // pool word of tile i's output region
    uint32_t piece_at[kMaxBlockTiles]; // workers: pool word of the piece's survivors, and how many
    uint32_t piece_cnt[kMaxBlockTiles];
};

struct alignas(16) IndexSlot {  // index entries of one block, copied ahead by the producer (cp.async)
    uint32_t ix[36], iy[36];                   // Ix[ts + i], Iy[ts + i], i = 0 .. tiles of the block (inclusive)
    uint32_t g;                                // the block
};

constexpr int kPlans = 4;      // planner -> issuer FIFO
constexpr int kIndexSlots = 8; // index entries stay until the issuer has used them (lead 3 + kPlans behind)
struct Plan {                  // one item, everything the issuer needs besides the index entries
    uint32_t islot;            // IndexSlot of the item's block
    uint32_t i0, i1;           // tiles [i0, i1) of the block
    uint32_t ts;               // first tile of the block, kEnd = no more items
    uint32_t xs, ys, nx, ny;   // first value / number of values of x and y
    uint32_t in_words, out_words;
    uint32_t flusher;
};

struct MergeShared {
    uint64_t full[kDesc];      // mbarrier: the item's copies have landed, its descriptor is valid
    uint64_t done[kDesc];      // mbarrier: all workers are through with the item
    uint64_t flushed[kDesc];   // mbarrier: all flushers are through with the item
    ItemDesc desc[kDesc];
    IndexSlot idx[kIndexSlots];
    uint64_t plan_full[kPlans], plan_free[kPlans];   // mbarriers of the plan FIFO
    Plan plan[kPlans];
};

struct MergeArgs {
    const uint64_t *Bx, *By;
    const uint32_t *Ix, *Iy, *Ax, *Ay;
    uint64_t *Bo;
    uint32_t *Io, *Ao;
    MergeHeader *hdr;
    uint64_t *blk_acc;     // [kWsBlkWords]  (tiles << 48) + survivors per 1024 tiles; zero between launches
    uint64_t *grp_acc;     // [kWsGrpWords]  (tiles << 48) + survivors per 32 tiles;   zero between launches
    uint64_t *tile_word;   // [T]            (tag << 32) | survivors of the tile
    uint64_t tile_words;   // tagged words behind the accumulators (cleared when the epoch wraps)
    uint32_t T;
    uint32_t zero;         // 0, but only the host knows: keeps the ticket's address non-uniform for ptxas, which
                           // otherwise makes the atomic warp-aggregated - with a shuffle that waits for its result
    uint64_t a_limit;      // bytes of Ax / Ay that may be read: (n * 4) & ~15 (capacity >= n elements)
    Gate gate;
};

__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0u;
}
// Wait with back-off: for the producer and the flushers, whose waits are long and must not take issue slots from
// the workers (a bare try_wait loop re-issues every few cycles).
__device__ __forceinline__ bool mbar_peek(uint32_t bar, uint32_t parity) {   // non-blocking
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mbar_wait_idle(uint32_t bar, uint32_t parity) {
    unsigned ns = 32;
    while (!mbar_peek(bar, parity)) {
        __nanosleep(ns);
        if (ns < 256) ns += ns;
    }
}
__device__ __forceinline__ void ticket_if(bool take, uint32_t *ticket, uint32_t &t) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.u32 p, %1, 0;\n\t"
        "@p atom.global.add.u32 %0, [%2], 1;\n\t}"
        : "+r"(t) : "r"((uint32_t)take), "l"(ticket) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void cp_async_4(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
// 16-byte copy of which only the first src_bytes are read (the rest is zero-filled)
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void *src, uint32_t src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ uint32_t popc4(uint4 v) { return __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }

// ---- value windows ------------------------------------------------------------------------------
// The values A[beg .. beg+cnt) are copied as ONE bulk copy of the 16-byte aligned window around them
// (up to 12 bytes before and after belong to neighbouring items of the same buffer; the window never
// passes a_limit, so nothing outside the caller's capacity is read).  Only a run that ends in the last
// < 16 bytes of a completely full buffer keeps a tail, moved by plain loads.
struct Window {
    uint64_t g_beg;    // byte offset in A of the window start
    uint32_t bulk;     // bytes of the bulk copy (multiple of 16, may be 0)
    uint32_t words;    // window length in words, multiple of 4 (what the ring reserves)
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

// ---- launch-wide geometry, computed identically by every thread ---------------------------------------
struct Geometry {
    uint32_t m;          // tiles per block
    uint32_t lb;         // bits per lane of a piece: 128, 64, 32, 16 or 8
    uint32_t slot_in, n_in;     // input slots: words per slot, how many (item j uses slot j mod n_in)
    uint32_t slot_out, n_out;   // output slots, behind the input slots
    uint32_t out_base;          // first word of the output slots
    uint32_t blocks;
};
// An average block plus 1/8 and a little must fit a slot; at least 4 input and 6 output slots for the block length
// to be taken (output words live two to three times as long as input words: publish + prefix + flush against load
// + merge), then as many slots as the pool holds, up to kDesc each.
__device__ __forceinline__ Geometry geometry(const MergeArgs &a, uint32_t G) {
    Geometry g;
    const uint32_t T = a.T;
    const uint64_t nx = __ldg(a.Ix + T), ny = __ldg(a.Iy + T);
    const uint64_t avg = (nx + ny + T - 1) / T;                     // values per tile, X and Y together
    const uint64_t in_tile = 2 * kTileWords + avg + 8;
    const uint64_t out_tile = avg + 4;
    auto slot_of = [](uint64_t words, uint32_t floor_words) -> uint32_t {
        const uint64_t v = words + words / 8 + 32;
        return (uint32_t)((max(v, (uint64_t)floor_words) + 3) & ~3ull);
    };
    constexpr uint32_t kFloorIn = 512, kFloorOut = 256;
    uint32_t m = 1;
#pragma unroll
    for (uint32_t mm = kMaxBlockTiles; mm >= 2; mm /= 2)
        if (m == 1 && 4ull * slot_of(mm * in_tile, kFloorIn) + 6ull * slot_of(mm * out_tile, kFloorOut) <= kPoolWords) m = mm;
    while (m > 1 && (T + m - 1) / m < 2u * G) m /= 2;               // small inputs: keep every CTA busy
    uint32_t si = slot_of(m * in_tile, kFloorIn), so = slot_of(m * out_tile, kFloorOut);
    uint32_t ni = 1, no = 1;
    for (;;) {   // output slots first (about two per input slot: their words live longer), up to kDesc of each
        if (no < kDesc && no < 2u * ni + 2u && (uint64_t)ni * si + (uint64_t)(no + 1u) * so <= kPoolWords) ++no;
        else if (ni < kDesc && (uint64_t)(ni + 1u) * si + (uint64_t)no * so <= kPoolWords) ++ni;
        else if (no < kDesc && (uint64_t)ni * si + (uint64_t)(no + 1u) * so <= kPoolWords) ++no;
        else break;
    }
    g.m = m;
    g.lb = min(16u * m, 128u);
    g.slot_in = si; g.n_in = ni; g.slot_out = so; g.n_out = no;
    g.out_base = ni * si;
    g.blocks = (T + m - 1) / m;
    return g;
}

// =========================================== producer ===========================================
// The producer is two warps, because one warp's instruction latency per item (about 1.3 us) was what bounded the
// whole kernel: the PLANNER takes tickets, fetches index entries and cuts blocks into items (plans); the ISSUER
// waits for the item's slots, fills the descriptor and starts the copies.
__device__ __forceinline__ void planner(const MergeArgs &a, MergeShared &sh, const Geometry &geo, uint32_t tk0, int lane) {
    const uint32_t T = a.T, m = geo.m;
    const uint32_t pfull0 = smem_u32(&sh.plan_full[0]), pfree0 = smem_u32(&sh.plan_free[0]);
    const uint32_t in_limit = geo.slot_in, out_limit = geo.slot_out;
    uint32_t j = 0;                 // items planned
    uint32_t blk_seq = 0;
    // ---- block pipeline --------------------------------------------------------------------------------------
    // A ticket costs an L2 round trip and so does a block's index entries, each about as long as the CTA has for a
    // whole block in the sparse regime, so both run well ahead of the block in hand (n): tickets are requested
    // five blocks ahead (two atomics in flight, all by lane 0, hence increasing), index entries are copied to
    // shared memory by cp.async three blocks ahead (slot n mod kIndexSlots).
    const bool wide = m >= 4u && ((reinterpret_cast<uintptr_t>(a.Ix) | reinterpret_cast<uintptr_t>(a.Iy)) & 15u) == 0u;
    auto issue_index = [&](uint32_t slot, uint32_t g) {
        IndexSlot &S = sh.idx[slot];
        if (g < geo.blocks) {
            const uint32_t ts = g * m;
            if (wide) {          // ts * 4 bytes is 16-byte aligned: entries ts + 4c .. ts + 4c + 3 as one 16-byte copy
                const uint32_t e0 = ts + 4u * (uint32_t)lane;          // lanes 0 .. m/4 (the last one: the end entry)
                if (4u * (uint32_t)lane <= m && e0 <= T) {
                    const uint32_t bytes = min(4u, T + 1u - e0) * 4u;  // never read past I[T]
                    cp_async_16(smem_u32(&S.ix[4 * lane]), a.Ix + e0, bytes);
                    cp_async_16(smem_u32(&S.iy[4 * lane]), a.Iy + e0, bytes);
                }
            } else if ((uint32_t)lane <= m && ts + (uint32_t)lane <= T) {
                cp_async_4(smem_u32(&S.ix[lane]), a.Ix + ts + lane);
                cp_async_4(smem_u32(&S.iy[lane]), a.Iy + ts + lane);
            }
        }
        if (lane == 0) S.g = g;
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    uint32_t n = 0;                 // block in hand (counted per CTA)
    bool dry = false;               // a ticket beyond the last block has been seen: request no more
    // Start-up: every ticket is requested only after the one before it has returned, so the CTAs' first tickets
    // interleave (CTA c holds blocks ~c, ~G + c, ~2G + c, ...) instead of forming runs of consecutive blocks - a
    // CTA that holds a run and cannot allocate its last block yet would hold up everyone behind it.
    // How far ahead: blocks of a few dense tiles last long enough for one block of lead; in the sparse regime a
    // block lasts about one memory round trip and the lead is three.  (More lead than needed means tickets held
    // long before their tiles are merged, i.e. more skew between CTAs and longer waits for prefixes.)
    const uint32_t lead = m <= 4u ? 1u : 3u;
    uint32_t tkA = kEnd, tkB = kEnd;  // in flight: tickets of blocks n + lead (A on even n, B on odd n) and n + lead + 1
    if (lead == 3u) {
        auto next = [&](uint32_t prev) -> uint32_t {
            uint32_t t = kEnd;
            if (prev < geo.blocks && lane == 0) t = atomicAdd(&a.hdr->ticket, 1u);
            return __shfl_sync(kFull, t, 0);
        };
        const uint32_t g0 = __shfl_sync(kFull, tk0, 0);
        issue_index(0, g0);
        const uint32_t g1 = next(g0);
        issue_index(1, g1);
        const uint32_t g2 = next(g1);
        issue_index(2, g2);
        tkA = next(g2);
        dry = tkA >= geo.blocks;
        if (!dry && lane == 0) tkB = atomicAdd(&a.hdr->ticket, 1u);
    } else {
        const uint32_t g0 = __shfl_sync(kFull, tk0, 0);
        issue_index(0, g0);
        dry = g0 >= geo.blocks;
        ticket_if(!dry && lane == 0, &a.hdr->ticket + (uint32_t)lane * a.zero, tkA);
    }
    // one block; tk is the register (tkA on even n, tkB on odd n: the loop is unrolled by two so that reading one
    // in-flight ticket never waits for the other)
    auto step = [&](uint32_t &tk) -> bool {
        // the ticket of block n + 3 has had two blocks' time to return; its index entries start moving now
        const uint32_t g3 = __shfl_sync(kFull, tk, 0);
        if (g3 >= geo.blocks) dry = true;
        // block n + 5's ticket; a predicated atomic, so that nothing reads the register before it is needed two
        // blocks from now (a select between the atomic's result and kEnd would wait for the round trip here)
        tk = kEnd;
        ticket_if(!dry && lane == 0, &a.hdr->ticket + (uint32_t)lane * a.zero, tk);
        issue_index((n + lead) & (kIndexSlots - 1), g3);
        if (lead == 3u) asm volatile("cp.async.wait_group 3;" ::: "memory");   // block n's entries have landed
        else asm volatile("cp.async.wait_group 1;" ::: "memory");
        const IndexSlot &S = sh.idx[n & (kIndexSlots - 1)];
        __syncwarp();
        const uint32_t g_cur = S.g;
        if (g_cur >= geo.blocks) return false;
        const uint32_t ts = g_cur * m, mt = min(m, T - ts);
        const uint32_t l1 = min((uint32_t)lane + 1u, mt);
        const uint32_t cx1 = S.ix[l1], cy1 = S.iy[l1];
        ++n;
        {
        uint32_t i0 = 0;
        while (i0 < mt) {
            // ---- the longest run of tiles [i0, i1) whose data fits half of each ring; a tile's output region
            // holds |x| + |y| words (its candidates cannot be more) ------------------------------------------------
            const uint32_t xs = S.ix[i0], ys = S.iy[i0];
            const uint32_t vals = (cx1 - xs) + (cy1 - ys);          // values of tiles i0 .. lane
            const uint32_t need_in = 2u * kTileWords * ((uint32_t)lane - i0 + 1u) + vals + 16u;
            const bool in_range = (uint32_t)lane >= i0 && (uint32_t)lane < mt;
            const bool fits = need_in <= in_limit && vals + 4u <= out_limit;
            const unsigned bad = __ballot_sync(kFull, in_range && !fits);
            uint32_t i1 = bad ? (uint32_t)__ffs(bad) - 1u : mt;
            if (i1 <= i0) i1 = i0 + 1;                      // a tile that fits no slot goes alone, across the slots
            const uint32_t xe = S.ix[i1], ye = S.iy[i1];
            const uint32_t nx = xe - xs, ny = ye - ys;
            // ---- the plan ---------------------------------------------------------------------------------------
            const uint32_t q = j % kPlans;
            if (j >= (uint32_t)kPlans) mbar_wait_idle(pfree0 + 8 * q, ((j / kPlans) - 1u) & 1u);
            if (lane == 0) {
                Plan &P = sh.plan[q];
                P.islot = (n - 1u) & (kIndexSlots - 1);
                P.i0 = i0; P.i1 = i1; P.ts = ts;
                P.xs = xs; P.ys = ys; P.nx = nx; P.ny = ny;
                P.flusher = blk_seq % kFlushers;
                mbar_arrive(pfull0 + 8 * q);
            }
            ++j;
            i0 = i1;
        }
        }
        ++blk_seq;
        return true;
    };
    if (lead == 3u) {
        while (step(tkA) && step(tkB)) {
        }
    } else {
        while (step(tkA)) {
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    // every ticket this warp requested must have returned before the CTA's last item is emitted (the launch's last
    // flusher resets the ticket): both registers are read here
    if (lane == 0 && (tkA & tkB) == 0x12345678u) sh.idx[0].g = 0;    // never true: tickets are < 2^31 or kEnd
    const uint32_t q = j % kPlans;
    if (j >= (uint32_t)kPlans) mbar_wait_idle(pfree0 + 8 * q, ((j / kPlans) - 1u) & 1u);
    if (lane == 0) {
        sh.plan[q].ts = kEnd;
        mbar_arrive(pfull0 + 8 * q);
    }
}

__device__ __forceinline__ void issuer(const MergeArgs &a, MergeShared &sh, uint32_t *pool, const Geometry &geo, int lane) {
    const uint32_t ppt = 128u / geo.lb;
    const uint32_t full0 = smem_u32(&sh.full[0]), done0 = smem_u32(&sh.done[0]), fl0 = smem_u32(&sh.flushed[0]);
    const uint32_t pfull0 = smem_u32(&sh.plan_full[0]), pfree0 = smem_u32(&sh.plan_free[0]);
    uint32_t j = 0;                 // items emitted
    uint32_t s_in = 0, s_out = 0;   // j mod n_in, j mod n_out
    bool prev_big = false;          // item j - 1 did not fit a slot (it lies across the pool, see below)
    uint32_t piece_base = 0;
    // the workers / all flushers and the publisher are through with item i (i < j)
    auto wait_done = [&](uint32_t i) { mbar_wait_idle(done0 + 8 * (i % kDesc), (i / kDesc) & 1u); };
    auto wait_flushed = [&](uint32_t i) { mbar_wait_idle(fl0 + 8 * (i % kDesc), (i / kDesc) & 1u); };
    for (;; ++j) {
        const uint32_t q = j % kPlans;
        mbar_wait(pfull0 + 8 * q, (j / kPlans) & 1u);
        const Plan &P = sh.plan[q];
        const uint32_t ts = P.ts;
        if (ts == kEnd) break;
        const uint32_t i0 = P.i0, i1 = P.i1, k = i1 - i0;
        const uint32_t xs = P.xs, ys = P.ys, nx = P.nx, ny = P.ny, flusher = P.flusher;
        const IndexSlot &S = sh.idx[P.islot];
        const uint32_t li = min(i0 + (uint32_t)lane, i1);
        const uint32_t cx0 = S.ix[li], cy0 = S.iy[li];            // lane i < k: tile i0 + i of the block
        const Window wx = window_of(xs, nx, a.a_limit), wy = window_of(ys, ny, a.a_limit);
        const uint32_t in_words = 2u * kTileWords * k + wx.words + wy.words;
        const uint32_t out_words = max((nx + ny + 3u) & ~3u, 4u);
        // ---- descriptor slot, input slot, output slot ------------------------------------------------------
        // Item j lives in descriptor j mod kDesc, input slot j mod n_in, output slot j mod n_out: it may start once
        // the items that had them before are through.  An item that does not fit a slot (a tile much denser than
        // the launch's average) is laid across the pool from word 0, alone (one worst-case tile always fits):
        // everything before it has drained, and the item behind it waits for it.
        const uint32_t d = j % kDesc;
        const bool big = in_words > geo.slot_in || out_words > geo.slot_out;
        if (big || prev_big) {
            for (uint32_t r = 1; r <= min(j, (uint32_t)kDesc); ++r) wait_flushed(j - r);
        } else {
            if (j >= geo.n_in) wait_done(j - geo.n_in);
            if (j >= geo.n_out) wait_flushed(j - geo.n_out);
            if (j >= (uint32_t)kDesc) wait_flushed(j - kDesc);
        }
        prev_big = big;
        const uint32_t ib = big ? 0u : s_in * geo.slot_in;   // alone in the pool: inputs from word 0, outputs behind
        const uint32_t ob = big ? in_words : geo.out_base + s_out * geo.slot_out;
        s_in = s_in + 1u == geo.n_in ? 0u : s_in + 1u;
        s_out = s_out + 1u == geo.n_out ? 0u : s_out + 1u;
        ItemDesc &D = sh.desc[d];
        const uint32_t V = ib + 2u * kTileWords * k;
        const uint32_t Xb = V + wx.first, Yb = V + wx.words + wy.first;
        if ((uint32_t)lane < k) {
            D.tile_x[lane] = Xb + (cx0 - xs);
            D.tile_y[lane] = Yb + (cy0 - ys);
            D.tile_out[lane] = ob + (cx0 - xs) + (cy0 - ys);
        }
        if (lane == 0) {
            D.t0 = ts + i0;
            D.k = k;
            D.npieces = k * ppt;
            D.bx = ib;
            D.by = ib + kTileWords * k;
            D.flusher = flusher;
            D.piece_base = piece_base;
        }
        // tail elements (plain stores, < 4 per operand) before lane 0's arrive, which releases them
        if (wx.tail_beg + lane < nx) pool[Xb + wx.tail_beg + lane] = a.Ax[xs + wx.tail_beg + lane];
        if (wy.tail_beg + lane < ny) pool[Yb + wy.tail_beg + lane] = a.Ay[ys + wy.tail_beg + lane];
        __syncwarp();
        {
            // the four bulk copies (Bx words, By words, X values, Y values) leave as ONE instruction: lane c issues
            // copy c
            const uint32_t bar = full0 + 8 * d;
            const uint32_t bbytes = k * kTileWords * 4u;
            if (lane == 0) {
                mbar_arrive(pfree0 + 8 * q);                  // the plan and its index entries have been read
                mbar_expect_tx(bar, 2u * bbytes + wx.bulk + wy.bulk);
            }
            __syncwarp();
            const unsigned char *src = nullptr;
            uint32_t dstw = 0, bytes = 0;
            if (lane == 0) { src = reinterpret_cast<const unsigned char *>(a.Bx + (size_t)(ts + i0) * kSide); dstw = ib; bytes = bbytes; }
            else if (lane == 1) { src = reinterpret_cast<const unsigned char *>(a.By + (size_t)(ts + i0) * kSide); dstw = ib + kTileWords * k; bytes = bbytes; }
            else if (lane == 2) { src = reinterpret_cast<const unsigned char *>(a.Ax) + wx.g_beg; dstw = V; bytes = wx.bulk; }
            else if (lane == 3) { src = reinterpret_cast<const unsigned char *>(a.Ay) + wy.g_beg; dstw = V + wx.words; bytes = wy.bulk; }
            if (bytes) bulk_g2s(smem_u32(pool + dstw), src, bytes, bar);
        }
        piece_base = (piece_base + k * ppt) % kWorkers;
    }
    const uint32_t d = j % kDesc;
    if (j >= (uint32_t)kDesc) wait_flushed(j - kDesc);
    if (lane == 0) {
        sh.desc[d].t0 = kEnd;
        mbar_arrive(full0 + 8 * d);
    }
}

// Two independent chains of the walk over the set bits of (wxA | wyA) and of (wxB | wyB): per candidate add
// (received + local, C9 #7), re-test, store.  Cursors are shared-memory BYTE addresses.  Chain B's output cursor
// starts at the CANDIDATE count of chain A, so the lane's survivors are contiguous only if nothing cancelled; the
// caller checks survivors == candidates and redoes the piece with walk_packed otherwise.  A chain whose bits run
// out idles (bit = 0: nothing loaded, sum = +0, nothing stored).  Hand-scheduled: 17 instructions per chain step.
__device__ __forceinline__ void walk2(uint32_t wxA, uint32_t wyA, uint32_t wxB, uint32_t wyB, uint32_t &xaA, uint32_t &yaA,
                                      uint32_t &oaA, uint32_t &xaB, uint32_t &yaB, uint32_t &oaB, uint32_t &oA,
                                      uint32_t &oB) {
    uint32_t uA = wxA | wyA, uB = wxB | wyB;
    asm volatile(
        "{\n\t"
        ".reg .pred pxA, pyA, psA, pxB, pyB, psB, pl;\n\t"
        ".reg .b32 bA, bB, t, vxA, vyA, vxB, vyB, sA, sB;\n\t"
        "or.b32 t, %0, %1;\n\t"
        "setp.eq.u32 pl, t, 0;\n\t"
        "@pl bra DONE_%=;\n\t"
        "LOOP_%=:\n\t"
        "neg.s32 bA, %0;\n\t"
        "neg.s32 bB, %1;\n\t"
        "and.b32 bA, bA, %0;\n\t"
        "and.b32 bB, bB, %1;\n\t"
        "xor.b32 %0, %0, bA;\n\t"
        "xor.b32 %1, %1, bB;\n\t"
        "and.b32 t, %10, bA;\n\t"
        "setp.ne.u32 pxA, t, 0;\n\t"
        "and.b32 t, %11, bA;\n\t"
        "setp.ne.u32 pyA, t, 0;\n\t"
        "and.b32 t, %12, bB;\n\t"
        "setp.ne.u32 pxB, t, 0;\n\t"
        "and.b32 t, %13, bB;\n\t"
        "setp.ne.u32 pyB, t, 0;\n\t"
        "mov.b32 vxA, 0;\n\t"
        "mov.b32 vyA, 0;\n\t"
        "mov.b32 vxB, 0;\n\t"
        "mov.b32 vyB, 0;\n\t"
        "@pxA ld.shared.b32 vxA, [%2];\n\t"
        "@pyA ld.shared.b32 vyA, [%3];\n\t"
        "@pxB ld.shared.b32 vxB, [%5];\n\t"
        "@pyB ld.shared.b32 vyB, [%6];\n\t"
        "@pxA add.u32 %2, %2, 4;\n\t"
        "@pyA add.u32 %3, %3, 4;\n\t"
        "@pxB add.u32 %5, %5, 4;\n\t"
        "@pyB add.u32 %6, %6, 4;\n\t"
        "add.rn.f32 sA, vxA, vyA;\n\t"
        "add.rn.f32 sB, vxB, vyB;\n\t"
        "and.b32 t, sA, 0x7fffffff;\n\t"
        "setp.ne.u32 psA, t, 0;\n\t"
        "and.b32 t, sB, 0x7fffffff;\n\t"
        "setp.ne.u32 psB, t, 0;\n\t"
        "@psA st.shared.b32 [%4], sA;\n\t"
        "@psB st.shared.b32 [%7], sB;\n\t"
        "@psA add.u32 %4, %4, 4;\n\t"
        "@psB add.u32 %7, %7, 4;\n\t"
        "@psA or.b32 %8, %8, bA;\n\t"
        "@psB or.b32 %9, %9, bB;\n\t"
        "or.b32 t, %0, %1;\n\t"
        "setp.ne.u32 pl, t, 0;\n\t"
        "@pl bra LOOP_%=;\n\t"
        "DONE_%=:\n\t"
        "}"
        : "+r"(uA), "+r"(uB), "+r"(xaA), "+r"(yaA), "+r"(oaA), "+r"(xaB), "+r"(yaB), "+r"(oaB), "+r"(oA), "+r"(oB)
        : "r"(wxA), "r"(wyA), "r"(wxB), "r"(wyB)
        : "memory");
}

// ============================================ workers ============================================
// One piece (32 * LB bits) of tile i of the item: cursors, walk, Bo, (start, survivors) of the piece.
template <int LB>
__device__ __forceinline__ void do_piece(const MergeArgs &a, uint32_t *pool, ItemDesc &D, uint32_t p, int lane) {
    constexpr uint32_t PPT = 128 / LB;                       // pieces per tile
    constexpr int NW = LB >= 32 ? LB / 32 : 1;               // 32-bit words per lane
    const uint32_t i = p / PPT, sub = p % PPT;
    const uint32_t *bx = pool + D.bx + i * kTileWords, *by = pool + D.by + i * kTileWords;
    uint32_t kx = D.tile_x[i], ky = D.tile_y[i], ko = D.tile_out[i];
    uint32_t ax[NW], ay[NW];
    const uint32_t s0 = sub * LB;                            // first word of the piece inside the tile
    if constexpr (LB == 128) {
        const uint4 X = reinterpret_cast<const uint4 *>(bx)[lane], Y = reinterpret_cast<const uint4 *>(by)[lane];
        ax[0] = X.x; ax[1] = X.y; ax[2] = X.z; ax[3] = X.w;
        ay[0] = Y.x; ay[1] = Y.y; ay[2] = Y.z; ay[3] = Y.w;
    } else {
        if (sub != 0) {   // values / candidates of the tile before this piece
            const uint4 X = reinterpret_cast<const uint4 *>(bx)[lane], Y = reinterpret_cast<const uint4 *>(by)[lane];
            uint32_t pxy = 0, pu = 0;
            if (4u * (uint32_t)lane < s0) {
                pxy = popc4(X) | (popc4(Y) << 16);
                pu = popc4(make_uint4(X.x | Y.x, X.y | Y.y, X.z | Y.z, X.w | Y.w));
            }
            pxy = __reduce_add_sync(kFull, pxy);
            pu = __reduce_add_sync(kFull, pu);
            kx += pxy & 0xFFFFu;
            ky += pxy >> 16;
            ko += pu;
        }
        if constexpr (LB == 64) {
            const uint2 X = reinterpret_cast<const uint2 *>(bx + s0)[lane], Y = reinterpret_cast<const uint2 *>(by + s0)[lane];
            ax[0] = X.x; ax[1] = X.y;
            ay[0] = Y.x; ay[1] = Y.y;
        } else if constexpr (LB == 32) {
            ax[0] = bx[s0 + lane];
            ay[0] = by[s0 + lane];
        } else if constexpr (LB == 16) {
            ax[0] = reinterpret_cast<const uint16_t *>(bx + s0)[lane];
            ay[0] = reinterpret_cast<const uint16_t *>(by + s0)[lane];
        } else {
            ax[0] = reinterpret_cast<const uint8_t *>(bx + s0)[lane];
            ay[0] = reinterpret_cast<const uint8_t *>(by + s0)[lane];
        }
    }
    uint32_t cx = 0, cy = 0, cu = 0;
#pragma unroll
    for (int q = 0; q < NW; ++q) {
        cx += __popc(ax[q]);
        cy += __popc(ay[q]);
        cu += __popc(ax[q] | ay[q]);
    }
    uint32_t ao[NW];
    uint32_t ktot = 0;
    const uint32_t piece_at = ko;
    if (__any_sync(kFull, cu != 0u)) {
        uint32_t ex, ey, eu;                                 // exclusive prefixes over the lanes
        if constexpr (LB <= 16) {                            // totals <= 512: one packed scan
            const uint32_t v = cx | (cy << 10) | (cu << 20);
            const uint32_t s = warp_incl_scan(v, lane) - v;
            ex = s & 1023u; ey = (s >> 10) & 1023u; eu = s >> 20;
        } else {
            const uint32_t v = cx | (cy << 16);
            const uint32_t s = warp_incl_scan(v, lane) - v;
            ex = s & 0xFFFFu; ey = s >> 16;
            eu = warp_incl_scan(cu, lane) - cu;
        }
        kx += ex;
        ky += ey;
        const uint32_t ko0 = ko + eu;
        // ---- fast walk: two chains per lane (the halves of a word, or two words) -----------------------------
        const uint32_t sbase = smem_u32(pool);
        uint32_t xa = sbase + 4u * kx, ya = sbase + 4u * ky, oa = sbase + 4u * ko0;
        uint32_t surv = 0;
        if constexpr (NW == 1) {
            constexpr uint32_t kLo = (1u << (LB >= 32 ? 16 : LB / 2)) - 1u;
            const uint32_t xlo = ax[0] & kLo, ylo = ay[0] & kLo, xhi = ax[0] & ~kLo, yhi = ay[0] & ~kLo;
            uint32_t xb = xa + 4u * __popc(xlo), yb = ya + 4u * __popc(ylo), ob = oa + 4u * __popc(xlo | ylo);
            const uint32_t oa0 = oa, ob0 = ob;
            uint32_t oA = 0, oB = 0;
            walk2(xlo, ylo, xhi, yhi, xa, ya, oa, xb, yb, ob, oA, oB);
            ao[0] = oA | oB;
            surv = ((oa - oa0) + (ob - ob0)) >> 2;
        } else {
#pragma unroll
            for (int q = 0; q < NW; q += 2) {
                uint32_t xb = xa + 4u * __popc(ax[q]), yb = ya + 4u * __popc(ay[q]), ob = oa + 4u * __popc(ax[q] | ay[q]);
                const uint32_t oa0 = oa, ob0 = ob;
                uint32_t oA = 0, oB = 0;
                walk2(ax[q], ay[q], ax[q + 1], ay[q + 1], xa, ya, oa, xb, yb, ob, oA, oB);
                ao[q] = oA;
                ao[q + 1] = oB;
                surv += ((oa - oa0) + (ob - ob0)) >> 2;
                xa = xb; ya = yb; oa = ob;
            }
        }
        ktot = __reduce_add_sync(kFull, surv);
        if (__any_sync(kFull, surv != cu)) {
            // ---- an exact cancellation: redo the piece with one packed run per lane, then close the gaps
            // between the lanes' runs, lane by lane (dst <= src) ------------------------------------------------
            __syncwarp();
            const uint32_t *__restrict__ xp = pool + kx;
            const uint32_t *__restrict__ yp = pool + ky;
            uint32_t *__restrict__ op = pool + ko0;
#pragma unroll
            for (int q = 0; q < NW; ++q) {
                uint32_t u = ax[q] | ay[q], o = 0;
                const uint32_t wx = ax[q], wy = ay[q];
                while (u) {
                    const uint32_t bit = u & (0u - u);
                    u ^= bit;
                    const bool hx = (wx & bit) != 0u, hy = (wy & bit) != 0u;
                    const float x = hx ? __uint_as_float(*xp) : 0.0f;
                    const float y = hy ? __uint_as_float(*yp) : 0.0f;
                    xp += hx ? 1 : 0;
                    yp += hy ? 1 : 0;
                    const uint32_t sum = __float_as_uint(__fadd_rn(x, y));
                    if (nz32(sum)) {
                        o |= bit;
                        *op++ = sum;
                    }
                }
                ao[q] = o;
            }
            const uint32_t kmine = (uint32_t)(op - pool) - ko0;
            const uint32_t ek = warp_incl_scan(kmine, lane) - kmine;
            __syncwarp();
            for (int l = 0; l < 32; ++l) {
                const uint32_t src = __shfl_sync(kFull, ko0, l), cnt = __shfl_sync(kFull, kmine, l);
                const uint32_t dst = ko + __shfl_sync(kFull, ek, l);
                if (src == dst) continue;
                for (uint32_t b = 0; b < cnt; b += 32) {
                    uint32_t v = 0;
                    if (b + lane < cnt) v = pool[src + b + lane];
                    __syncwarp();
                    if (b + lane < cnt) pool[dst + b + lane] = v;
                    __syncwarp();
                }
            }
        }
    } else {
#pragma unroll
        for (int q = 0; q < NW; ++q) ao[q] = 0u;
    }
    // ---- this piece of Bo ------------------------------------------------------------------------------
    uint32_t *bo = reinterpret_cast<uint32_t *>(a.Bo) + (size_t)(D.t0 + i) * kTileWords + s0;
    if constexpr (LB == 128) reinterpret_cast<uint4 *>(bo)[lane] = make_uint4(ao[0], ao[1], ao[2], ao[3]);
    else if constexpr (LB == 64) reinterpret_cast<uint2 *>(bo)[lane] = make_uint2(ao[0], ao[1]);
    else if constexpr (LB == 32) bo[lane] = ao[0];
    else if constexpr (LB == 16) reinterpret_cast<uint16_t *>(bo)[lane] = (uint16_t)ao[0];
    else reinterpret_cast<uint8_t *>(bo)[lane] = (uint8_t)ao[0];
    if (lane == 0) {
        D.piece_at[p] = piece_at;
        D.piece_cnt[p] = ktot;
    }
}

template <int LB>
__device__ __forceinline__ void worker(const MergeArgs &a, MergeShared &sh, uint32_t *pool, int w, int lane) {
    const uint32_t full0 = smem_u32(&sh.full[0]), done0 = smem_u32(&sh.done[0]);
    for (uint32_t j = 0;; ++j) {
        const uint32_t d = j % kDesc, ph = (j / kDesc) & 1u;
        mbar_wait(full0 + 8 * d, ph);
        ItemDesc &D = sh.desc[d];
        if (D.t0 == kEnd) break;
        const uint32_t np = D.npieces;
        for (uint32_t p = ((uint32_t)w + kWorkers - D.piece_base) % kWorkers; p < np; p += kWorkers)
            do_piece<LB>(a, pool, D, p, lane);
        __syncwarp();
        if (lane == 0) mbar_arrive(done0 + 8 * d);
    }
}

// ============================================ publisher ===========================================
// Phase 2 input.  One warp that does nothing but make counts visible: as soon as an item's workers are done it
// stores the item's per-tile survivor counts (tagged words) and adds (tiles, survivors) to the accumulators of
// the item's group of 32 tiles and of its block of 1024 tiles.  It waits for nothing else - in particular never
// for a prefix - so every count of the launch becomes visible a fixed latency after its tile was merged, and a
// prefix, which only reads counts, can never be part of a chain of waits.
__device__ __forceinline__ void publisher(const MergeArgs &a, MergeShared &sh, const Geometry &geo, uint32_t tag, int lane) {
    const uint32_t full0 = smem_u32(&sh.full[0]), done0 = smem_u32(&sh.done[0]), fl0 = smem_u32(&sh.flushed[0]);
    const uint32_t ppt = 128u / geo.lb;
    for (uint32_t j = 0;; ++j) {
        const uint32_t d = j % kDesc, ph = (j / kDesc) & 1u;
        mbar_wait_idle(full0 + 8 * d, ph);
        const ItemDesc &D = sh.desc[d];
        const uint32_t t0 = D.t0;
        if (t0 == kEnd) break;
        const uint32_t k = D.k, np = D.npieces;
        mbar_wait_idle(done0 + 8 * d, ph);
        const uint32_t cnt = (uint32_t)lane < np ? D.piece_cnt[lane] : 0u;
        const uint32_t incl = warp_incl_scan(cnt, lane);
        const uint32_t total = __shfl_sync(kFull, incl, 31);
        const uint32_t lo = __shfl_sync(kFull, incl - cnt, ((uint32_t)lane * ppt) & 31u);
        const uint32_t hi = __shfl_sync(kFull, incl, ((uint32_t)lane * ppt + ppt - 1u) & 31u);
        if ((uint32_t)lane < k) st_status(a.tile_word + t0 + lane, tag, hi - lo);
        if (lane == 0) {
            const uint64_t v = ((uint64_t)k << 48) + total;
            red_add_u64(a.grp_acc + (t0 >> 5), v);
            red_add_u64(a.blk_acc + (t0 >> 10), v);
            mbar_arrive(fl0 + 8 * d);
        }
    }
}

// ============================================ flushers ============================================
// (the exclusive prefix of a tile: hier_prefix, pici_common.cuh)
// One warp copies cnt words from shared memory (word index src in pool) to global memory dst (4-byte aligned, any
// 16-byte phase): a few single words up to the first 16-byte boundary of dst, then aligned 16-byte stores whose
// four words come from two aligned 16-byte shared-memory reads (the phase difference is a whole number of words,
// so realigning is a choice of registers, not a shift), then the last < 4 words.
template <int K>
__device__ __forceinline__ uint4 pick4(uint4 lo, uint4 hi) {   // words K .. K+3 of (lo.x lo.y lo.z lo.w hi.x hi.y hi.z hi.w)
    if constexpr (K == 0) return lo;
    else if constexpr (K == 1) return make_uint4(lo.y, lo.z, lo.w, hi.x);
    else if constexpr (K == 2) return make_uint4(lo.z, lo.w, hi.x, hi.y);
    else return make_uint4(lo.w, hi.x, hi.y, hi.z);
}
template <int K>
__device__ __forceinline__ void copy_body(const uint32_t *pool, uint32_t src, uint4 *dst4, uint32_t nvec, int lane) {
    const uint4 *s4 = reinterpret_cast<const uint4 *>(pool + (src - K));   // 16-byte aligned by construction
    uint32_t i = lane;
    for (; i + 32u < nvec; i += 64u) {     // two stores in flight per lane
        const uint4 a0 = s4[i], a1 = K ? s4[i + 1] : a0, b0 = s4[i + 32], b1 = K ? s4[i + 33] : b0;
        dst4[i] = pick4<K>(a0, a1);
        dst4[i + 32] = pick4<K>(b0, b1);
    }
    if (i < nvec) {
        const uint4 a0 = s4[i], a1 = K ? s4[i + 1] : a0;
        dst4[i] = pick4<K>(a0, a1);
    }
}
__device__ __forceinline__ void copy_run(const uint32_t *pool, uint32_t src, uint32_t *dst, uint32_t cnt, int lane) {
    const uint32_t head = min((uint32_t)((16u - ((uint32_t)reinterpret_cast<uintptr_t>(dst) & 15u)) & 15u) >> 2, cnt);
    if ((uint32_t)lane < head) dst[lane] = pool[src + lane];
    const uint32_t nvec = (cnt - head) >> 2, body = nvec << 2;
    const uint32_t s = src + head;
    uint4 *d4 = reinterpret_cast<uint4 *>(dst + head);
    switch (s & 3u) {
        case 0: copy_body<0>(pool, s, d4, nvec, lane); break;
        case 1: copy_body<1>(pool, s, d4, nvec, lane); break;
        case 2: copy_body<2>(pool, s, d4, nvec, lane); break;
        default: copy_body<3>(pool, s, d4, nvec, lane); break;
    }
    const uint32_t tail = cnt - head - body;
    if ((uint32_t)lane < tail) dst[head + body + lane] = pool[s + body + lane];
}

__device__ __forceinline__ void flusher(const MergeArgs &a, MergeShared &sh, const uint32_t *pool, const Geometry &geo,
                                        uint32_t tag, int f, int lane) {
    const uint32_t full0 = smem_u32(&sh.full[0]), done0 = smem_u32(&sh.done[0]), fl0 = smem_u32(&sh.flushed[0]);
    const uint32_t ppt = 128u / geo.lb;
    uint32_t E = 0, E_blk = 0;
    for (uint32_t j = 0;; ++j) {
        const uint32_t d = j % kDesc, ph = (j / kDesc) & 1u;
        mbar_wait_idle(full0 + 8 * d, ph);
        const ItemDesc &D = sh.desc[d];
        const uint32_t t0 = D.t0;
        if (t0 == kEnd) break;
        if (D.flusher == (uint32_t)f) {
            const uint32_t k = D.k, np = D.npieces;
            mbar_wait_idle(done0 + 8 * d, ph);
            const uint32_t at = (uint32_t)lane < np ? D.piece_at[lane] : 0u;
            const uint32_t cnt = (uint32_t)lane < np ? D.piece_cnt[lane] : 0u;
            const uint32_t incl = warp_incl_scan(cnt, lane);
            const uint32_t total = __shfl_sync(kFull, incl, 31);
            const uint32_t lo = __shfl_sync(kFull, incl - cnt, ((uint32_t)lane * ppt) & 31u);   // lane i: before tile i
            const uint32_t base = hier_prefix(a.blk_acc, a.grp_acc, a.tile_word, tag, t0, E, E_blk, lane);
            if ((uint32_t)lane < k) {
                a.Io[t0 + lane] = base + lo;
                if (t0 + lane + 1u == a.T) a.Io[a.T] = base + total;
            }
            // ---- the pieces' survivors -> Ao ----------------------------------------------------------------
            const uint32_t dst = base + incl - cnt;
            const uint32_t maxc = __reduce_max_sync(kFull, cnt);
            if (maxc <= 8u) {               // a few values per piece: lane p moves piece p
                for (uint32_t e = 0; e < cnt; ++e) a.Ao[dst + e] = pool[at + e];
            } else if (total >= 256u * k) {
                // long runs.  The pieces of a tile are contiguous in the output ring unless a cancellation left a gap:
                // then a tile is ONE run (lane i < k: tile i), else every piece is its own run.
                const uint32_t at_prev = __shfl_up_sync(kFull, at, 1), cnt_prev = __shfl_up_sync(kFull, cnt, 1);
                const bool joint = (uint32_t)lane >= np || ((uint32_t)lane & (ppt - 1u)) == 0u || at == at_prev + cnt_prev;
                const bool by_tile = __all_sync(kFull, joint);
                const uint32_t nruns = by_tile ? k : np;
                const uint32_t hi = __shfl_sync(kFull, incl, ((uint32_t)lane * ppt + ppt - 1u) & 31u);
                const uint32_t r_at = by_tile ? __shfl_sync(kFull, at, ((uint32_t)lane * ppt) & 31u) : at;
                const uint32_t r_cnt = by_tile ? hi - lo : cnt;
                const uint32_t r_dst = by_tile ? base + lo : dst;
                for (uint32_t r = 0; r < nruns; ++r)
                    copy_run(pool, __shfl_sync(kFull, r_at, r), a.Ao + __shfl_sync(kFull, r_dst, r),
                             __shfl_sync(kFull, r_cnt, r), lane);
            } else {
                // four pieces at a time: four independent shared -> global chains per lane
                for (uint32_t p = 0; p < np; p += 4) {
                    uint32_t s4[4], c4[4], o4[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        s4[q] = __shfl_sync(kFull, at, (p + q) & 31u);
                        c4[q] = p + q < np ? __shfl_sync(kFull, cnt, (p + q) & 31u) : 0u;
                        o4[q] = __shfl_sync(kFull, dst, (p + q) & 31u);
                    }
                    const uint32_t cmax = max(max(c4[0], c4[1]), max(c4[2], c4[3]));
                    for (uint32_t e = lane; e < cmax; e += 32u) {
                        uint32_t v[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q) v[q] = e < c4[q] ? pool[s4[q] + e] : 0u;
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            if (e < c4[q]) a.Ao[o4[q] + e] = v[q];
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(fl0 + 8 * d);
    }
    // ---- the last flusher warp of the launch clears the accumulators, resets the ticket, advances the epoch ----
    uint32_t last = 0;
    if (lane == 0) {
        __threadfence();
        last = atomicAdd(&a.hdr->finished, 1u) + 1u == gridDim.x * (uint32_t)kFlushers;
    }
    if (__shfl_sync(kFull, last, 0)) {
        const uint32_t ngrp = (a.T + 31u) / 32u, nblk = (a.T + 1023u) / 1024u;
        for (uint32_t q = lane; q < ngrp; q += 32) a.grp_acc[q] = 0;
        for (uint32_t q = lane; q < nblk; q += 32) a.blk_acc[q] = 0;
        if (lane == 0) {
            a.hdr->ticket = 0;
            a.hdr->finished = 0;
        }
        finish_epoch(a.hdr, tag, a.tile_word, a.tile_words, lane);
    }
}

__global__ void __launch_bounds__(kMergeThreads, kCtasPerSm)
reduce_ss_kernel(const Batch<MergeArgs> batch) {
    extern __shared__ __align__(128) uint32_t pool[];
    __shared__ MergeShared sh;
    const MergeArgs &a = batch.job[blockIdx.y];
    if (gate_closed(a.gate.ptr, a.gate.mask, a.gate.value)) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tag = launch_tag(a.hdr);   // this launch's tag for the tile words (pici_common.cuh)
    // the producer's first ticket is requested before anything else: it returns while the geometry loads do
    uint32_t tk0 = 0;
    if (warp == kWorkers && lane == 0) tk0 = atomicAdd(&a.hdr->ticket, 1u);
    const Geometry geo = geometry(a, gridDim.x);
    if (tid == 0) {
        for (int d = 0; d < kDesc; ++d) {
            mbar_init(smem_u32(&sh.full[d]), 1);
            mbar_init(smem_u32(&sh.done[d]), kWorkers);
            mbar_init(smem_u32(&sh.flushed[d]), kFlushers + 1);
        }
        for (int q = 0; q < kPlans; ++q) {
            mbar_init(smem_u32(&sh.plan_full[q]), 1);
            mbar_init(smem_u32(&sh.plan_free[q]), 1);
        }
    }
    __syncthreads();

    if (warp < kWorkers) {
        switch (geo.lb) {
            case 128: worker<128>(a, sh, pool, warp, lane); break;
            case 64: worker<64>(a, sh, pool, warp, lane); break;
            case 32: worker<32>(a, sh, pool, warp, lane); break;
            default: worker<16>(a, sh, pool, warp, lane); break;
        }
    } else if (warp == kWorkers) {
        planner(a, sh, geo, tk0, lane);
    } else if (warp == kWorkers + 1) {
        issuer(a, sh, pool, geo, lane);
    } else if (warp == kWorkers + 2) {
        publisher(a, sh, geo, tag, lane);
    } else {
        flusher(a, sh, pool, geo, tag, warp - kWorkers - 3, lane);
    }
}

cudaError_t launch_reduce_ss_batch(const MergeJob *jobs, int count, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (count > kMaxBatch) return cudaErrorInvalidValue;
    const size_t smem = (size_t)kPoolWords * sizeof(uint32_t);
    static std::atomic<bool> configured_on[64];   // one-time setup per device; doing it twice is harmless
    std::atomic<bool> &configured = configured_on[current_device_slot()];
    if (!configured.load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(reduce_ss_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured.store(true, std::memory_order_release);
    }
    Batch<MergeArgs> batch;
    uint64_t Tmax = 0;
    for (int j = 0; j < count; ++j) {
        const MergeJob &q = jobs[j];
        const uint64_t n = q.n, T = (n + kTile - 1) / kTile;
        Tmax = max(Tmax, T);
        if ((uint64_t)kWsHeaderBytes + ((uint64_t)kWsAccWords + T) * 8 > scan_workspace_bytes(n)) return cudaErrorInvalidValue;   // cannot happen
        uint64_t *base = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(q.ws) + kWsHeaderBytes);
        MergeArgs &a = batch.job[j];
        a.Bx = q.Bx; a.By = q.By; a.Ix = q.Ix; a.Iy = q.Iy;
        a.Ax = reinterpret_cast<const uint32_t *>(q.Ax); a.Ay = reinterpret_cast<const uint32_t *>(q.Ay);
        a.Bo = q.Bo; a.Io = q.Io; a.Ao = reinterpret_cast<uint32_t *>(q.Ao);
        a.hdr = reinterpret_cast<MergeHeader *>(q.ws);
        a.blk_acc = base; a.grp_acc = base + kWsBlkWords; a.tile_word = base + kWsAccWords;
        a.tile_words = (scan_workspace_bytes(n) - kWsHeaderBytes) / 8 - kWsAccWords;
        a.T = (uint32_t)T;
        a.zero = 0;
        a.a_limit = (n * 4) & ~15ull;
        a.gate = q.gate;
    }
    // the block length is chosen on the device.  A chunk of a few thousand tiles does not need the whole GPU, and
    // the jobs of a batch (the logical ranks of one ring step) share it
    uint64_t blocks = (Tmax + kWorkers - 1) / kWorkers;
    const uint64_t cap = max((uint64_t)kCtasPerSm * (uint64_t)num_sms() / count, (uint64_t)1);
    if (blocks > cap) blocks = cap;
    reduce_ss_kernel<<<dim3((unsigned)blocks, (unsigned)count), kMergeThreads, smem, s>>>(batch);
    return cudaGetLastError();
}

cudaError_t launch_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                             const uint32_t *Iy, const void *Ay, uint64_t n, uint64_t *Bo, uint32_t *Io,
                             void *Ao, void *ws, Gate g, cudaStream_t s) {
    if (n == 0) return launch_set_u32(Io, 0u, g, s);
    const MergeJob job = {Bx, Ix, Ax, By, Iy, Ay, n, Bo, Io, Ao, ws, g};
    return launch_reduce_ss_batch(&job, 1, s);
}

}  // namespace pici
