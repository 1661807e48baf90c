// expand.cu - the "Phase 3 reversed" family: pici_decompress, pici_reduce_sd (the
// scatter-add "decompression"), pici_maybe_densify.
//
// One warp owns one 64x64 tile at a time; lane l owns the ADJACENT columns 2l and 2l+1 (the paper's
// Phase-3 mapping), i.e. the two 64-bit words B[64t+2l], B[64t+2l+1] - one 16-byte load
// per lane, 512 contiguous bytes per warp.  Because A is ordered tile -> column -> row, the values of
// lane l's two columns are ONE contiguous run of A that starts at
//     I[t] + (exclusive warp scan of popc(word 2l) + popc(word 2l+1)).
// The kernel is written as a GATHER over rows, not a scatter over set bits:
//   * the tile's segment of A, A[I[t] .. I[t+1]), is staged in shared memory by ONE 1-D TMA bulk copy
//     (cp.async.bulk on a 16-byte aligned window; the < 16-byte tail goes through plain loads so
//     nothing past the segment is ever read) - no per-value global latency;
//   * for row r = 0..63 (fully unrolled) the lane tests bit r of its two words, reads the next value
//     of the column's run from the stage if the bit is set (running cursor), and the warp writes the
//     row as one coalesced 256-byte (fp32) / 128-byte (bf16) streaming store straight to global
//     memory.  No tile buffer, no zero fill, no shared-memory scatter, no copy-out.
//   * reduce_sd, streaming form (out != local, or a tile with many values): same walk, the row of
//     `local` is loaded 16 rows ahead and `a` is added where the bit is set; elements without a bit
//     keep their bits exactly (a -0.0 survives).
//   * reduce_sd, sparse form (in place and <= kSparseTileNnz values in the tile): the lanes first turn
//     their words into a tile-local index list in shared memory (A order), then the warp walks that
//     list 32 values at a time - coalesced loads of A, gather of the touched elements, add, scatter -
//     with every load of the tile in flight before the first store (sector-granular traffic,
//     SURVEY.md S7 #4).
// The next tile's words and I[t] are prefetched into registers while the current tile is processed.
#include <atomic>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

#ifndef PICI_RMW_WAVES
#define PICI_RMW_WAVES 2   // waves of CTAs of the read-modify-write kernel (1 -> 2: 0.302 -> 0.292 ms at 95 %; 4, 8: the same)
#endif
constexpr int kExpandWarps = 1;
#ifndef PICI_DECOMPRESS_WAVES
#define PICI_DECOMPRESS_WAVES 12
#endif
constexpr uint64_t kDecompressWaves = PICI_DECOMPRESS_WAVES;   // waves of CTAs a decompress launch is cut into
#ifndef PICI_SPARSE_TILE_NNZ
#define PICI_SPARSE_TILE_NNZ 128
#endif
constexpr uint32_t kSparseTileNnz = PICI_SPARSE_TILE_NNZ;   // in-place add: tiles with <= this many values use RMW
static_assert(kSparseTileNnz % 32 == 0 && kSparseTileNnz <= 1024, "sparse list is walked 32 values at a time");

enum { kModeDecompress = 0, kModeAdd = 1 };

// In-place scatter-add picks its kernel ON THE DEVICE from the measured total I[T] (no host sync): with
// at most kSparseAvgNnz values per tile on average the launch is a read-modify-write of the touched
// elements only (scatter_add_sparse_kernel, sector-granular traffic); above it the
// dense buffer is streamed through (expand_kernel).  Both kernels are enqueued, one returns at once.
#ifndef PICI_SPARSE_AVG_NNZ
#define PICI_SPARSE_AVG_NNZ 224
#endif
constexpr uint32_t kSparseAvgNnz = PICI_SPARSE_AVG_NNZ;
constexpr uint32_t kSparseListMax = 256;   // values of one tile that fit the per-warp index list
__device__ __forceinline__ bool sparse_regime(const uint32_t *__restrict__ I, uint32_t T) {
    return (uint64_t)__ldg(I + T) <= (uint64_t)kSparseAvgNnz * T;
}

template <int DT>
struct ExpandCfg {
    using Elem = typename ElemOf<DT>::type;
    static constexpr uint32_t kStageBytes = kTile * sizeof(Elem) + 32;   // segment + alignment slack
};

__device__ __forceinline__ uint2 ld_coherent_u2(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p) : "memory");
    return v;
}
// Gather load of the scatter-add: a miss fetches 64 bytes from DRAM instead of the default 128-byte
// line pair (probe on B200: 185 MB instead of 403 MB of DRAM reads for 2.7 M random 4-byte gathers).
__device__ __forceinline__ uint32_t ld_gather_u32(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.global.L2::64B.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ ulonglong2 ldg_nc_u64x2(const uint64_t *p) {
    ulonglong2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p));
    return v;
}

template <int DT, int MODE>
__global__ void __launch_bounds__(kExpandWarps * 32)
expand_kernel(const Batch<ExpandJob> batch) {
    using Elem = typename ExpandCfg<DT>::Elem;
    constexpr uint32_t ES = sizeof(Elem);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t mbar_mem[kExpandWarps];
    const ExpandJob &job = batch.job[blockIdx.y];
    if (gate_closed(job.gate.ptr, job.gate.mask, job.gate.value)) return;
    const uint64_t *__restrict__ B = job.B;
    const uint32_t *__restrict__ I = job.I;
    const void *__restrict__ A = job.A;
    const uint64_t n = job.n;
    const void *local = job.local;
    void *out = job.out;
    const DensifyCtl ctl = job.ctl;

    const uint32_t T = (uint32_t)((n + kTile - 1) / kTile);
    if constexpr (MODE == kModeAdd && DT == PICI_F32) {  // in place: the sparse regime belongs to scatter_add_sparse_kernel
        if (local == out && sparse_regime(I, T)) return;       // (bf16 sums always stream: include/pici.h)
    }
    if (ctl.d_flag != nullptr) {  // maybe_densify: integer compare on the measured nnz (C9 #9/#10)
        const bool switched = (uint64_t)I[T] >= ctl.nnz_switch;
        if (blockIdx.x == 0 && threadIdx.x == 0) *ctl.d_flag = switched ? ctl.on_value : ctl.off_value;
        if (!switched || out == nullptr) return;
    }

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    unsigned char *stage_raw = smem_raw + (size_t)warp * ExpandCfg<DT>::kStageBytes;
    Elem *stage = reinterpret_cast<Elem *>(stage_raw);
    const uint32_t stage_s = smem_u32(stage_raw);
    const uint32_t bar = smem_u32(&mbar_mem[warp]);
    if (lane == 0) mbar_init(bar, 1);
    __syncwarp();
    uint32_t parity = 0;

    const Elem *Ain = reinterpret_cast<const Elem *>(A);
    const Elem *Lin = reinterpret_cast<const Elem *>(local);
    Elem *Dout = reinterpret_cast<Elem *>(out);
    const bool in_place = (MODE == kModeAdd) && (local == out);
    const uint32_t Tfull = (uint32_t)(n / kTile);
    const uint32_t stride = gridDim.x * kExpandWarps;

    uint32_t t = blockIdx.x * kExpandWarps + warp;
    ulonglong2 wn = make_ulonglong2(0, 0);
    uint32_t segn = 0;
    if (t < T) {
        wn = ldg_nc_u64x2(B + (size_t)t * kSide + 2 * lane);
        segn = __ldg(I + t);
    }
    for (; t < T; t += stride) {
        const ulonglong2 w = wn;
        const uint32_t seg = segn;
        if (t + stride < T) {  // prefetch the next tile's words and segment start
            wn = ldg_nc_u64x2(B + (size_t)(t + stride) * kSide + 2 * lane);
            segn = __ldg(I + t + stride);
        }
        const uint32_t cnt0 = __popcll(w.x), cnt1 = __popcll(w.y);
        const uint32_t incl = warp_incl_scan(cnt0 + cnt1, lane);
        const uint32_t tile_nnz = __shfl_sync(kFull, incl, 31);
        const uint32_t excl = incl - cnt0 - cnt1;   // tile-local slot of this lane's first value
        const size_t base = (size_t)t * kTile;
        const bool full = t < Tfull;

        if constexpr (MODE == kModeAdd) {
            if (in_place && tile_nnz == 0) continue;
        }
        if constexpr (MODE == kModeAdd && DT == PICI_F32) {
            if (in_place && tile_nnz <= kSparseTileNnz) {
                // ---- sparse form: index list, then batched gather / add / scatter ------------------
                uint16_t *list = reinterpret_cast<uint16_t *>(stage_raw);
                uint32_t k = excl;
                uint64_t u = w.x;
                while (u) {
                    const uint32_t r = __ffsll((long long)u) - 1;
                    u &= u - 1;
                    list[k++] = (uint16_t)(r * kSide + 2 * lane);
                }
                u = w.y;
                while (u) {
                    const uint32_t r = __ffsll((long long)u) - 1;
                    u &= u - 1;
                    list[k++] = (uint16_t)(r * kSide + 2 * lane + 1);
                }
                __syncwarp();
                constexpr int kIt = kSparseTileNnz / 32;
                const uint32_t *Au = reinterpret_cast<const uint32_t *>(A) + seg;
                uint32_t *Du = reinterpret_cast<uint32_t *>(out) + base;
                uint32_t av[kIt], dv[kIt], ix[kIt];
#pragma unroll
                for (int j = 0; j < kIt; ++j) {
                    const uint32_t jj = 32 * j + lane;
                    if (jj < tile_nnz) {
                        ix[j] = list[jj];
                        av[j] = ldg_stream_u32(Au + jj);
                        dv[j] = ld_gather_u32(Du + ix[j]);
                    }
                }
#pragma unroll
                for (int j = 0; j < kIt; ++j) {
                    const uint32_t jj = 32 * j + lane;
                    if (jj < tile_nnz)
                        Du[ix[j]] = __float_as_uint(__fadd_rn(__uint_as_float(dv[j]), __uint_as_float(av[j])));
                }
                __syncwarp();
                continue;
            }
        }
        if constexpr (MODE == kModeDecompress) {
            if (tile_nnz == 0 && full) {  // an empty tile: 16 KB / 8 KB of +0.0
                uint4 *dst = reinterpret_cast<uint4 *>(Dout + base);
                constexpr int kVec = kTile * ES / 16;
#pragma unroll
                for (int i = 0; i < kVec / 32; ++i) stg_stream_u4(dst + 32 * i + lane, make_uint4(0, 0, 0, 0));
                continue;
            }
        }

        // ---- stage the tile's segment of A: one TMA bulk copy + a < 16-byte tail ---------------------
        const uint64_t a_beg = (uint64_t)seg * ES, a_end = a_beg + (uint64_t)tile_nnz * ES;
        const uint64_t start_al = a_beg & ~15ull, end_dn = a_end & ~15ull;
        const uint32_t bulk = end_dn > start_al ? (uint32_t)(end_dn - start_al) : 0u;
        if (tile_nnz != 0) {
            if (bulk != 0 && lane == 0) {
                fence_proxy_async_smem();
                mbar_expect_tx(bar, bulk);
                bulk_g2s(stage_s, reinterpret_cast<const unsigned char *>(A) + start_al, bulk, bar);
            }
            const uint64_t tail_beg = bulk != 0 ? end_dn : a_beg;
            const uint32_t tail_cnt = (uint32_t)(a_end - tail_beg) / ES;
            if ((uint32_t)lane < tail_cnt)
                stage[(uint32_t)(tail_beg - start_al) / ES + lane] = Ain[tail_beg / ES + lane];
        }
        uint32_t k0 = (uint32_t)(a_beg - start_al) / ES + excl;   // cursor of column 2l in the stage
        uint32_t k1 = k0 + cnt0;                                  // cursor of column 2l+1
        const uint32_t w0lo = (uint32_t)w.x, w0hi = (uint32_t)(w.x >> 32);
        const uint32_t w1lo = (uint32_t)w.y, w1hi = (uint32_t)(w.y >> 32);
        // rows of the tile that hold any value at all (at 99 % sparsity half of them do not: those rows are
        // one store of zeros, no bit tests, no shared-memory reads)
        const uint32_t rows_lo = __reduce_or_sync(kFull, w0lo | w1lo), rows_hi = __reduce_or_sync(kFull, w0hi | w1hi);

        if (full) {
            constexpr int kChunk = 16;
#pragma unroll
            for (int c = 0; c < kSide / kChunk; ++c) {
                uint2 loc[kChunk];
                if constexpr (MODE == kModeAdd && DT == PICI_F32) {
                    const uint2 *src = reinterpret_cast<const uint2 *>(Lin + base) + lane;
#pragma unroll
                    for (int j = 0; j < kChunk; ++j) loc[j] = ld_coherent_u2(src + 32 * (kChunk * c + j));
                } else if constexpr (MODE == kModeAdd) {      // bf16: a row is 128 bytes, one 32-bit word per lane
                    const uint32_t *src = reinterpret_cast<const uint32_t *>(Lin + base) + lane;
#pragma unroll
                    for (int j = 0; j < kChunk; ++j) {
                        uint32_t x;
                        asm volatile("ld.global.L1::no_allocate.u32 %0, [%1];" : "=r"(x) : "l"(src + 32 * (kChunk * c + j)) : "memory");
                        loc[j].x = x;
                    }
                }
                if (c == 0) {
                    if (bulk != 0) {
                        mbar_wait(bar, parity);
                        parity ^= 1u;
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int j = 0; j < kChunk; ++j) {
                    const int r = kChunk * c + j;
                    const uint32_t m = 1u << (r & 31);
                    const bool b0 = ((r < 32 ? w0lo : w0hi) & m) != 0u;
                    const bool b1 = ((r < 32 ? w1lo : w1hi) & m) != 0u;
                    if constexpr (MODE == kModeDecompress) {
                        uint32_t v0 = 0, v1 = 0;
                        if (DT != PICI_F32 || ((r < 32 ? rows_lo : rows_hi) & m)) {   // warp-uniform: some lane has a value in
                                                                                      // this row (bf16: the test costs more
                                                                                      // than it saves, measured)
                            if (b0) v0 = stage[k0++];
                            if (b1) v1 = stage[k1++];
                        }
                        if constexpr (DT == PICI_F32) {
                            stg_stream_u2(reinterpret_cast<uint2 *>(Dout + base) + lane + 32 * r, make_uint2(v0, v1));
                        } else {
                            stg_stream_u32(reinterpret_cast<uint32_t *>(Dout + base) + lane + 32 * r, v0 | (v1 << 16));
                        }
                    } else if constexpr (DT == PICI_F32) {
                        uint2 v = loc[j];
                        if (b0) v.x = __float_as_uint(__fadd_rn(__uint_as_float(v.x), __uint_as_float(stage[k0++])));
                        if (b1) v.y = __float_as_uint(__fadd_rn(__uint_as_float(v.y), __uint_as_float(stage[k1++])));
                        stg_stream_u2(reinterpret_cast<uint2 *>(Dout + base) + lane + 32 * r, v);
                    } else {                                  // bf16: columns 2l (low half) and 2l + 1 (high half)
                        uint32_t lo = loc[j].x & 0xFFFFu, hi = loc[j].x >> 16;
                        if (b0) lo = bf16_add_bits(lo, stage[k0++]);
                        if (b1) hi = bf16_add_bits(hi, stage[k1++]);
                        stg_stream_u32(reinterpret_cast<uint32_t *>(Dout + base) + lane + 32 * r, lo | (hi << 16));
                    }
                }
            }
        } else {
            // ---- ragged last tile: elements >= n do not exist (their bits are 0, C9 #4) -------------
            const uint32_t valid = (uint32_t)(n - base);
            if (bulk != 0) {
                mbar_wait(bar, parity);
                parity ^= 1u;
            }
            __syncwarp();
            for (uint32_t r = 0; r < (uint32_t)kSide; ++r) {
                const uint32_t i0 = r * kSide + 2 * lane;
                const bool b0 = (w.x >> r) & 1ull, b1 = (w.y >> r) & 1ull;
                Elem a0 = 0, a1 = 0;
                if (b0) a0 = stage[k0++];
                if (b1) a1 = stage[k1++];
                if constexpr (MODE == kModeDecompress) {
                    if (i0 < valid) Dout[base + i0] = a0;
                    if (i0 + 1 < valid) Dout[base + i0 + 1] = a1;
                } else if constexpr (DT == PICI_F32) {
                    if (i0 < valid) {
                        const uint32_t l0 = Lin[base + i0];
                        Dout[base + i0] = b0 ? __float_as_uint(__fadd_rn(__uint_as_float(l0), __uint_as_float(a0))) : l0;
                    }
                    if (i0 + 1 < valid) {
                        const uint32_t l1 = Lin[base + i0 + 1];
                        Dout[base + i0 + 1] = b1 ? __float_as_uint(__fadd_rn(__uint_as_float(l1), __uint_as_float(a1))) : l1;
                    }
                } else {
                    if (i0 < valid) {
                        const uint16_t l0 = Lin[base + i0];
                        Dout[base + i0] = b0 ? (uint16_t)bf16_add_bits(l0, a0) : l0;
                    }
                    if (i0 + 1 < valid) {
                        const uint16_t l1 = Lin[base + i0 + 1];
                        Dout[base + i0 + 1] = b1 ? (uint16_t)bf16_add_bits(l1, a1) : l1;
                    }
                }
            }
        }
        __syncwarp();  // every lane is done with the stage before the next tile's copy lands in it
    }
}

// ---- reduce_sd, sparse regime (in place) ---------------------------------------------------------
// One warp per tile, 8 warps per CTA and only 512 bytes of shared memory per warp, so ~40 warps per SM
// keep enough read-modify-writes in flight to cover HBM latency (the 16 KB stage of expand_kernel
// limits it to 13 warps per SM; profiles/r1b: 52 % long-scoreboard stalls at 15 % issue activity).
// Per tile: the lanes turn their two column words into a tile-local index list in A order (shared
// memory), then the warp walks the list 32 values at a time - coalesced loads of A, gather of the
// touched elements, one __fadd_rn each, scatter - with up to 128 gathers in flight per warp before the
// first store.  Tiles are disjoint ranges of the dense buffer and a tile's list has no duplicates, so
// no two threads touch the same element.  A tile with more than kSparseListMax values (rare here:
// the regime is chosen from the average) is walked lane by lane without the list.
constexpr int kSparseWarps = 8;
constexpr uint32_t kSparseGroup = 8;   // tiles whose index entries a warp fetches at once
constexpr uint32_t kSparseRowMajorNnz = 112;   // tiles with at least this many values get a row-major list
__global__ void __launch_bounds__(kSparseWarps * 32, 5)
scatter_add_sparse_kernel(const uint64_t *__restrict__ B, const uint32_t *__restrict__ I,
                          const uint32_t *__restrict__ A, uint64_t n, uint32_t *dense, Gate gate) {
    // per warp: the tile's touched elements as a list in ROW-MAJOR (address) order - dense position and index into
    // the tile's run of A - so that the 32 lanes of a gather touch ascending, neighbouring addresses
    __shared__ uint16_t lists[kSparseWarps][kSparseListMax], alists[kSparseWarps][kSparseListMax];
    if (gate_closed(gate.ptr, gate.mask, gate.value)) return;
    const uint32_t T = (uint32_t)((n + kTile - 1) / kTile);
    if (!sparse_regime(I, T)) return;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint16_t *list = lists[warp], *alist = alists[warp];
    const uint32_t ngroups = (T + kSparseGroup - 1) / kSparseGroup;
    const uint32_t stride = gridDim.x * kSparseWarps;
    const unsigned lt = (1u << lane) - 1u;
    for (uint32_t g = blockIdx.x * kSparseWarps + warp; g < ngroups; g += stride) {
        // index entries of the group's tiles in one request; empty tiles cost nothing more
        const uint32_t t0 = g * kSparseGroup;
        const uint32_t ie = __ldg(I + min(t0 + (uint32_t)lane, T));           // lanes 0 .. kSparseGroup
        const uint32_t tn = __shfl_down_sync(kFull, ie, 1) - ie;               // lane j < group: values of tile t0 + j
        unsigned todo = __ballot_sync(kFull, (uint32_t)lane < kSparseGroup && t0 + lane < T && tn != 0u);
        ulonglong2 wn = make_ulonglong2(0, 0);
        if (todo) wn = ldg_nc_u64x2(B + (size_t)(t0 + __ffs(todo) - 1) * kSide + 2 * lane);
        while (todo) {
            const uint32_t j = __ffs(todo) - 1;
            todo &= todo - 1;
            const uint32_t t = t0 + j;
            const uint32_t seg = __shfl_sync(kFull, ie, j), tile_nnz = __shfl_sync(kFull, tn, j);
            const ulonglong2 w = wn;
            if (todo) wn = ldg_nc_u64x2(B + (size_t)(t0 + __ffs(todo) - 1) * kSide + 2 * lane);   // the next tile's words
            const uint32_t cnt0 = __popcll(w.x), cnt1 = __popcll(w.y);
            const uint32_t excl = warp_incl_scan(cnt0 + cnt1, lane) - cnt0 - cnt1;
            const uint32_t *Au = A + seg;
            uint32_t *Du = dense + (size_t)t * kTile;
            if (tile_nnz > kSparseListMax) {   // outlier tile: every lane walks its own two columns
                uint32_t k = excl;
                for (uint64_t u = w.x; u; u &= u - 1) {
                    const uint32_t i = (__ffsll((long long)u) - 1) * kSide + 2 * lane;
                    Du[i] = __float_as_uint(__fadd_rn(__uint_as_float(Du[i]), __uint_as_float(Au[k++])));
                }
                for (uint64_t u = w.y; u; u &= u - 1) {
                    const uint32_t i = (__ffsll((long long)u) - 1) * kSide + 2 * lane + 1;
                    Du[i] = __float_as_uint(__fadd_rn(__uint_as_float(Du[i]), __uint_as_float(Au[k++])));
                }
                continue;
            }
            // ---- the list.  Few values: every lane walks its own two columns (A order; the gathers are far apart
            // anyway).  Many: row by row, so that a gather's 32 lanes touch neighbouring addresses ---------------------
            if (tile_nnz < kSparseRowMajorNnz) {
                uint32_t k = excl;
                for (uint64_t u = w.x; u; u &= u - 1) {
                    list[k] = (uint16_t)((__ffsll((long long)u) - 1) * kSide + 2 * lane);
                    alist[k] = (uint16_t)k;
                    ++k;
                }
                for (uint64_t u = w.y; u; u &= u - 1) {
                    list[k] = (uint16_t)((__ffsll((long long)u) - 1) * kSide + 2 * lane + 1);
                    alist[k] = (uint16_t)k;
                    ++k;
                }
            } else {
                uint32_t k0 = excl, k1 = excl + cnt0, pos = 0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const uint32_t x = h ? (uint32_t)(w.x >> 32) : (uint32_t)w.x, y = h ? (uint32_t)(w.y >> 32) : (uint32_t)w.y;
                    uint32_t rows = __reduce_or_sync(kFull, x | y);
                    while (rows) {
                        const uint32_t r = __ffs(rows) - 1;
                        rows &= rows - 1;
                        const bool b0 = (x >> r) & 1u, b1 = (y >> r) & 1u;
                        const unsigned m0 = __ballot_sync(kFull, b0), m1 = __ballot_sync(kFull, b1);
                        const uint32_t at = pos + __popc(m0 & lt) + __popc(m1 & lt);
                        const uint32_t e = (32u * h + r) * kSide + 2 * lane;
                        if (b0) { list[at] = (uint16_t)e; alist[at] = (uint16_t)k0++; }
                        if (b1) { list[at + (b0 ? 1u : 0u)] = (uint16_t)(e + 1); alist[at + (b0 ? 1u : 0u)] = (uint16_t)k1++; }
                        pos += __popc(m0) + __popc(m1);
                    }
                }
            }
            __syncwarp();
            for (uint32_t b0 = 0; b0 < tile_nnz; b0 += 128) {
                uint32_t av[4], dv[4], ix[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t jj = b0 + 32 * q + lane;
                    if (jj < tile_nnz) {
                        ix[q] = list[jj];
                        av[q] = __ldg(Au + alist[jj]);
                        dv[q] = ld_gather_u32(Du + ix[q]);
                    }
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t jj = b0 + 32 * q + lane;
                    if (jj < tile_nnz) Du[ix[q]] = __float_as_uint(__fadd_rn(__uint_as_float(dv[q]), __uint_as_float(av[q])));
                }
            }
            __syncwarp();   // the list is rebuilt by the next tile
        }
    }
}

cudaError_t launch_scatter_add_sparse(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, void *dense,
                                      Gate g, cudaStream_t s) {
    const uint64_t T = (n + kTile - 1) / kTile;
    uint64_t blocks = ((T + kSparseGroup - 1) / kSparseGroup + kSparseWarps - 1) / kSparseWarps;
    const uint64_t cap = (uint64_t)num_sms() * 5 * PICI_RMW_WAVES;
    if (blocks > cap) blocks = cap;
    if (blocks == 0) return cudaSuccess;
    scatter_add_sparse_kernel<<<(unsigned)blocks, kSparseWarps * 32, 0, s>>>(
        B, I, reinterpret_cast<const uint32_t *>(A), n, reinterpret_cast<uint32_t *>(dense), g);
    return cudaGetLastError();
}

template <int DT, int MODE>
static cudaError_t launch_expand_t(const ExpandJob *jobs, int count, cudaStream_t s) {
    const size_t smem = (size_t)kExpandWarps * ExpandCfg<DT>::kStageBytes;
    static std::atomic<bool> configured_on[64];   // one-time setup per device; doing it twice is harmless
    std::atomic<bool> &configured = configured_on[current_device_slot()];
    if (!configured.load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(expand_kernel<DT, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured.store(true, std::memory_order_release);
    }
    Batch<ExpandJob> batch;
    uint64_t T = 0;
    bool flag_only = true;
    for (int j = 0; j < count; ++j) {
        batch.job[j] = jobs[j];
        T = max(T, (jobs[j].n + kTile - 1) / kTile);
        flag_only = flag_only && jobs[j].out == nullptr;
    }
    uint64_t per_sm = (227u * 1024u) / (smem + 1024);
    if (per_sm > 32) per_sm = 32;
    uint64_t blocks = (T + kExpandWarps - 1) / kExpandWarps;
    // Decompress is write-bound, and a grid of exactly one resident wave with a fixed stride gives every SM the same
    // share of the tiles: the launch then ends with the slowest SM (a plain 16-byte-store fill of 1 GiB: 6.0 TB/s with
    // 1184 persistent CTAs, 7.2 TB/s with 65536).  kDecompressWaves waves of CTAs let the block scheduler balance the
    // SMs while a warp still walks several tiles with the next tile's words prefetched (fp32, 99 %: 0.202 -> 0.171 ms;
    // 6 / 8 / 12 / 16 waves: 0.176 / 0.175 / 0.171 / 0.171).
    // (single ungated launches only: a batch of gated ring jobs, half of which return at once, pays for every extra CTA)
    const uint64_t waves = (MODE == kModeDecompress && count == 1 && jobs[0].gate.ptr == nullptr) ? kDecompressWaves : 1;
    const uint64_t cap = max((uint64_t)num_sms() * (per_sm ? per_sm : 1) * waves / count, (uint64_t)1);
    if (blocks > cap) blocks = cap;
    if (blocks == 0 || flag_only) blocks = 1;  // n == 0 or no output: only the densify flag is written (by block 0)
    expand_kernel<DT, MODE><<<dim3((unsigned)blocks, (unsigned)count), kExpandWarps * 32, smem, s>>>(batch);
    return cudaGetLastError();
}

cudaError_t launch_expand_batch(const ExpandJob *jobs, int count, int dtype, int mode, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (count > kMaxBatch) return cudaErrorInvalidValue;
    if (mode == kModeAdd)
        return dtype == PICI_F32 ? launch_expand_t<PICI_F32, kModeAdd>(jobs, count, s) : launch_expand_t<PICI_BF16, kModeAdd>(jobs, count, s);
    return dtype == PICI_F32 ? launch_expand_t<PICI_F32, kModeDecompress>(jobs, count, s)
                             : launch_expand_t<PICI_BF16, kModeDecompress>(jobs, count, s);
}

cudaError_t launch_expand(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                          const void *local, void *out, int mode, DensifyCtl ctl, Gate g, cudaStream_t s) {
    if (n == 0 && ctl.d_flag == nullptr) return cudaSuccess;
    if (mode == kModeAdd && local == out && dtype == PICI_F32) {  // in place: the sparse-regime kernel and the streaming kernel pick on the device
        cudaError_t e = launch_scatter_add_sparse(B, I, A, n, out, g, s);
        if (e != cudaSuccess) return e;
    }
    const ExpandJob job = {B, I, A, n, local, out, ctl, g};
    return launch_expand_batch(&job, 1, dtype, mode, s);
}

}  // namespace pici
