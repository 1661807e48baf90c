// merge.cu - pici_reduce_ss: O = compress(decompress(X) + decompress(Y)) without the dense buffer.
//
// This is the fused form of the paper's reduce-scatter step "accumulate into a dense buffer using
// our Pici scatter-add kernel ... this accumulated dense buffer must be recompressed";
// the sparse+sparse merge itself is not in the paper.  Semantics (S8(c) C5):
// o_i = x_i + y_i wherever X or Y has its bit set (an absent operand reads as +0.0, one fp32 add in
// the order "received + local" = x + y), the nonzero predicate is RE-APPLIED to the sum, so an exact
// cancellation is dropped from the output mask.
//
// One warp per tile, same 32-bit half-column words as expand.cu (pass p, lane l <-> column 16p+l/2,
// rows 32(l&1)..): x's and y's slots come from the popc prefix of their own words, the candidate
// slot from the popc prefix of the OR.  Every lane compacts its surviving sums into its own run of a
// shared-memory tile stage (runs start at the OR-prefix, so they never overlap); the tile's real
// count goes through the same decoupled look-back scan as compress (Phase 2) and the stage is
// written to Ao with coalesced stores.  Only tiles that actually had a cancellation take the
// lane-by-lane copy.
#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

constexpr int kMergeWarps = 2;
constexpr int kMergePass = 1024;

__global__ void __launch_bounds__(kMergeWarps * 32)
reduce_ss_kernel(const uint64_t *__restrict__ Bx, const uint32_t *__restrict__ Ix, const uint32_t *__restrict__ Ax,
                 const uint64_t *__restrict__ By, const uint32_t *__restrict__ Iy, const uint32_t *__restrict__ Ay,
                 uint64_t n, uint64_t *__restrict__ Bo, uint32_t *__restrict__ Io, uint32_t *__restrict__ Ao,
                 uint32_t *ticket, uint64_t *status, const int32_t *gate, int32_t gate_value) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (gate_closed(gate, gate_value)) return;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *so = reinterpret_cast<uint32_t *>(smem_raw) + (size_t)warp * (kTile + 2 * kMergePass);
    uint32_t *sx = so + kTile;
    uint32_t *sy = sx + kMergePass;
    const uint32_t T = (uint32_t)((n + kTile - 1) / kTile);

    uint32_t t = next_ticket(ticket, lane);
    while (t < T) {
        uint32_t t_next = 0;
        if (lane == 0) t_next = atomicAdd(ticket, 1u);

        const uint32_t *Bxw = reinterpret_cast<const uint32_t *>(Bx + (size_t)t * kSide);
        const uint32_t *Byw = reinterpret_cast<const uint32_t *>(By + (size_t)t * kSide);
        uint32_t wx[4], wy[4], wo[4], kk[4], eu[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            wx[p] = __ldg(Bxw + 32 * p + lane);
            wy[p] = __ldg(Byw + 32 * p + lane);
        }
        uint32_t xbase = __ldg(Ix + t), ybase = __ldg(Iy + t);
        uint32_t cand_base = 0;

#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const uint32_t u0 = wx[p] | wy[p];
            const uint32_t cx = __popc(wx[p]), cy = __popc(wy[p]), cu = __popc(u0);
            const uint32_t sxy = warp_incl_scan(cx | (cy << 16), lane);
            const uint32_t su = warp_incl_scan(cu, lane);
            const uint32_t txy = __shfl_sync(kFull, sxy, 31);
            const uint32_t tx = txy & 0xFFFFu, ty = txy >> 16;
            const uint32_t tu = __shfl_sync(kFull, su, 31);
            uint32_t px = (sxy & 0xFFFFu) - cx, py = (sxy >> 16) - cy;
            eu[p] = cand_base + su - cu;
            wo[p] = 0;
            kk[p] = 0;
            if (tu != 0) {  // warp-uniform
                for (uint32_t i = lane; i < tx; i += 32) sx[i] = __ldg(Ax + xbase + i);
                for (uint32_t i = lane; i < ty; i += 32) sy[i] = __ldg(Ay + ybase + i);
                __syncwarp();
                uint32_t u = u0, k = 0, o = 0;
                uint32_t *dst = so + eu[p];
                while (u) {
                    const uint32_t bit = u & (0u - u);
                    u ^= bit;
                    const float x = (wx[p] & bit) ? __uint_as_float(sx[px++]) : 0.0f;
                    const float y = (wy[p] & bit) ? __uint_as_float(sy[py++]) : 0.0f;
                    const uint32_t s = __float_as_uint(__fadd_rn(x, y));  // received + local (C9 #7)
                    if (nz32(s)) {
                        o |= bit;
                        dst[k++] = s;
                    }
                }
                wo[p] = o;
                kk[p] = k;
                __syncwarp();
            }
            xbase += tx;
            ybase += ty;
            cand_base += tu;
        }

        // real (post-cancellation) offsets: order is (pass, lane)
        const uint32_t r01 = warp_incl_scan(kk[0] | (kk[1] << 16), lane);
        const uint32_t r23 = warp_incl_scan(kk[2] | (kk[3] << 16), lane);
        const uint32_t q01 = __shfl_sync(kFull, r01, 31), q23 = __shfl_sync(kFull, r23, 31);
        const uint32_t n0 = q01 & 0xFFFFu, n1 = q01 >> 16, n2 = q23 & 0xFFFFu, n3 = q23 >> 16;
        const uint32_t tile_nnz = n0 + n1 + n2 + n3;

        publish_count(status, t, tile_nnz, lane);

        uint32_t *Bow = reinterpret_cast<uint32_t *>(Bo + (size_t)t * kSide);
#pragma unroll
        for (int p = 0; p < 4; ++p) Bow[32 * p + lane] = wo[p];

        const uint32_t excl = lookback_prefix(status, t, tile_nnz, T, Io, lane);

        uint32_t *dst = Ao + excl;
        if (tile_nnz == cand_base) {  // no cancellation anywhere in the tile: the stage is already packed
            for (uint32_t i = lane; i < tile_nnz; i += 32) dst[i] = so[i];
        } else {
            const uint32_t ro[4] = {(r01 & 0xFFFFu) - kk[0], n0 + (r01 >> 16) - kk[1],
                                    n0 + n1 + (r23 & 0xFFFFu) - kk[2], n0 + n1 + n2 + (r23 >> 16) - kk[3]};
#pragma unroll
            for (int p = 0; p < 4; ++p)
                for (uint32_t j = 0; j < kk[p]; ++j) dst[ro[p] + j] = so[eu[p] + j];
        }
        __syncwarp();

        t = __shfl_sync(kFull, t_next, 0);
    }
}

cudaError_t launch_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                             const uint32_t *Iy, const void *Ay, uint64_t n, uint64_t *Bo, uint32_t *Io,
                             void *Ao, void *ws, Gate g, cudaStream_t s) {
    if (n == 0) return launch_set_u32(Io, 0u, g, s);
    const uint64_t T = (n + kTile - 1) / kTile;
    const size_t smem = (size_t)kMergeWarps * (kTile + 2 * kMergePass) * sizeof(uint32_t);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(reduce_ss_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    cudaError_t e = cudaMemsetAsync(ws, 0, scan_workspace_bytes(n), s);
    if (e != cudaSuccess) return e;
    const uint64_t per_sm = (227u * 1024u) / (smem + 1024);
    uint64_t blocks = (T + kMergeWarps - 1) / kMergeWarps;
    const uint64_t cap = (uint64_t)num_sms() * per_sm;             // persistent: one resident wave
    if (blocks > cap) blocks = cap;
    uint32_t *ticket = reinterpret_cast<uint32_t *>(ws);
    uint64_t *status = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(ws) + kWsHeaderBytes);
    reduce_ss_kernel<<<(unsigned)blocks, kMergeWarps * 32, smem, s>>>(
        Bx, Ix, reinterpret_cast<const uint32_t *>(Ax), By, Iy, reinterpret_cast<const uint32_t *>(Ay), n, Bo, Io,
        reinterpret_cast<uint32_t *>(Ao), ticket, status, g.ptr, g.value);
    return cudaGetLastError();
}

}  // namespace pici
