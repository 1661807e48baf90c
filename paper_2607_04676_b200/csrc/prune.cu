// prune.cu - sampled top-k pruning threshold (include/pici_prune.h) and the C ABI of the fused
// prune-and-compress pass (the pass itself is compress_kernel<F32, PRUNE>, compress.cu).
//
// Threshold: (1) a grid-wide gather writes the m sampled magnitudes |g_s + leak * e_s| as bit patterns (a NaN as
// +inf) into the workspace; (2) the k-th largest is selected by a four-pass, 8-bits-per-pass radix selection from
// the most significant byte down (bit patterns of non-negative floats order like the floats): per pass a histogram
// of the keys that match the prefix found so far, then the bin in which the k-th largest lies.  Each pass is one
// grid-wide launch (a single CTA took 0.12 ms for the 2.7e5 keys of n = 2^28: 20 % of a prune step).
#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"
#include "../../include/pici_prune.h"

namespace pici {

constexpr uint32_t kSelWords = 4 * 256 + 5 * 4;    // scratch of the selection: 4 histograms + per-pass {prefix, rank, blocks done, -}

__global__ void __launch_bounds__(256) prune_gather_kernel(const float *__restrict__ g, const float *__restrict__ e, float leak,
                                                           const uint32_t *__restrict__ sample, uint64_t m, uint64_t k,
                                                           uint32_t *sel, uint32_t *keys) {
    if (blockIdx.x == 0) {                       // the selection's scratch starts from zero; pass 0: no prefix, rank k
        for (uint32_t i = threadIdx.x; i < kSelWords; i += blockDim.x) sel[i] = i == 4 * 256 + 1 ? (uint32_t)k : 0u;
    }
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; j < m; j += stride) {
        const uint32_t s = sample[j];
        const float acc = __fadd_rn(g[s], __fmul_rn(leak, e[s]));
        const float a = fabsf(acc);
        keys[j] = (a != a) ? 0x7F800000u : __float_as_uint(a);
    }
}

// One pass (8 bits, most significant first) of the radix selection, grid-wide: every CTA histograms its share of the
// keys that match the prefix found so far (shared-memory atomics, then one global add per non-empty bin); the LAST CTA
// to finish - a counter behind a fence - finds the bin in which the rank lies and leaves {prefix, rank} for the next
// pass; the last pass writes the threshold.
__global__ void __launch_bounds__(256) prune_hist_kernel(const uint32_t *__restrict__ keys, uint64_t m, int pass, uint32_t *sel,
                                                         float *d_tau) {
    __shared__ uint32_t h[256];
    __shared__ uint32_t s_last;
    uint32_t *hist = sel + 256 * pass, *state = sel + 4 * 256 + 4 * pass;
    const uint32_t prefix = state[0], kk = state[1];
    const int shift = 24 - 8 * pass;
    const uint32_t mask = pass ? (0xFFFFFFFFu << (shift + 8)) : 0u;
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    for (uint64_t j0 = (uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); j0 < m; j0 += stride) {   // warp-uniform trip count
        const uint64_t j = j0 + lane;
        const uint32_t key = j < m ? keys[j] : 0u;
        const bool hit = j < m && (key & mask) == prefix;
        const unsigned act = __ballot_sync(kFull, hit);
        if (hit) {      // most keys share a few bins (the exponent byte): one shared-memory atomic per distinct bin per warp
            const uint32_t bin = (key >> shift) & 255u;
            const unsigned same = __match_any_sync(act, bin);
            if (lane == __ffs(same) - 1) atomicAdd(&h[bin], (uint32_t)__popc(same));
        }
    }
    __syncthreads();
    if (h[threadIdx.x]) atomicAdd(&hist[threadIdx.x], h[threadIdx.x]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&state[2], 1u) == gridDim.x - 1u;
    __syncthreads();
    if (s_last) {       // the last CTA: all 256 bins at once, then the walk from the top over shared memory
        __threadfence();
        h[threadIdx.x] = __ldcg(hist + threadIdx.x);
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t above = 0;
            int b = 255;
            for (; b > 0; --b) {
                if (above + h[b] >= kk) break;
                above += h[b];
            }
            const uint32_t np = prefix | ((uint32_t)b << shift);
            if (pass == 3) *d_tau = __uint_as_float(np);
            else {
                state[4] = np;
                state[5] = kk - above;
            }
        }
    }
}

static uint64_t prune_workspace_bytes(uint64_t n, uint64_t m) {
    return scan_workspace_bytes(n) + ((kSelWords * 4 + 15) & ~15ull) + ((m * 4 + 15) & ~15ull);
}

}  // namespace pici

using namespace pici;
namespace {
inline bool al(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }
inline int rc_of(cudaError_t e) { return e == cudaSuccess ? PICI_OK : PICI_ERR_CUDA; }
}  // namespace

extern "C" {

int pici_prune_sizes(uint64_t n, uint64_t m, uint64_t *workspace_bytes) {
    if (n == 0 || n >= (1ull << 32) || m > n) return PICI_ERR_INVALID_ARG;
    if (workspace_bytes) *workspace_bytes = prune_workspace_bytes(n, m);
    return PICI_OK;
}

int pici_prune_threshold(const void *g, const void *e, uint64_t n, float leak, const uint32_t *d_sample, uint64_t m,
                         uint64_t k, float *d_tau, void *ws, uint64_t ws_bytes, void *stream) {
    if (g == nullptr || e == nullptr || d_sample == nullptr || d_tau == nullptr || ws == nullptr) return PICI_ERR_INVALID_ARG;
    if (n == 0 || n >= (1ull << 32) || m == 0 || m > n || k == 0 || k > m) return PICI_ERR_INVALID_ARG;
    if (!al(g, 16) || !al(e, 16) || !al(ws, 16) || !al(d_sample, 4) || !al(d_tau, 4)) return PICI_ERR_ALIGN;
    if (ws_bytes < prune_workspace_bytes(n, m)) return PICI_ERR_WORKSPACE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    uint32_t *sel = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + scan_workspace_bytes(n));
    uint32_t *keys = sel + ((kSelWords + 3) & ~3u);
    uint64_t blocks = (m + 255) / 256;
    const uint64_t cap = (uint64_t)num_sms() * 8;
    if (blocks > cap) blocks = cap;
    prune_gather_kernel<<<(unsigned)blocks, 256, 0, s>>>(reinterpret_cast<const float *>(g), reinterpret_cast<const float *>(e),
                                                         leak, d_sample, m, k, sel, keys);
    uint64_t hb = (m + 256 * 8 - 1) / (256 * 8);
    if (hb > (uint64_t)num_sms() * 2) hb = (uint64_t)num_sms() * 2;
    for (int pass = 0; pass < 4; ++pass) prune_hist_kernel<<<(unsigned)hb, 256, 0, s>>>(keys, m, pass, sel, d_tau);
    return rc_of(cudaGetLastError());
}

int pici_prune_compress(const void *g, void *e_inout, uint64_t n, float leak, const float *d_tau, uint64_t *B, uint32_t *I,
                        void *A, uint64_t A_capacity, void *ws, uint64_t ws_bytes, void *stream) {
    if (g == nullptr || e_inout == nullptr || d_tau == nullptr || B == nullptr || I == nullptr || A == nullptr || ws == nullptr)
        return PICI_ERR_INVALID_ARG;
    if (n == 0 || n >= (1ull << 32) || g == e_inout) return PICI_ERR_INVALID_ARG;
    if (!al(g, 16) || !al(e_inout, 16) || !al(B, 16) || !al(A, 16) || !al(ws, 16) || !al(I, 4) || !al(d_tau, 4)) return PICI_ERR_ALIGN;
    if (A_capacity < n) return PICI_ERR_CAPACITY;
    if (ws_bytes < scan_workspace_bytes(n)) return PICI_ERR_WORKSPACE;
    const CompressJob job = {g, n, B, I, A, ws, Gate{nullptr, 0, 0}, reinterpret_cast<float *>(e_inout), d_tau, leak};
    return rc_of(launch_prune_compress(job, static_cast<cudaStream_t>(stream)));
}

}  // extern "C"
