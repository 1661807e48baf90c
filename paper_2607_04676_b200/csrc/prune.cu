// prune.cu - sampled top-k pruning threshold (include/pici_prune.h) and the C ABI of the fused
// prune-and-compress pass (the pass itself is compress_kernel<F32, PRUNE>, compress.cu).
//
// Threshold: (1) a grid-wide gather writes the m sampled magnitudes |g_s + leak * e_s| as bit patterns (a NaN as
// +inf) into the workspace; (2) one CTA selects the k-th largest by a four-pass, 8-bits-per-pass radix selection
// from the most significant byte down (bit patterns of non-negative floats order like the floats): per pass a
// shared-memory histogram of the keys that match the prefix found so far, then the bin in which the k-th largest
// lies.  m is 0.1 % of the gradient (2.7e5 keys at n = 2^28): the selection is ~1000 keys per thread per pass.
#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"
#include "../../include/pici_prune.h"

namespace pici {

__global__ void __launch_bounds__(256) prune_gather_kernel(const float *__restrict__ g, const float *__restrict__ e, float leak,
                                                           const uint32_t *__restrict__ sample, uint64_t m, uint32_t *keys) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; j < m; j += stride) {
        const uint32_t s = sample[j];
        const float acc = __fadd_rn(g[s], __fmul_rn(leak, e[s]));
        const float a = fabsf(acc);
        keys[j] = (a != a) ? 0x7F800000u : __float_as_uint(a);
    }
}

constexpr int kSelectThreads = 1024;
__global__ void __launch_bounds__(kSelectThreads) prune_select_kernel(const uint32_t *__restrict__ keys, uint64_t m, uint64_t k,
                                                                      float *d_tau) {
    __shared__ uint32_t hist[256];
    __shared__ uint32_t s_prefix, s_k;
    uint32_t prefix = 0, mask = 0;
    uint32_t kk = (uint32_t)k;          // rank (1-based, from the top) still to find inside the matching keys
    for (int shift = 24; shift >= 0; shift -= 8) {
        if (threadIdx.x < 256) hist[threadIdx.x] = 0;
        __syncthreads();
        for (uint64_t j = threadIdx.x; j < m; j += kSelectThreads) {
            const uint32_t key = keys[j];
            if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t above = 0;
            int b = 255;
            for (; b > 0; --b) {
                if (above + hist[b] >= kk) break;
                above += hist[b];
            }
            s_prefix = prefix | ((uint32_t)b << shift);
            s_k = kk - above;
        }
        __syncthreads();
        prefix = s_prefix;
        kk = s_k;
        mask |= 255u << shift;
        __syncthreads();
    }
    if (threadIdx.x == 0) *d_tau = __uint_as_float(prefix);
}

static uint64_t prune_workspace_bytes(uint64_t n, uint64_t m) { return scan_workspace_bytes(n) + ((m * 4 + 15) & ~15ull); }

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
    uint32_t *keys = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + scan_workspace_bytes(n));
    uint64_t blocks = (m + 255) / 256;
    const uint64_t cap = (uint64_t)num_sms() * 8;
    if (blocks > cap) blocks = cap;
    prune_gather_kernel<<<(unsigned)blocks, 256, 0, s>>>(reinterpret_cast<const float *>(g), reinterpret_cast<const float *>(e),
                                                         leak, d_sample, m, keys);
    prune_select_kernel<<<1, kSelectThreads, 0, s>>>(keys, m, k, d_tau);
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
