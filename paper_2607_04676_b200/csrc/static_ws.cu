// static_ws.cu - pici_compress_static (include/pici_static.h): pici_compress with its scan scratch in a file-scope
// device array instead of a caller-owned workspace, for callers that may not allocate.  Nothing here or below
// allocates: the array is part of the library's image on every GPU that loads it.
//
// g_scratch is named in HOST code only as the argument of cudaGetSymbolAddress - in host code the name is a host-side
// stand-in, not a device address; the kernels get the address that call returns, taken once per device with that
// device current.
#include <atomic>

#include "../../include/pici.h"
#include "../../include/pici_static.h"
#include "launch.h"
#include "pici_common.cuh"

namespace pici {
namespace {

constexpr uint64_t kStaticMaxN = PICI_STATIC_MAX_N;
constexpr uint64_t kStaticMaxTiles = kStaticMaxN / kTile;
// = scan_workspace_bytes(kStaticMaxN) (pici_common.cuh tile_words_end); checked at set-up
constexpr uint64_t kStaticBytes = (uint64_t)kWsHeaderBytes + ((uint64_t)kWsAccWords + ((kStaticMaxTiles + 65) & ~1ull)) * 8;
static_assert(kStaticBytes == PICI_STATIC_SCRATCH_BYTES, "pici_static.h states the array's size");

static __device__ __align__(256) unsigned char g_scratch[kStaticBytes];   // zero when the module is loaded

// What a launch expects to be zero (ticket and exit counters, the scan service's done words = reduce_ss's
// accumulator area); the WsHeader in front of it - the launch epoch - must SURVIVE: it is what makes the tagged
// per-tile words of earlier calls stale.
constexpr size_t kZeroBegin = kWsCompressTicket;
constexpr size_t kZeroEnd = (size_t)kWsHeaderBytes + (size_t)kWsAccWords * 8;

// Device address of g_scratch on the current device, taken once per device (slots for devices 0..63; others ask the
// runtime every time).  No allocation: cudaGetSymbolAddress only loads the module that holds the array.
cudaError_t scratch_address(void **out) {
    static std::atomic<void *> cached[64];
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool slot = dev >= 0 && dev < 64;
    void *p = slot ? cached[dev].load(std::memory_order_acquire) : nullptr;
    if (p == nullptr) {
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr || scan_workspace_bytes(kStaticMaxN) != kStaticBytes) return cudaErrorInvalidValue;
        if (slot) cached[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

inline bool al(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

}  // namespace
}  // namespace pici

using namespace pici;

extern "C" int pici_static_limits(uint64_t *max_n, uint64_t *scratch_bytes) {
    if (max_n) *max_n = kStaticMaxN;
    if (scratch_bytes) *scratch_bytes = kStaticBytes;
    return PICI_OK;
}

extern "C" int pici_compress_static(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                                    uint64_t A_capacity, void *stream) {
    // the checks of pici_compress (api.cu do_compress), then the limit
    if (dtype != PICI_F32 && dtype != PICI_BF16) return PICI_ERR_DTYPE;
    if (n >= (1ull << 32) || I == nullptr) return PICI_ERR_INVALID_ARG;
    if (n != 0 && (B == nullptr || A == nullptr || dense == nullptr)) return PICI_ERR_INVALID_ARG;
    if (!al(B, 16) || !al(A, 16) || !al(I, 4) || !al(dense, 16)) return PICI_ERR_ALIGN;
    if (A_capacity < n) return PICI_ERR_CAPACITY;
    if (n > kStaticMaxN) return PICI_ERR_WORKSPACE;     // the static scratch is too small: use pici_compress
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    void *ws = nullptr;
    if (scratch_address(&ws) != cudaSuccess) return PICI_ERR_CUDA;
    if (n != 0 &&
        cudaMemsetAsync(static_cast<unsigned char *>(ws) + kZeroBegin, 0, kZeroEnd - kZeroBegin, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    return launch_compress(dense, n, dtype, B, I, A, ws, Gate{nullptr, 0, 0}, s) == cudaSuccess ? PICI_OK : PICI_ERR_CUDA;
}
