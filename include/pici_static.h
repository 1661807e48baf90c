/*
 * pici_static.h - pici_compress for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the scan scratch that pici_compress takes as `ws` lives INSIDE the
 * library, in a file-scope `static __device__` array, so the call needs no workspace and allocates nothing - no
 * cudaMalloc, cudaFree or allocating library routine, here or in anything it calls.
 *
 * Same operation, same outputs bit for bit, same conventions as pici_compress (include/pici.h; PAPER.md:118-126,
 * Alg. 1): DEVICE pointers, the call only enqueues on `stream`, the caller owns dense / B / I / A.
 *
 * The limit: n <= PICI_STATIC_MAX_N = 2^28 elements (1 GiB of fp32, configs[1]).  The array is
 * PICI_STATIC_SCRATCH_BYTES = 796 288 bytes (the workspace pici_sizes() reports for that n); every GPU that loads the
 * library holds it until the process exits.  A larger n returns PICI_ERR_WORKSPACE ("scratch too small") before
 * anything is enqueued: use pici_compress with a caller-owned workspace instead.
 *
 * The array is SHARED by every call on a device and keeps what the last call left: each call first clears (one
 * cudaMemsetAsync on `stream`) the words that must be zero when the kernel starts - ticket and exit counters, the scan
 * service's done words - and the launch epoch in the array's header makes every other word of an earlier call stale
 * (include/pici.h, "Conventions").  Calls that may OVERLAP on the GPU (two streams, two host threads with a stream
 * each, a captured graph replayed beside an eager call) RACE on the array and give wrong results: serialise them on
 * one stream, or use pici_compress with one workspace per stream.
 */
#ifndef PICI_STATIC_H_
#define PICI_STATIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PICI_STATIC_MAX_N (1ull << 28)
#define PICI_STATIC_SCRATCH_BYTES 796288ull

/* The limit above, for callers that bind at run time.  Host-only.  Outputs may be NULL. */
int pici_static_limits(uint64_t *max_n, uint64_t *scratch_bytes);

/* pici_compress (include/pici.h) without `ws`: dense[n] -> (B, I, A).  dtype PICI_F32 / PICI_BF16; dense, B, A
 * 16-byte aligned, I 4-byte; A_capacity >= n ELEMENTS.  Errors: those of pici_compress, PICI_ERR_WORKSPACE if
 * n > PICI_STATIC_MAX_N, PICI_ERR_CUDA if the array's device address cannot be taken or the enqueue fails. */
int pici_compress_static(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                         uint64_t A_capacity, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PICI_STATIC_H_ */
