/*
 * pici_prune.h - C ABI of the upstream workload step: sampled top-k gradient pruning with leaky
 * error feedback, fused with Pici compression (arxiv/paper_2607_04676, SVI-B: "gradient pruning
 * using a sampling-based top-k approach, imposing 99% collective input sparsity and determining the pruning threshold
 * by sampling 0.1% of gradients ... a leaky error feedback (EF) mechanism").  Hand-written CUDA for sm_100a.
 *
 * What is computed (the paper gives the recipe in two sentences; readings DESIGN.md S2 #20-#24), all fp32:
 *   acc_i  = g_i + leak * e_i        two roundings (product, then sum; never a fused multiply-add);
 *   tau    = the k-th largest of |acc_s| over the m sampled positions s (exact selection; a NaN counts as +inf);
 *   sent_i = |acc_i| >= tau ? acc_i : +0.0     (a NaN is never sent);      e_i <- sent ? +0.0 : acc_i;
 *   message = Pici(sent)   (pici.h format, same nonzero predicate).
 * The sample is the CALLER's draw (the paper: 0.1 % of the gradient): m distinct positions < n in device memory.
 *
 * Conventions are those of pici.h (device pointers, calls only enqueue, caller-owned buffers, PICI_ERR_* codes).
 * g, e, B, A, ws 16-byte aligned; d_sample, I, d_tau 4-byte.  0 < n < 2^32, 1 <= k <= m <= n.
 * ws: pici_prune_sizes() bytes, cleared once (pici_workspace_init), reusable on one stream.
 */
#ifndef PICI_PRUNE_H_
#define PICI_PRUNE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Scratch bytes for an n-element gradient and an m-element sample (covers both calls below). */
int pici_prune_sizes(uint64_t n, uint64_t m, uint64_t *workspace_bytes);

/* *d_tau = k-th largest |g_s + leak * e_s| over the sample: a gather of the m magnitudes followed by a four-pass
 * 8-bit radix selection on their bit patterns (order-preserving for non-negative floats). */
int pici_prune_threshold(const void *g, const void *e, uint64_t n, float leak, const uint32_t *d_sample, uint64_t m,
                         uint64_t k, float *d_tau, void *ws, uint64_t ws_bytes, void *stream);

/* ONE pass over g and e: prune against *d_tau, write the residual back into e_inout, emit Pici(sent) into (B, I, A)
 * (capacity >= n as in pici_compress).  Reads 8 and writes 4 bytes per element plus the Pici object. */
int pici_prune_compress(const void *g, void *e_inout, uint64_t n, float leak, const float *d_tau, uint64_t *B,
                        uint32_t *I, void *A, uint64_t A_capacity, void *ws, uint64_t ws_bytes, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PICI_PRUNE_H_ */
