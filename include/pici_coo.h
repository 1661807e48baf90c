/*
 * pici_coo.h - C ABI of the COO variant in libpici_b200: the second sparse format of
 * SpCCL (arxiv/paper_2607_04676), hand-written CUDA for sm_100a.
 *
 * The format (SII-B): "A common variant of COO treats inputs as one-dimensional, storing only a
 * single flat index per nonzero ... COO refers to this variant ... 32-bit indices and 32-bit values."
 *   idx   : uint32_t[nnz]  flat dense index of every nonzero, ASCENDING;
 *   val   : fp32 bits [nnz] copied bit for bit, same order (structure of arrays);
 *   d_nnz : uint32_t on the DEVICE (a message's length is only known there).
 * Nonzero predicate: the one of pici.h (IEEE x != 0).  Size: 8 * nnz bytes; smaller than the bitvector's metadata
 * only above 96.875 % sparsity.  The paper's COO path (SIV-D): "compression is
 * similar to Pici in structure (identify nonzeros, build an index for stream compaction, compact nonzeros),
 * decompression only requires reading index-value pairs".
 *
 * Conventions are those of pici.h: DEVICE pointers, calls only enqueue on `stream`, the caller owns every buffer,
 * error codes (PICI_OK / PICI_ERR_*), no allocation.  idx / val must have capacity >= n ELEMENTS ("COO's worst-case,
 * in which one index is needed per nonzero value").  dense, idx, val, ws 16-byte aligned, d_nnz 4-byte.
 * 0 <= n < 2^32.  fp32 only (the paper's space calculations assume 32-bit values).  `ws` is scratch of
 * pici_coo_sizes().workspace_bytes bytes, cleared ONCE after allocation (pici_workspace_init) and then reusable by
 * any sequence of calls on one stream, of any n it is large enough for, mixed with the calls of pici.h (same
 * launch-epoch scheme); one workspace per stream.
 * A COO object handed to decompress / reduce_sd / reduce_ss must have ascending, distinct indices < n (what
 * pici_coo_compress and pici_coo_reduce_ss produce); anything else is undefined behaviour on the device.
 */
#ifndef PICI_COO_H_
#define PICI_COO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Required idx / val capacity in ELEMENTS (n) and scratch bytes.  Host-only.  Outputs may be NULL. */
int pici_coo_sizes(uint64_t n, uint64_t *capacity, uint64_t *workspace_bytes);

/* dense[n] -> (idx, val, *d_nnz) in ONE pass over `dense`: nonzero test, device-wide single-pass exclusive scan of
 * per-4096-element counts (a scan service inside the launch, as in pici_compress), compaction staged through shared
 * memory. */
int pici_coo_compress(const void *dense, uint64_t n, uint32_t *idx, void *val, uint64_t capacity,
                      uint32_t *d_nnz, void *ws, uint64_t ws_bytes, void *stream);

/* (idx, val, *d_nnz) -> dense_out[n]; EVERY element is written (absent elements +0.0), each byte of dense_out
 * once: 4096-element blocks are assembled in shared memory from their index range. */
int pici_coo_decompress(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n,
                        void *dense_out, void *ws, uint64_t ws_bytes, void *stream);

/* Scatter-add of a COO message into the dense accumulator (the reduce-scatter step of PAPER.md:219 with COO in
 * Pici's place): dense_inout[idx[k]] = dense_inout[idx[k]] + val[k], one fp32 add each; everything else untouched. */
int pici_coo_reduce_sd(const uint32_t *idx, const void *val, const uint32_t *d_nnz, uint64_t n,
                       void *dense_inout, void *stream);

/* Sparse + sparse merge: O = compress(decompress(X) + decompress(Y)) without a dense buffer; o_i = x_i + y_i where
 * either has an entry, the predicate re-applied to the sum (an exact cancellation is dropped), output ascending.
 * Outputs must not alias inputs. */
int pici_coo_reduce_ss(const uint32_t *ix, const void *vx, const uint32_t *d_nx,
                       const uint32_t *iy, const void *vy, const uint32_t *d_ny, uint64_t n,
                       uint32_t *io, void *vo, uint64_t capacity, uint32_t *d_no,
                       void *ws, uint64_t ws_bytes, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PICI_COO_H_ */
