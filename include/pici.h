/*
 * pici.h - C ABI of libpici_b200: the per-GPU data-parallel hot path of SpCCL's sparse collectives
 * (arxiv/paper_2607_04676), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations are "PAPER.md:<line>" of the paper text plus its section / algorithm, and
 * "SURVEY.md S8(x)" for the scope table and the readings taken where the paper is silent.
 *
 * ------------------------------------------------------------------------------------------------
 * The Pici format (SIII-B)
 *   An n-element dense buffer is viewed as T = ceil(n/4096) row-major 64x64 "virtual" tiles.
 *   B : uint64_t[64*T]  B[64*t + c] is COLUMN c of tile t; bit r (LSB = row 0) is set iff the element
 *                       at dense index 4096*t + 64*r + c is nonzero.  Bits for indices >= n are 0.
 *   I : uint32_t[T+1]   I[t] = number of nonzeros in tiles 0..t-1 (exclusive prefix sum);
 *                       I[T] = nnz of the whole buffer.
 *   A : packed nonzero values (bit-for-bit copies), ordered tile -> column -> row.
 *   Nonzero predicate: nz(x) := (bits(x) & ~signbit) != 0, i.e. IEEE x != 0:
 *   +0.0 and -0.0 are zeros (never stored; -0.0 decompresses to +0.0); NaN, +-Inf, subnormals are
 *   nonzero.  No flush-to-zero anywhere.
 *
 * Conventions common to every call
 *   - All data pointers are DEVICE pointers unless the name starts with h_ (host).  `stream` is a
 *     cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Calls only enqueue work on `stream` and return; nothing synchronises the device.  Results,
 *     including nnz and switch flags, live in device memory.
 *   - The caller owns every buffer.  The library never allocates, frees or retains pointers and has
 *     no global state; it is re-entrant.  `ws` is scratch that must not be shared by calls that may
 *     run concurrently (one workspace per stream).  A workspace must be cleared ONCE after it is
 *     allocated (pici_workspace_init, or any memset to 0); after that any sequence of calls on one
 *     stream - of any n the workspace is large enough for, compress, reduce_ss, the COO and prune calls
 *     mixed - may reuse it without clearing: its first 64 bytes hold a launch epoch that the kernels
 *     advance themselves, every scan word is tagged with it, and everything that must be zero between
 *     launches lies at offsets that do not depend on n, so no call starts with a memset.
 *   - Alignment: dense, B, A, ws pointers 16-byte aligned; I 4-byte aligned.  Violations return
 *     PICI_ERR_ALIGN.
 *   - Sizes: B holds 64*T words and I holds T+1 entries even when n % 4096 != 0; A (and Ao) must
 *     have capacity >= n elements - the worst case, mirroring the paper's enlarged FIFOs
 *      - so no device-side overflow can occur.
 *   - A Pici object handed to decompress / reduce_sd / reduce_ss / maybe_densify must be one that pici_compress
 *     or pici_reduce_ss produced (or a bit-identical copy): the kernels trust that B, I and A agree with one
 *     another (popcount of a tile's words == I[t+1] - I[t] <= 4096); an inconsistent object is undefined
 *     behaviour on the device, not an error code.
 *   - Thread safety: calls may be made from several host threads (one stream and one workspace per thread); the
 *     only shared state is a per-device "kernel attributes set" flag, kept in atomics.
 *   - Limits: 0 <= n < 2^32 (I is 32-bit).  n == 0 is valid: I[0] = 0 is written.
 *   - dtype: PICI_F32 or PICI_BF16 for compress / decompress / nnz / maybe_densify / reduce_sd / dense_add; a bf16
 *     sum is taken in fp32 (both operands widened exactly, one fp32 add) and rounded to nearest even (SURVEY.md
 *     S8(b)), and bf16 reduce_sd always streams the dense buffer (the read-modify-write regime is fp32).
 *     reduce_ss and the ring engine are PICI_F32 only (PICI_ERR_DTYPE otherwise).
 *   - Return value: PICI_OK (0) or a negative PICI_ERR_* code; pici_strerror() names it.  No call
 *     throws, aborts or prints.
 *   - Gating: calls that take `d_gate` run only if d_gate == NULL or *d_gate == gate_value when the
 *     kernel starts (read on the device, no host sync); otherwise they leave every output untouched.
 *     This is how the ring driver takes format decisions without reading flags back
 *     (SURVEY.md S7 hard part 6).
 */
#ifndef PICI_H_
#define PICI_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PICI_VERSION 100

enum { PICI_F32 = 0, PICI_BF16 = 1 };

enum {
    PICI_OK = 0,
    PICI_ERR_INVALID_ARG = -1, /* NULL pointer where one is required, n >= 2^32, bad flag          */
    PICI_ERR_DTYPE       = -2, /* unknown dtype, or dtype not supported by this call               */
    PICI_ERR_ALIGN       = -3, /* a pointer violates the alignment rule above                      */
    PICI_ERR_CAPACITY    = -4, /* A_capacity / Ao_capacity < n                                     */
    PICI_ERR_WORKSPACE   = -5, /* ws_bytes < pici_sizes(..).workspace_bytes                        */
    PICI_ERR_CUDA        = -6  /* a CUDA runtime call or the launch failed (cudaGetLastError)      */
};

/* Message formats used by the ring entry points (the paper's per-message header carries the same
 * fact). */
enum { PICI_FMT_PICI = 0, PICI_FMT_DENSE = 1 };

int         pici_version(void);
const char *pici_strerror(int code);

/* Sizes for an n-element buffer: number of B words (64*T), I entries (T+1), the required A capacity
 * in ELEMENTS (n) and the scratch bytes compress / reduce_ss / nnz_dense need.  Any output pointer
 * may be NULL.  Host-only, no CUDA call. */
int pici_sizes(uint64_t n, int dtype, uint64_t *bitvec_words, uint64_t *index_entries,
               uint64_t *values_capacity, uint64_t *workspace_bytes);

/* Clears a workspace of ws_bytes bytes (one cudaMemsetAsync on `stream`).  Required once per
 * allocation before the first pici_compress / pici_reduce_ss that uses it (see "ws" above). */
int pici_workspace_init(void *ws, uint64_t ws_bytes, void *stream);

/* a1-a3. Compress (Algorithm 1): dense[n] -> (B, I, A) in ONE pass over `dense`:
 * mask words + tile counts (Phase 1), a device-wide exclusive scan of the tile counts taken by a scan service inside
 * the same launch over the counts the compressing warps publish (Phase 2; the paper scans block-locally per segment,
 * here I is one global prefix, reading C9 #3), compaction staged through shared memory (Phase 3).
 * Reads dense; writes all 64*T words of B, all T+1 entries of I and A[0 .. nnz).  ws is scratch. */
int pici_compress(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                  uint64_t A_capacity, void *ws, uint64_t ws_bytes, void *stream);

/* a4. Decompress: (B, I, A) -> dense_out[n].  EVERY element of dense_out is written
 * (absent elements become +0.0). */
int pici_decompress(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                    void *dense_out, void *stream);

/* a5. reduce_sd, the scatter-add "decompression" used by reduce-scatter / all-reduce
 * (PAPER.md:193, 219): dense_inout[i] = dense_inout[i] + a_i for every set bit, one fp32 add each;
 * all other elements are left untouched (bit-exact, a -0.0 there survives).  fp32 or bf16 (see "dtype"). */
int pici_reduce_sd(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                   void *dense_inout, void *stream);

/* a6. reduce_ss, sparse + sparse merge: O = compress(decompress(X) + decompress(Y)) without
 * materialising a dense buffer - the fused form of the paper's "scatter-add into dense, then
 * recompress" ring step.  o_i = x_i + y_i (an absent operand reads as +0.0) for every
 * position where X or Y has its bit set; the predicate is RE-APPLIED to the sum, so an exact
 * cancellation is not stored.  Outputs must not alias inputs.  fp32 only. */
int pici_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax,
                   const uint64_t *By, const uint32_t *Iy, const void *Ay, uint64_t n, int dtype,
                   uint64_t *Bo, uint32_t *Io, void *Ao, uint64_t Ao_capacity,
                   void *ws, uint64_t ws_bytes, void *stream);

/* a7. nnz of a Pici buffer = I[T], copied to *d_nnz on the device. */
int pici_nnz(const uint32_t *I, uint64_t n, uint32_t *d_nnz, void *stream);

/* a7'. nnz of a dense buffer: *d_nnz = #{ i : nz(dense[i]) } (the measurement the paper lacks after
 * a scatter-add).  ws needs 0 bytes today; pass what pici_sizes() reports. */
int pici_nnz_dense(const void *dense, uint64_t n, int dtype, uint32_t *d_nnz, void *ws,
                   uint64_t ws_bytes, void *stream);

/* a8. maybe_densify: the sparse -> dense switch "when sparsity sigma is <= tau",
 * taken ON THE DEVICE on the measured nnz as an integer compare (readings C9 #9/#10):
 *   switched = (I[T] >= nnz_switch);  *d_switched = switched (int32 0/1, always written);
 *   if switched: dense_out[n] = decompress(B, I, A); else dense_out is untouched.
 * dense_out may be NULL: then only the flag is written (the caller already holds the dense data). */
int pici_maybe_densify(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                       uint64_t nnz_switch, void *dense_out, int32_t *d_switched, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Device-gated forms used by the host ring driver (a9).  Same arithmetic as above.
 * ---------------------------------------------------------------------------------------------- */

/* compress that runs only if *d_gate == gate_value (see "Gating"). */
int pici_compress_gated(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                        uint64_t A_capacity, void *ws, uint64_t ws_bytes, const int32_t *d_gate,
                        int32_t gate_value, void *stream);

/* reduce_ss that runs only if *d_gate == gate_value (see "Gating"). */
int pici_reduce_ss_gated(const uint64_t *Bx, const uint32_t *Ix, const void *Ax,
                         const uint64_t *By, const uint32_t *Iy, const void *Ay, uint64_t n, int dtype,
                         uint64_t *Bo, uint32_t *Io, void *Ao, uint64_t Ao_capacity,
                         void *ws, uint64_t ws_bytes, const int32_t *d_gate, int32_t gate_value,
                         void *stream);

/* maybe_densify that runs only if *d_gate == gate_value; *d_fmt_out = PICI_FMT_DENSE if switched
 * else PICI_FMT_PICI.  When the gate is closed *d_fmt_out is left untouched.  d_fmt_out must not be
 * the gate word itself (PICI_ERR_INVALID_ARG). */
int pici_maybe_densify_gated(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                             uint64_t nnz_switch, void *dense_out, int32_t *d_fmt_out,
                             const int32_t *d_gate, int32_t gate_value, void *stream);

/* out[i] = recv[i] + local[i], fp32 or bf16 (the dense ring step once a chunk has switched, the paper's
 * reduceCopy).  Runs only if the gate is open; then also sets *d_fmt_out (if not
 * NULL) to PICI_FMT_DENSE.  out may alias recv or local. */
int pici_dense_add_gated(const void *recv, const void *local, uint64_t n, int dtype, void *out,
                         int32_t *d_fmt_out, const int32_t *d_gate, int32_t gate_value, void *stream);

/* out[i] = local[i] + (bit_i ? a_i : nothing): reduce_sd with a separate output (the last
 * reduce-scatter step writes the rank's result buffer).  out may alias local (then == reduce_sd).
 * Runs only if the gate is open. */
int pici_reduce_sd_out_gated(const uint64_t *B, const uint32_t *I, const void *A, const void *local,
                             uint64_t n, int dtype, void *out, const int32_t *d_gate,
                             int32_t gate_value, void *stream);

/* dst[i] = src[i] (bit copy of n elements) if the gate is open: a DENSE message landing in its
 * all-gather slot.  src and dst must not overlap. */
int pici_dense_copy_gated(const void *src, void *dst, uint64_t n, int dtype, const int32_t *d_gate,
                          int32_t gate_value, void *stream);

/* decompress that runs only if the gate is open. */
int pici_decompress_gated(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                          void *dense_out, const int32_t *d_gate, int32_t gate_value, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Ring engine (a9): SpCCL's sparse ring collectives (PAPER.md:207 all-gather; 219 reduce-scatter and
 * all-reduce = RS + AG; 227-247 the dense switch and the adaptive policy) over P LOGICAL ranks whose buffers
 * all live in this GPU's memory - no NCCL, no inter-GPU traffic; a "send" is a pointer hand-off inside the
 * arena.  Schedule (NCCL's): rank r sends to r + 1 and ends owning chunk r.
 * A call enqueues the WHOLE collective on `stream` and returns: one launch per kernel family per ring step
 * (every launch handles all P ranks), every format decision taken on the device.  fp32 only.
 *
 * X / shards / out are HOST arrays of P DEVICE pointers (16-byte aligned):
 *   reduce_scatter: X[r] = rank r's P*chunk elements; out[r] = chunk elements (reduced chunk r).
 *   all_gather:     shards[r] = chunk elements;       out[r] = P*chunk elements, identical on every rank.
 *   all_reduce:     X[r] = P*chunk elements;          out[r] = P*chunk elements.
 * Sums are taken in ring order, acc = received + local: out_c = ((X_{c+1}[c] + X_{c+2}[c]) + ...) + X_c[c].
 * arena: device scratch of pici_ring_arena_bytes() bytes, 256-byte aligned, cleared ONCE after allocation
 * (pici_workspace_init) and then reusable by any number of collectives of the same config on one stream.
 * It also holds the log: per message a format word, the measured nnz (0xFFFFFFFF for a dense send, for which
 * no count is computed) and, in policy mode, the sparsity the decision was taken on (pici_ring_layout()).
 * h_launches (host, may be NULL) receives the number of kernel launches enqueued.
 * Errors: PICI_ERR_INVALID_ARG (NULL, ranks outside 2..16, chunk not a positive multiple of 4096 or >= 2^32,
 * unknown strategy / decision), PICI_ERR_ALIGN, PICI_ERR_WORKSPACE (arena too small), PICI_ERR_CUDA.
 * ---------------------------------------------------------------------------------------------- */
enum { PICI_RING_FUSED = 0,  /* RS step = compress local chunk + sparse+sparse merge (pici_reduce_ss)          */
       PICI_RING_PAPER = 1   /* RS step = scatter-add into dense + recompress, as PAPER.md:219 has it           */ };
enum { PICI_RING_DECIDE_MEASURED = 0, /* dense once the measured nnz >= nnz_switch (readings C9 #9/#10)        */
       PICI_RING_DECIDE_POLICY = 1    /* the paper's policy: Eq. 7 extrapolation, intra / inter / ag thresholds */ };

typedef struct pici_ring_config {
    int32_t  ranks;            /* P, 2 .. 16                                                                    */
    int32_t  strategy;         /* PICI_RING_FUSED | PICI_RING_PAPER                                             */
    int32_t  decision;         /* PICI_RING_DECIDE_MEASURED | PICI_RING_DECIDE_POLICY                           */
    int32_t  keep_messages;    /* != 0: every message keeps its own slot (tests compare them with the oracle)   */
    uint64_t chunk;            /* n: elements per chunk, a multiple of 4096                                     */
    uint64_t nnz_switch_rs;    /* MEASURED: a reduce-scatter message travels dense once nnz >= this             */
    uint64_t nnz_switch_ag;    /* MEASURED: same for the all-gather's messages (chunk + 1 = never)              */
    double   intra_thresh;     /* POLICY: dense when the decision sparsity <= threshold of the outgoing link;   */
    double   inter_thresh;     /*         0.6 / 0.5 for Pici fp32 reduce-scatter                  */
    double   ag_thresh;        /* POLICY: all-reduce's RS -> AG transition (0.1)                  */
    int32_t  ranks_per_node;   /* POLICY: ranks r with equal r / ranks_per_node share a node (intra link)       */
    int32_t  reserved;
} pici_ring_config;

typedef struct pici_ring_layout_info {   /* byte offsets into the arena */
    uint64_t records;          /* messages logged: rs_records + ranks                                            */
    uint64_t rs_records;       /* reduce-scatter: record of (step s < P-1, rank r) = s * P + r                   */
    uint64_t off_fmt;          /* int32  [records]: PICI_FMT_PICI | PICI_FMT_DENSE; all-gather step 0: rs_records + r */
    uint64_t off_nnz;          /* uint32 [records]                                                               */
    uint64_t off_sigma;        /* double [records] (policy mode)                                                 */
    uint64_t off_messages;     /* message slot k at off_messages + k * message_bytes: B at +0, I at +message_I,
                                  A at +message_A, the dense form at +message_dense                              */
    uint64_t message_bytes, message_I, message_A, message_dense;
    uint64_t off_reduced, reduced_bytes;   /* all-reduce: reduced chunk of rank r at off_reduced + r * reduced_bytes */
    uint64_t slots;            /* keep_messages: slot = record; else RS (step & 1) * P + r, AG 2 * P + r         */
} pici_ring_layout_info;

int pici_ring_arena_bytes(const pici_ring_config *cfg, uint64_t *bytes);
int pici_ring_layout(const pici_ring_config *cfg, pici_ring_layout_info *info);
int pici_ring_reduce_scatter(const pici_ring_config *cfg, const void *const *X, void *const *out, void *arena,
                             uint64_t arena_bytes, int *h_launches, void *stream);
int pici_ring_all_gather(const pici_ring_config *cfg, const void *const *shards, void *const *out, void *arena,
                         uint64_t arena_bytes, int *h_launches, void *stream);
int pici_ring_all_reduce(const pici_ring_config *cfg, const void *const *X, void *const *out, void *arena,
                         uint64_t arena_bytes, int *h_launches, void *stream);

/* Measurement aid, not part of the path: dense_inout[d_idx[i]] += 1.0f for i < m (d_idx: m DISTINCT uint32
 * indices < n on the device), one thread per index, through the same gather instruction as reduce_sd's
 * read-modify-write regime.  bench.py times it on the index set of a sparse buffer to report what the memory
 * system gives for that access pattern (the "irregular memory access" of PAPER.md:237) beside reduce_sd. */
int pici_probe_random_rmw(const uint32_t *d_idx, uint64_t m, void *dense_inout, uint64_t n, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Host-buffer forms (end-to-end path): h_* are HOST pointers (pinned for full speed), d_* device
 * scratch owned by the caller.  These DO synchronise `stream` before returning.
 * ---------------------------------------------------------------------------------------------- */

/* h_dense[n] -> host (h_B[64T], h_I[T+1], h_A[nnz]); returns nnz in *h_nnz.  Device scratch:
 * d_dense (n elements), d_B, d_I, d_A (capacity n), ws. */
int pici_compress_host(const void *h_dense, uint64_t n, int dtype, uint64_t *h_B, uint32_t *h_I,
                       void *h_A, uint64_t *h_nnz, void *d_dense, uint64_t *d_B, uint32_t *d_I,
                       void *d_A, void *ws, uint64_t ws_bytes, void *stream);

/* host (h_B, h_I, h_A[nnz]) -> h_dense_out[n]. */
int pici_decompress_host(const uint64_t *h_B, const uint32_t *h_I, const void *h_A, uint64_t nnz,
                         uint64_t n, int dtype, void *h_dense_out, uint64_t *d_B, uint32_t *d_I,
                         void *d_A, void *d_dense, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* PICI_H_ */
