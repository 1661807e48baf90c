/*
 * coo_oracle.c - TEST INFRASTRUCTURE.  Plain, slow, single-threaded CPU statement of the COO variant
 * the paper uses beside Pici (SII-B: "A common variant of COO treats inputs as
 * one-dimensional, storing only a single flat index per nonzero ... COO refers to this variant ...
 * Space overhead calculations assume 32-bit indices and 32-bit values", SIV-D:
 * "compression is similar to Pici in structure (identify nonzeros, build an index for stream
 * compaction, compact nonzeros), decompression only requires reading index-value pairs").
 * It shares NO code with the CUDA path and with pici_oracle.c; only tests/, smoke() and bench.py's
 * CPU legs may call it.
 *
 * Format (readings, S2 #17-#19; the paper gives no layout beyond "index + value"):
 *   idx : u32[nnz]  flat dense index of every nonzero, ASCENDING (the order stream compaction of a
 *                   left-to-right scan produces);
 *   val : u32[nnz]  the fp32 value bits, copied bit for bit, same order (structure of arrays);
 *   nnz : count.
 *   Nonzero predicate: the same C1 as Pici, nz(x) := (bits & 0x7FFFFFFF) != 0.
 *   Size: 8 * nnz bytes (4 index + 4 value); against BV's N/8 bytes of metadata COO's 4 * nnz bytes of
 *   metadata are smaller iff nnz < N/32, i.e. above 96.875 % sparsity.
 *
 * Parity status: pinned by tests/test_oracle_coo.py (numpy.flatnonzero, the Pici oracle's dense
 * results, closed forms, a hand-merged example, brute force).  Nothing here is "parity unpinned".
 */
#include <stdint.h>

static int nz_f32(uint32_t u) { return (u & 0x7FFFFFFFu) != 0u; }

/* compress: left-to-right scan, append (i, D[i]) for every nonzero.  Returns nnz. */
uint64_t oracle_coo_compress_f32(const uint32_t *D, uint64_t n, uint32_t *idx, uint32_t *val)
{
    uint64_t k = 0;
    for (uint64_t i = 0; i < n; ++i)
        if (nz_f32(D[i])) {
            idx[k] = (uint32_t)i;
            val[k] = D[i];
            ++k;
        }
    return k;
}

/* decompress: every element written; absent elements +0.0 ("reading index-value pairs"). */
void oracle_coo_decompress_f32(const uint32_t *idx, const uint32_t *val, uint64_t nnz, uint64_t n,
                               uint32_t *D)
{
    for (uint64_t i = 0; i < n; ++i) D[i] = 0u;
    for (uint64_t k = 0; k < nnz; ++k) D[idx[k]] = val[k];
}

/* reduce_sd: the scatter-add of a COO message into the dense accumulator (the paper's reduce-scatter
 * step, with COO in Pici's place): D[idx[k]] = D[idx[k]] + val[k], one fp32 add each,
 * in the order "accumulator + received" = the commutative twin of Pici's reading C9 #7. */
void oracle_coo_reduce_sd_f32(const uint32_t *idx, const float *val, uint64_t nnz, float *D)
{
    for (uint64_t k = 0; k < nnz; ++k) {
        volatile float s = D[idx[k]] + val[k];
        D[idx[k]] = s;
    }
}

/* reduce_ss: O = compress(decompress(X) + decompress(Y)), the definition ("accumulate
 * into a dense buffer ... must be recompressed"); predicate re-applied to the sum, so an exact
 * cancellation is dropped (reading C9 #6).  scratch holds 2 * n floats.  Returns nnz of O. */
uint64_t oracle_coo_reduce_ss_f32(const uint32_t *ix, const uint32_t *vx, uint64_t nx,
                                  const uint32_t *iy, const uint32_t *vy, uint64_t ny, uint64_t n,
                                  uint32_t *io, uint32_t *vo, float *scratch)
{
    float *dx = scratch, *dy = scratch + n;
    oracle_coo_decompress_f32(ix, vx, nx, n, (uint32_t *)dx);
    oracle_coo_decompress_f32(iy, vy, ny, n, (uint32_t *)dy);
    for (uint64_t i = 0; i < n; ++i) {
        volatile float s = dx[i] + dy[i]; /* received + local */
        dx[i] = s;
    }
    return oracle_coo_compress_f32((const uint32_t *)dx, n, io, vo);
}
