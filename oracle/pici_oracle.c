/*
 * pici_oracle.c - TEST INFRASTRUCTURE.  Plain, slow, single-threaded CPU statement of what the
 * Pici hot path computes, written from the paper (arxiv/paper_2607_04676, /root/reference/PAPER.md)
 * and from SURVEY.md S8(c).  It shares NO code with the CUDA path (paper_2607_04676_b200/csrc) and
 * neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  No blocking, fusion or reordering beyond the definitions.
 *
 * Parity status: every function below is pinned by tests/test_oracle_pins.py (library-routine
 * reduction via numpy packbits / boolean-mask compaction, worked example in tests/golden/,
 * closed forms, invariants, brute force).  Nothing here is "parity unpinned".
 *
 * Format (SIII-B):
 *   The N-element dense input is viewed as T = ceil(N/4096) row-major 64x64 "virtual" tiles.
 *   B : u64[64*T]  - word B[64*t + c] is COLUMN c of tile t; bit r (LSB = row 0; reading C9 #1,
 *                    __ffsll walks from the least-significant bit) is set iff the
 *                    element at dense index 4096*t + 64*r + c is nonzero.
 *   I : u32[T+1]   - I[t] = exclusive prefix sum of per-tile nnz; I[T] = total nnz.
 *   A : packed nonzeros ordered by tile, then column, then intra-column (row) position
 *                    (PAPER.md:112).
 *   Elements with index >= N are virtual zeros (reading C9 #4).
 *
 * Nonzero predicate (stated once for both implementations):
 *   nz(x) := (bits(x) & ~signbit) != 0   <=>  IEEE x != 0.
 *   +0.0 and -0.0 are zeros; NaN, +-Inf and subnormals are nonzero.
 */
#include <stdint.h>
#include <string.h>

#define PICI_TILE 4096u
#define PICI_SIDE 64u

static int nz_f32(uint32_t u) { return (u & 0x7FFFFFFFu) != 0u; }
static int nz_b16(uint16_t u) { return (u & 0x7FFFu) != 0u; }

static uint64_t num_tiles(uint64_t n) { return (n + PICI_TILE - 1) / PICI_TILE; }

/* ------------------------------------------------------------------------------------------
 * C2. Compress (Algorithm 1).  Column-major walk of each
 * row-major tile; values are copied bit for bit.  Returns nnz.
 * ---------------------------------------------------------------------------------------- */
uint64_t oracle_compress_f32(const uint32_t *D, uint64_t n, uint64_t *B, uint32_t *I, uint32_t *A)
{
    uint64_t T = num_tiles(n), k = 0;
    for (uint64_t t = 0; t < T; ++t) {
        I[t] = (uint32_t)k;
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = 0;
            for (uint64_t r = 0; r < PICI_SIDE; ++r) {
                uint64_t i = PICI_TILE * t + PICI_SIDE * r + c;
                if (i < n && nz_f32(D[i])) {
                    w |= (uint64_t)1 << r;
                    A[k++] = D[i];
                }
            }
            B[PICI_SIDE * t + c] = w;
        }
    }
    I[T] = (uint32_t)k;
    return k;
}

uint64_t oracle_compress_b16(const uint16_t *D, uint64_t n, uint64_t *B, uint32_t *I, uint16_t *A)
{
    uint64_t T = num_tiles(n), k = 0;
    for (uint64_t t = 0; t < T; ++t) {
        I[t] = (uint32_t)k;
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = 0;
            for (uint64_t r = 0; r < PICI_SIDE; ++r) {
                uint64_t i = PICI_TILE * t + PICI_SIDE * r + c;
                if (i < n && nz_b16(D[i])) {
                    w |= (uint64_t)1 << r;
                    A[k++] = D[i];
                }
            }
            B[PICI_SIDE * t + c] = w;
        }
    }
    I[T] = (uint32_t)k;
    return k;
}

/* ------------------------------------------------------------------------------------------
 * C3. Decompress ("essentially the same procedure as Phase 3 of compression but
 * moves values from the compacted values array into a dense buffer").  Every element of D is
 * written; absent elements become +0.  Returns the number of values consumed.
 * ---------------------------------------------------------------------------------------- */
uint64_t oracle_decompress_f32(const uint64_t *B, const uint32_t *I, const uint32_t *A, uint64_t n,
                               uint32_t *D)
{
    uint64_t T = num_tiles(n), k = 0;
    (void)I; /* the sequential walk re-derives every offset; I is checked by the pins */
    for (uint64_t i = 0; i < n; ++i) D[i] = 0u;
    for (uint64_t t = 0; t < T; ++t)
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = B[PICI_SIDE * t + c];
            for (uint64_t r = 0; r < PICI_SIDE; ++r)
                if ((w >> r) & 1u) D[PICI_TILE * t + PICI_SIDE * r + c] = A[k++];
        }
    return k;
}

uint64_t oracle_decompress_b16(const uint64_t *B, const uint32_t *I, const uint16_t *A, uint64_t n,
                               uint16_t *D)
{
    uint64_t T = num_tiles(n), k = 0;
    (void)I;
    for (uint64_t i = 0; i < n; ++i) D[i] = 0u;
    for (uint64_t t = 0; t < T; ++t)
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = B[PICI_SIDE * t + c];
            for (uint64_t r = 0; r < PICI_SIDE; ++r)
                if ((w >> r) & 1u) D[PICI_TILE * t + PICI_SIDE * r + c] = A[k++];
        }
    return k;
}

/* Same walk, but every lookup goes through I (random access by tile): used by the pins to prove
 * that I really is the per-tile offset table the paper describes. */
uint64_t oracle_decompress_via_index_f32(const uint64_t *B, const uint32_t *I, const uint32_t *A,
                                         uint64_t n, uint32_t *D)
{
    uint64_t T = num_tiles(n), used = 0;
    for (uint64_t i = 0; i < n; ++i) D[i] = 0u;
    for (uint64_t tt = T; tt-- > 0;) { /* tiles visited in REVERSE: only I makes this possible */
        uint64_t k = I[tt];
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = B[PICI_SIDE * tt + c];
            for (uint64_t r = 0; r < PICI_SIDE; ++r)
                if ((w >> r) & 1u) { D[PICI_TILE * tt + PICI_SIDE * r + c] = A[k++]; ++used; }
        }
    }
    return used;
}

/* ------------------------------------------------------------------------------------------
 * C4. reduce_sd: scatter-add "decompression".  D[i] = D[i] + a for every set
 * bit, in fp32; all other elements untouched.
 * ---------------------------------------------------------------------------------------- */
uint64_t oracle_reduce_sd_f32(const uint64_t *B, const uint32_t *I, const float *A, uint64_t n,
                              float *D)
{
    uint64_t T = num_tiles(n), k = 0;
    (void)I;
    for (uint64_t t = 0; t < T; ++t)
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = B[PICI_SIDE * t + c];
            for (uint64_t r = 0; r < PICI_SIDE; ++r)
                if ((w >> r) & 1u) {
                    uint64_t i = PICI_TILE * t + PICI_SIDE * r + c;
                    volatile float s = D[i] + A[k++]; /* one fp32 add, no contraction */
                    D[i] = s;
                }
        }
    return k;
}

/* ------------------------------------------------------------------------------------------
 * C5. reduce_ss: O = compress(decompress(X) + decompress(Y)) - the paper's "accumulate into a
 * dense buffer using our Pici scatter-add kernel ... this accumulated dense buffer must be
 * recompressed" written out as its definition.  The predicate is re-applied to the
 * sum, so exact cancellation x + (-x) is NOT stored (reading C9 #6).  `scratch` holds 2*n floats.
 * Returns nnz of O.
 * ---------------------------------------------------------------------------------------- */
uint64_t oracle_reduce_ss_f32(const uint64_t *Bx, const uint32_t *Ix, const uint32_t *Ax,
                              const uint64_t *By, const uint32_t *Iy, const uint32_t *Ay, uint64_t n,
                              uint64_t *Bo, uint32_t *Io, uint32_t *Ao, float *scratch)
{
    float *dx = scratch, *dy = scratch + n;
    oracle_decompress_f32(Bx, Ix, Ax, n, (uint32_t *)dx);
    oracle_decompress_f32(By, Iy, Ay, n, (uint32_t *)dy);
    for (uint64_t i = 0; i < n; ++i) {
        volatile float s = dx[i] + dy[i]; /* acc = received + local (C9 #7) */
        dx[i] = s;
    }
    return oracle_compress_f32((const uint32_t *)dx, n, Bo, Io, Ao);
}

/* ------------------------------------------------------------------------------------------
 * C6. nnz.  Pici: the trailing entry of I.  Dense: count of nz(D[i]).
 * ---------------------------------------------------------------------------------------- */
uint64_t oracle_nnz_pici(const uint32_t *I, uint64_t n) { return I[num_tiles(n)]; }

uint64_t oracle_nnz_dense_f32(const uint32_t *D, uint64_t n)
{
    uint64_t k = 0;
    for (uint64_t i = 0; i < n; ++i) k += (uint64_t)nz_f32(D[i]);
    return k;
}

uint64_t oracle_nnz_dense_b16(const uint16_t *D, uint64_t n)
{
    uint64_t k = 0;
    for (uint64_t i = 0; i < n; ++i) k += (uint64_t)nz_b16(D[i]);
    return k;
}

/* ------------------------------------------------------------------------------------------
 * C7. maybe_densify: "switches to communicating a dense representation when sparsity sigma is
 * <= tau", taken on the MEASURED nnz as an integer compare (readings C9 #9, #10):
 * switched = (nnz >= nnz_switch); if switched, decompress into dense_out.  Returns switched.
 * ---------------------------------------------------------------------------------------- */
int oracle_maybe_densify_f32(const uint64_t *B, const uint32_t *I, const uint32_t *A, uint64_t n,
                             uint64_t nnz_switch, uint32_t *dense_out)
{
    int switched = (uint64_t)I[num_tiles(n)] >= nnz_switch;
    if (switched) oracle_decompress_f32(B, I, A, n, dense_out);
    return switched;
}

/* Dense + dense fp32 add used by the ring once a chunk has switched to dense: acc = recv + local. */
void oracle_dense_add_f32(const float *recv, const float *local, uint64_t n, float *out)
{
    for (uint64_t i = 0; i < n; ++i) {
        volatile float s = recv[i] + local[i];
        out[i] = s;
    }
}

/* ------------------------------------------------------------------------------------------
 * bf16 reductions (SURVEY.md S8(b) "bf16 reductions are optional: add in fp32, round-to-nearest-even"; reading
 * DESIGN.md S2 #24): both operands are widened to fp32 exactly (a bf16 is the high half of an fp32), added with
 * ONE fp32 rounding, and the sum is rounded to bf16 to nearest, ties to even; a NaN sum becomes a quiet NaN that
 * keeps the sum's sign and high payload bits.  Pinned by torch's bf16 addition in tests/test_oracle_pins.py.
 * ---------------------------------------------------------------------------------------- */
static float b16_to_f32(uint16_t h)
{
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

static uint16_t f32_to_b16_rne(float f)
{
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x0040u); /* NaN stays NaN */
    return (uint16_t)((u + 0x7FFFu + ((u >> 16) & 1u)) >> 16);
}

static uint16_t add_b16(uint16_t a, uint16_t b)
{
    volatile float s = b16_to_f32(a) + b16_to_f32(b);
    return f32_to_b16_rne(s);
}

/* C4 for bf16: D[i] = bf16(D[i] + a) on set bits, everything else untouched. */
uint64_t oracle_reduce_sd_b16(const uint64_t *B, const uint32_t *I, const uint16_t *A, uint64_t n, uint16_t *D)
{
    uint64_t T = num_tiles(n), k = 0;
    (void)I;
    for (uint64_t t = 0; t < T; ++t)
        for (uint64_t c = 0; c < PICI_SIDE; ++c) {
            uint64_t w = B[PICI_SIDE * t + c];
            for (uint64_t r = 0; r < PICI_SIDE; ++r)
                if ((w >> r) & 1u) {
                    uint64_t i = PICI_TILE * t + PICI_SIDE * r + c;
                    D[i] = add_b16(D[i], A[k++]);
                }
        }
    return k;
}

void oracle_dense_add_b16(const uint16_t *recv, const uint16_t *local, uint64_t n, uint16_t *out)
{
    for (uint64_t i = 0; i < n; ++i) out[i] = add_b16(recv[i], local[i]);
}
