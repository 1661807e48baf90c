/*
 * prune_oracle.c - TEST INFRASTRUCTURE.  Plain single-threaded CPU statement of the upstream workload step of the
 * paper's case study (SVI-B): "gradient pruning using a sampling-based top-k approach, imposing
 * 99% collective input sparsity and determining the pruning threshold by sampling 0.1% of gradients.  We further
 * implement a leaky error feedback (EF) mechanism".  Shares NO code with the CUDA path; only tests/, smoke() and
 * bench.py's CPU legs may call it.
 *
 * The paper gives the recipe in those two sentences only; the readings taken (S2 #20-#24):
 *   acc_i  = g_i + leak * e_i          fp32, TWO roundings (the product, then the sum; no fused multiply-add);
 *                                      e is the residual carried from the previous iteration, leak in [0, 1]
 *                                      ("leaky": the residual decays; leak = 1 is plain error feedback);
 *   sample : m caller-chosen positions s_0 .. s_{m-1} (the paper: 0.1 % of the gradient; which ones is the caller's
 *            seeded draw, an INPUT here - the method's random numbers are passed in);
 *   tau    = the k-th largest of |acc_{s_j}| (k >= 1; the paper keeps 1 %: k = ceil(0.01 m)), an exact selection;
 *   sent_i = acc_i  if |acc_i| >= tau  else +0.0     (IEEE compare: a NaN is never sent);
 *   e'_i   = +0.0   if sent            else acc_i     (what was not sent is remembered);
 *   the message is Pici(sent) (pici_oracle.c's compress on the sent buffer).
 *
 * Parity status: pinned by tests/test_oracle_prune.py (numpy sort / partition, sent + e' == acc, leak = 0 and
 * leak = 1 special cases, a hand-worked example in tests/golden/prune_example_n12.txt, kept fraction ~ k / m).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static float acc_of(float g, float e, float leak)
{
    volatile float t = leak * e;   /* rounded product */
    volatile float a = g + t;      /* rounded sum */
    return a;
}

static int cmp_desc(const void *a, const void *b)
{
    float x = *(const float *)a, y = *(const float *)b;
    return (x < y) - (x > y);
}

/* tau = k-th largest |acc| over the sample (1 <= k <= m).  A NaN magnitude sorts as +inf would not: it is replaced by
 * +inf first (a NaN in the sample counts as "large", so that it cannot make the selection undefined). */
float oracle_prune_threshold_f32(const float *g, const float *e, uint64_t n, float leak, const uint32_t *sample,
                                 uint64_t m, uint64_t k, float *scratch /* m floats */)
{
    (void)n;
    for (uint64_t j = 0; j < m; ++j) {
        float a = fabsf(acc_of(g[sample[j]], e[sample[j]], leak));
        scratch[j] = isnan(a) ? INFINITY : a;
    }
    qsort(scratch, m, sizeof(float), cmp_desc);
    return scratch[k - 1];
}

/* sent / e' from acc and tau; returns the number of elements sent (incl. zeros that pass tau = 0). */
uint64_t oracle_prune_ef_f32(const float *g, const float *e, uint64_t n, float leak, float tau, float *sent,
                             float *e_out)
{
    uint64_t c = 0;
    for (uint64_t i = 0; i < n; ++i) {
        float a = acc_of(g[i], e[i], leak);
        if (fabsf(a) >= tau) {
            sent[i] = a;
            e_out[i] = 0.0f;
            ++c;
        } else {
            sent[i] = 0.0f;
            e_out[i] = a;
        }
    }
    return c;
}
