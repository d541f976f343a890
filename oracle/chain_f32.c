/* Config 1 -- chain of four elementwise fp32 stages and a sum.
 * TEST INFRASTRUCTURE (see oracle.h).  Source: BASELINE.json:configs[1]; SURVEY.md §8(c) config 1.
 *   t1 = fl(fl(2.5f*x) + 0.1f)   (C1-1: no FMA contraction; build with -ffp-contract=off)
 *   t2 = fl(t1 + bias)           (C1-4: bias is a per-job vector of n fp32)
 *   t3 = max(t2, 0)
 *   t4 = fl(t3*t3)
 *   out = fl32( sum_i (double) t4[i] )   (C1-2: accumulate in double, round once) */
#include "oracle.h"
#include <float.h>
#if FLT_EVAL_METHOD != 0
#error "fp32 expressions must be evaluated in fp32 (reading C1-1)"
#endif

float oracle_config1(const float *x, const float *bias, int64_t n, float *t4_out) {
    double acc = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        float m = 2.5f * x[i];               /* each line is one correctly rounded fp32 operation */
        float t1 = m + 0.1f;
        float t2 = t1 + bias[i];
        float t3 = t2 > 0.0f ? t2 : 0.0f;
        float t4 = t3 * t3;
        if (t4_out) t4_out[i] = t4;
        acc += (double)t4;
    }
    return (float)acc;
}

/* The same chain with every intermediate written out (any of t1..t4 may be NULL): what the GPU's four elementwise
 * kernels K3..K6 must reproduce bit for bit, one kernel per line (reading C1-1: every line is one correctly rounded
 * fp32 operation; reading C1-5: the stages stay unfused).  Same statements as oracle_config1, no sum. */
void oracle_config1_chain(const float *x, const float *bias, int64_t n, float *t1_out, float *t2_out, float *t3_out,
                          float *t4_out) {
    for (int64_t i = 0; i < n; ++i) {
        float m = 2.5f * x[i];
        float t1 = m + 0.1f;
        float t2 = t1 + bias[i];
        float t3 = t2 > 0.0f ? t2 : 0.0f;
        float t4 = t3 * t3;
        if (t1_out) t1_out[i] = t1;
        if (t2_out) t2_out[i] = t2;
        if (t3_out) t3_out[i] = t3;
        if (t4_out) t4_out[i] = t4;
    }
}
