/* Config 3 -- C = bf16( GELU(A*B + bias) ).
 * TEST INFRASTRUCTURE (see oracle.h).  Source: BASELINE.json:configs[3]; SURVEY.md §8(c) config 3.
 *   z[m][n] = sum_k A[m][k]*B[k][n] + bias[n]   A row-major MxK, B row-major KxN (C3-1), bias by n (C3-2)
 *   C[m][n] = bf16_rne( 0.5*z*(1 + erf(z/sqrt 2)) )   (C3-3 exact-erf GELU; C3-4 round-to-nearest-even)
 * Naive triple loop; products and accumulation in double (a bf16*bf16 product is exact in double),
 * GELU in double, one rounding at the end. */
#include "oracle.h"
#include <math.h>
#include <string.h>

double oracle_bf16_to_f64(uint16_t b) {
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/* double -> bf16, round-to-nearest-even straight from the double (no double rounding via fp32) */
uint16_t oracle_f64_to_bf16_rne(double x) {
    if (isnan(x)) return 0x7FC0;
    uint16_t sign = signbit(x) ? 0x8000 : 0;
    double a = fabs(x);
    if (a == 0.0) return sign;
    if (isinf(a)) return sign | 0x7F80;
    int e;
    double f = frexp(a, &e);            /* a = f * 2^e, f in [0.5,1) */
    int E = e - 1;                      /* a = (2f) * 2^E, 2f in [1,2) */
    if (E < -126) E = -126;             /* subnormal range: fixed quantum 2^-133 */
    /* quantum of bf16 at exponent E is 2^(E-7) */
    double q = nearbyint(ldexp(a, 7 - E));   /* default rounding mode = nearest-even; exact scaling */
    (void)f;
    /* q in [0, 256]; value = q * 2^(E-7) */
    if (q >= 256.0) { q = 128.0; E += 1; }
    if (E > 127) return sign | 0x7F80;
    uint32_t qi = (uint32_t)q;
    uint16_t bits;
    if (qi < 128) bits = (uint16_t)qi;                        /* subnormal (E == -126) or zero */
    else bits = (uint16_t)(((uint32_t)(E + 127) << 7) | (qi - 128));
    return sign | bits;
}

double oracle_gelu_erf(double z) { return 0.5 * z * (1.0 + erf(z / sqrt(2.0))); }

double oracle_gemm_z_at(const uint16_t *A, const uint16_t *B, const float *bias,
                        int64_t N, int64_t K, int64_t m, int64_t n) {
    double acc = 0.0;
    for (int64_t k = 0; k < K; ++k)
        acc += oracle_bf16_to_f64(A[m * K + k]) * oracle_bf16_to_f64(B[k * N + n]);
    return acc + (double)bias[n];
}

void oracle_config3(const uint16_t *A, const uint16_t *B, const float *bias,
                    int64_t M, int64_t N, int64_t K, uint16_t *C) {
    for (int64_t m = 0; m < M; ++m)
        for (int64_t n = 0; n < N; ++n)
            C[m * N + n] = oracle_f64_to_bf16_rne(oracle_gelu_erf(oracle_gemm_z_at(A, B, bias, N, K, m, n)));
}

void oracle_config3_sampled(const uint16_t *A, const uint16_t *B, const float *bias,
                            int64_t N, int64_t K, const int64_t *ms, const int64_t *ns,
                            int64_t count, uint16_t *c_out) {
    for (int64_t i = 0; i < count; ++i)
        c_out[i] = oracle_f64_to_bf16_rne(oracle_gelu_erf(oracle_gemm_z_at(A, B, bias, N, K, ms[i], ns[i])));
}
