/* Config 2 -- 5-point Jacobi, zero halo, ping-pong sweeps.
 * TEST INFRASTRUCTURE (see oracle.h).  Source: BASELINE.json:configs[2]; SURVEY.md §8(c) config 2.
 *   u'[i][j] = 0.2f * ((((c + w) + e) + n) + s)     (C2-1 equal weights incl. centre; C2-3 order)
 *   c=u[i][j], w=u[i][j-1], e=u[i][j+1], n=u[i-1][j], s=u[i+1][j]; outside the grid reads 0.0f
 *   (C2-2 zero halo; every grid cell is updated every sweep). */
#include "oracle.h"
#include <string.h>
#include <float.h>
#if FLT_EVAL_METHOD != 0
#error "fp32 expressions must be evaluated in fp32 (reading C2-3)"
#endif

static float at(const float *u, int64_t h, int64_t w, int64_t i, int64_t j) {
    if (i < 0 || i >= h || j < 0 || j >= w) return 0.0f;
    return u[i * w + j];
}

void oracle_jacobi5_sweep(const float *u, int64_t h, int64_t w, float *out) {
    for (int64_t i = 0; i < h; ++i)
        for (int64_t j = 0; j < w; ++j) {
            float a = at(u, h, w, i, j) + at(u, h, w, i, j - 1);   /* (c + w)           */
            float b = a + at(u, h, w, i, j + 1);                   /* ((c + w) + e)     */
            float c = b + at(u, h, w, i - 1, j);                   /* (... + n)         */
            float d = c + at(u, h, w, i + 1, j);                   /* (... + s)         */
            out[i * w + j] = 0.2f * d;
        }
}

/* `sweeps` sweeps; result in out.  tmp is caller scratch of h*w floats; u is not modified. */
void oracle_config2(const float *u, int64_t h, int64_t w, int sweeps, float *out, float *tmp) {
    if (sweeps == 0) { memcpy(out, u, (size_t)(h * w) * sizeof(float)); return; }
    /* choose the ping-pong parity so that the last sweep lands in out */
    float *dst = (sweeps & 1) ? out : tmp;
    const float *src = u;
    for (int t = 0; t < sweeps; ++t) {
        oracle_jacobi5_sweep(src, h, w, dst);
        src = dst;
        dst = (dst == out) ? tmp : out;
    }
}
