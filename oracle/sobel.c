/* Config 6 -- five-stage Sobel chain on an RGB frame.
 * TEST INFRASTRUCTURE (see oracle.h).  Source: PAPER.md:215 (section 5.1, workload 1: "applies normalization, edge
 * detection, mean filtering, binary thresholding, and blending operation to input images"); SURVEY.md 8(f)4.  The paper
 * gives no arithmetic; readings S6-1..S6-6 in DESIGN.md section 2, all integer, all bit-exact:
 *   S6-1  normalization   n = (77 R + 150 G + 29 B) >> 8          (three channels to one intensity in [0, 255]; config 4's gray)
 *   S6-2  edge detection  e = min(255, |gx| + |gy|), gx = [-1 0 1; -2 0 2; -1 0 1] * n, gy = its transpose, clamp-to-edge
 *   S6-3  mean filter     m = (sum of the 3 x 3 neighbourhood of e, clamp-to-edge) / 9, integer division
 *   S6-4  threshold       t = m >= 64 ? 255 : 0
 *   S6-5  blend           out = (128 t + 128 n) >> 8              (edge mask over the normalised image, alpha = 1/2)
 *   S6-6  pixel layout as config 4 (interleaved HWC RGB, tight pitch); the job's output is `out`, uint8[h][w] */
#include "oracle.h"

static int64_t clampi(int64_t v, int64_t lo, int64_t hi) { return v < lo ? lo : (v > hi ? hi : v); }

void oracle_sobel_u8(const uint8_t *n, int64_t h, int64_t w, uint8_t *e) {
    static const int kx[3][3] = {{-1, 0, 1}, {-2, 0, 2}, {-1, 0, 1}};
    for (int64_t y = 0; y < h; ++y)
        for (int64_t x = 0; x < w; ++x) {
            int gx = 0, gy = 0;
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int p = n[clampi(y + dy, 0, h - 1) * w + clampi(x + dx, 0, w - 1)];
                    gx += kx[dy + 1][dx + 1] * p;
                    gy += kx[dx + 1][dy + 1] * p;
                }
            int mag = (gx < 0 ? -gx : gx) + (gy < 0 ? -gy : gy);
            e[y * w + x] = (uint8_t)(mag > 255 ? 255 : mag);
        }
}

void oracle_mean3x3_u8(const uint8_t *e, int64_t h, int64_t w, uint8_t *m) {
    for (int64_t y = 0; y < h; ++y)
        for (int64_t x = 0; x < w; ++x) {
            int s = 0;
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) s += e[clampi(y + dy, 0, h - 1) * w + clampi(x + dx, 0, w - 1)];
            m[y * w + x] = (uint8_t)(s / 9);
        }
}

void oracle_threshold_u8(const uint8_t *m, int64_t n, int32_t thresh, uint8_t *t) {
    for (int64_t i = 0; i < n; ++i) t[i] = m[i] >= thresh ? 255 : 0;
}

void oracle_blend_u8(const uint8_t *t, const uint8_t *n, int64_t count, uint8_t *out) {
    for (int64_t i = 0; i < count; ++i) out[i] = (uint8_t)((128 * (int)t[i] + 128 * (int)n[i]) >> 8);
}

/* whole chain; tmp: 3 * h * w bytes of scratch */
void oracle_sobel_chain(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *tmp, uint8_t *out) {
    uint8_t *n = tmp, *a = tmp + h * w, *b = tmp + 2 * h * w;
    oracle_gray_u8(rgb, h, w, n);
    oracle_sobel_u8(n, h, w, a);
    oracle_mean3x3_u8(a, h, w, b);
    oracle_threshold_u8(b, h * w, 64, a);
    oracle_blend_u8(a, n, h * w, out);
}
