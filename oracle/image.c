/* Config 4 -- gray -> 3x3 Gaussian blur -> 256-bin histogram, all integer.
 * TEST INFRASTRUCTURE (see oracle.h).  Source: BASELINE.json:configs[4]; SURVEY.md §8(c) config 4.
 *   g = (77R + 150G + 29B) >> 8                                  (C4-1 interleaved HWC RGB; C4-2 truncation)
 *   b[y][x] = ( sum_{dy,dx in -1..1} k[dy][dx] * g[clamp(y+dy)][clamp(x+dx)] ) >> 4,
 *   k = [1 2 1; 2 4 2; 1 2 1]                                     (clamp-to-edge)
 *   hist[v] = #{ (y,x) : b[y][x] == v }                           (C4-4 histogram of the blurred image)
 * C4-3: output image = [blur uint8[h*w]][hist uint32[256]]. */
#include "oracle.h"

void oracle_gray_u8(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *gray) {
    for (int64_t p = 0; p < h * w; ++p) {
        uint32_t r = rgb[3 * p + 0], g = rgb[3 * p + 1], b = rgb[3 * p + 2];
        gray[p] = (uint8_t)((77u * r + 150u * g + 29u * b) >> 8);
    }
}

static int64_t clampi(int64_t v, int64_t lo, int64_t hi) { return v < lo ? lo : (v > hi ? hi : v); }

void oracle_blur3x3_u8(const uint8_t *g, int64_t h, int64_t w, uint8_t *blur) {
    static const uint32_t k[3][3] = {{1, 2, 1}, {2, 4, 2}, {1, 2, 1}};
    for (int64_t y = 0; y < h; ++y)
        for (int64_t x = 0; x < w; ++x) {
            uint32_t acc = 0;
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int64_t yy = clampi(y + dy, 0, h - 1), xx = clampi(x + dx, 0, w - 1);
                    acc += k[dy + 1][dx + 1] * (uint32_t)g[yy * w + xx];
                }
            blur[y * w + x] = (uint8_t)(acc >> 4);
        }
}

void oracle_hist256_u8(const uint8_t *p, int64_t n, uint32_t *hist) {
    for (int v = 0; v < 256; ++v) hist[v] = 0;
    for (int64_t i = 0; i < n; ++i) hist[p[i]] += 1u;
}

void oracle_config4(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *gray_tmp, void *out) {
    uint8_t *blur = (uint8_t *)out;
    uint32_t hist[256];
    oracle_gray_u8(rgb, h, w, gray_tmp);
    oracle_blur3x3_u8(gray_tmp, h, w, blur);
    oracle_hist256_u8(blur, h * w, hist);
    /* the histogram follows the image with no padding; h*w may be any value, so copy bytewise */
    uint8_t *dst = (uint8_t *)out + h * w;
    const uint8_t *src = (const uint8_t *)hist;
    for (int i = 0; i < 1024; ++i) dst[i] = src[i];
}
