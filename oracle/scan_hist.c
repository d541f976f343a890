/* Config 0 -- inclusive prefix sum + 64-bin histogram of (value mod 64).
 * TEST INFRASTRUCTURE (see oracle.h).  Source: BASELINE.json:configs[0]; SURVEY.md §8(c) config 0.
 * Reading C0-1: the histogram is taken over the SCAN OUTPUT (hist_of_input=0); the input-valued
 * variant (hist_of_input=1) is kept for the alternative reading.  C0-3: all values >= 0, so the
 * C `%` operator is the mathematical mod. */
#include "oracle.h"
#include <string.h>

/* scan[i] = sum_{k<=i} v[k], int32 (max 4096*999 = 4,091,904: no overflow) */
void oracle_scan_i32(const int32_t *v, int64_t n, int32_t *scan) {
    int32_t acc = 0;
    for (int64_t i = 0; i < n; ++i) {
        acc += v[i];
        scan[i] = acc;
    }
}

/* hist[b] = #{ i : s[i] mod bins == b } */
void oracle_hist_mod(const int32_t *s, int64_t n, int32_t bins, uint32_t *hist) {
    for (int32_t b = 0; b < bins; ++b) hist[b] = 0;
    for (int64_t i = 0; i < n; ++i) hist[s[i] % bins] += 1u;
}

/* C0-2: output image = [scan int32[n]][hist uint32[64]] contiguous */
void oracle_config0(const int32_t *v, int64_t n, int hist_of_input, void *out) {
    int32_t *scan = (int32_t *)out;
    uint32_t *hist = (uint32_t *)((char *)out + n * (int64_t)sizeof(int32_t));
    oracle_scan_i32(v, n, scan);
    oracle_hist_mod(hist_of_input ? v : scan, n, 64, hist);
}
