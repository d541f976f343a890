/* oracle.h -- CPU oracle for the SET workloads (configs 0-4 of BASELINE.json and the two paper workloads 5, 6).  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with the CUDA path (paper_2606_05495_b200/csrc) and neither
 * includes the other.
 *
 * What the method computes (SURVEY.md §8(c) "Plain definition"): SET (§4, lines 96-203)
 * is a scheduler; its numerical result is exactly out_j = F(in_j) for every submitted job j,
 * independent of stream, slot, stealing or completion order ("preserving per-job
 * ordering and memory safety").  The oracle is therefore the serial loop
 *     for j: out_j = F_cpu(in_j)
 * with F the stage chain of the workload.  The paper is silent on the workloads' arithmetic
 * (PAPER.md:215-220 give one sentence each); F follows BASELINE.json:configs[i] under the
 * readings C0-1 .. C4-5 listed in DESIGN.md §"Readings".
 *
 * Plain single-threaded C, compiled with -O2 -ffp-contract=off (reading C1-1: no FMA
 * contraction).  Every function below is pinned by tests/test_oracle_pins.py.
 */
#ifndef SET_ORACLE_H
#define SET_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* config 0 (BASELINE.json:configs[0]; readings C0-1..C0-3) */
void oracle_scan_i32(const int32_t *v, int64_t n, int32_t *scan);
void oracle_hist_mod(const int32_t *s, int64_t n, int32_t bins, uint32_t *hist);
/* whole stage chain: out = [scan int32[n]][hist uint32[64]]; hist_of_input selects the C0-1 variant */
void oracle_config0(const int32_t *v, int64_t n, int hist_of_input, void *out);

/* config 1 (configs[1]; readings C1-1..C1-6).  t4 (optional, may be NULL) receives the chain before the sum */
float oracle_config1(const float *x, const float *bias, int64_t n, float *t4);
/* the chain's intermediates t1 = affine, t2 = + bias, t3 = relu, t4 = square (each may be NULL): what K3..K6 write */
void oracle_config1_chain(const float *x, const float *bias, int64_t n, float *t1, float *t2, float *t3, float *t4);

/* config 2 (configs[2]; readings C2-1..C2-4).  u, out: fp32[h][w] row-major; tmp: scratch fp32[h*w] */
void oracle_jacobi5_sweep(const float *u, int64_t h, int64_t w, float *out);
void oracle_config2(const float *u, int64_t h, int64_t w, int sweeps, float *out, float *tmp);

/* config 3 (configs[3]; readings C3-1..C3-5).  bf16 values travel as uint16 bit patterns */
double   oracle_bf16_to_f64(uint16_t b);
uint16_t oracle_f64_to_bf16_rne(double x);
double   oracle_gelu_erf(double z);
double   oracle_gemm_z_at(const uint16_t *A, const uint16_t *B, const float *bias,
                          int64_t N, int64_t K, int64_t m, int64_t n);
void     oracle_config3(const uint16_t *A, const uint16_t *B, const float *bias,
                        int64_t M, int64_t N, int64_t K, uint16_t *C);
void     oracle_config3_sampled(const uint16_t *A, const uint16_t *B, const float *bias,
                                int64_t N, int64_t K, const int64_t *ms, const int64_t *ns,
                                int64_t count, uint16_t *c_out);

/* config 4 (configs[4]; readings C4-1..C4-5).  rgb: uint8[h][w][3]; out = [blur uint8[h*w]][hist uint32[256]] */
void oracle_gray_u8(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *gray);
void oracle_blur3x3_u8(const uint8_t *g, int64_t h, int64_t w, uint8_t *blur);
void oracle_hist256_u8(const uint8_t *p, int64_t n, uint32_t *hist);
void oracle_config4(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *gray_tmp, void *out);

/* config 5: frontier Bellman-Ford SSSP (readings S5-1..S5-4).  Returns the number of synchronous rounds.
 * scratch: int32[2V] followed by 2V bytes, i.e. at least 3V int32 */
#define ORACLE_SSSP_INF 0x7fffffff
int32_t oracle_sssp_frontier_bf(const int32_t *row_ptr, const int32_t *col, const int32_t *w, int64_t V, int32_t src,
                                int32_t *dist, int32_t *scratch);
void oracle_sssp_job(const int32_t *image, int32_t *out, int32_t *scratch);

/* config 6: five-stage Sobel chain (readings S6-1..S6-6) */
void oracle_sobel_u8(const uint8_t *n, int64_t h, int64_t w, uint8_t *e);
void oracle_mean3x3_u8(const uint8_t *e, int64_t h, int64_t w, uint8_t *m);
void oracle_threshold_u8(const uint8_t *m, int64_t n, int32_t thresh, uint8_t *t);
void oracle_blend_u8(const uint8_t *t, const uint8_t *n, int64_t count, uint8_t *out);
void oracle_sobel_chain(const uint8_t *rgb, int64_t h, int64_t w, uint8_t *tmp, uint8_t *out);

#ifdef __cplusplus
}
#endif
#endif
