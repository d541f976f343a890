/* set_trace.h -- C ABI of libsettrace: device-timeline gaps of a SET run from CUPTI activity records.
 *
 * What it measures (SURVEY.md §8(d) "Gaps"; BASELINE.json:metric "mean inter-kernel gap us"):
 * the paper's motivation is the idle "white space" between kernels on the device timeline
 * and its overhead fraction  t_schedule / T  (Eq. 1).
 * For overlapped multi-stream runs Eq. 1's single-batch form does not apply (reading S12), so
 *     t_schedule = T - |union over all streams of the device activity intervals|.
 *
 * Tracing costs throughput (CUPTI serialises part of the launch path), so bench.py times jobs/s WITHOUT
 * this library loaded and measures gaps in a second pass.  libset.so does not depend on this library.
 *
 * Environment: SET_TRACE_DUMP=<file> makes set_trace_stop append one CSV line per activity record
 * (stream, job, kind, start_ns, end_ns, kernel name) before reducing them.
 *
 * All pointers are HOST.  Calls are single-caller.  Return 0 on success, negative on failure
 * (text in set_trace_error()).  The library never aborts.
 */
#ifndef SET_TRACE_H
#define SET_TRACE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Records are grouped into JOBS by the correlation id of their cudaGraphLaunch (CUPTI gives the parallel branches of a job
 * graph stream ids of their own, so the id is no guide to which work stream an operation belongs to); a job's work stream
 * is the id most of its kernels ran under.  Gaps are in microseconds. */
typedef struct set_gap_summary {
    uint64_t count;
    double mean_us, p50_us, p99_us, max_us;
} set_gap_summary;

typedef struct set_trace_stats {
    uint64_t kernels;          /* kernel records (completion-signal kernels included)                  */
    uint64_t signal_kernels;   /* of those, set_k_signal (SET_CB_FLAG_POLL's one-thread end node)      */
    uint64_t memcpys, memsets;
    uint64_t streams;          /* distinct work streams (see above)                                    */
    uint64_t dropped;          /* records CUPTI reported as dropped                                    */
    uint64_t jobs;             /* distinct correlation ids                                             */
    uint64_t kernel_kernel_overlapped; /* kernel_kernel gaps that are negative (PDL overlap)           */
    double wall_us;            /* T: last end - first start over all records                           */
    double busy_us;            /* |union of activity intervals| over all streams                       */
    double idle_frac;          /* t_schedule / T = 1 - busy/wall                                       */
    double kernel_mean_us;     /* mean duration of the stage kernels (signal kernels excluded)         */
    double sum_op_us;          /* sum of all op durations (> busy_us when streams overlap)             */
    set_gap_summary kernel_kernel; /* stage kernel -> next stage kernel of the SAME job with no copy or memset between them,
                                      start(next) - end(previous), SIGNED: negative when a programmatic edge lets the next
                                      kernel start early.  The "inter-kernel gap" of BASELINE.json:metric.              */
    set_gap_summary intra_job; /* consecutive ops of ONE job in start order: start(next) - latest end so far, >= 0      */
    set_gap_summary inter_job; /* end of a job (its last op) -> start of the next job on the same work stream, >= 0     */
    set_gap_summary any_op;    /* every consecutive pair under one CUPTI stream id, >= 0 (the raw view)                 */
} set_trace_stats;

/* Enable kernel / memcpy / memset activity collection for the process.  Records accumulate in host
 * memory until set_trace_stop.  Call with the device idle. */
int set_trace_start(void);
/* Flush, disable collection, reduce the records to *out and discard them.  Synchronise the device first. */
int set_trace_stop(set_trace_stats *out);
/* Reduce a caller-supplied timeline instead (host-only; used by the CPU tests of the reduction):
 * n records of {stream, job (correlation), kind 0=kernel 1=signal kernel 2=memcpy 3=memset, start_ns, end_ns}. */
typedef struct set_trace_rec {
    uint32_t stream, job, kind, reserved;
    uint64_t start_ns, end_ns;
} set_trace_rec;
int set_trace_reduce(const set_trace_rec *recs, uint64_t n, set_trace_stats *out);
const char *set_trace_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SET_TRACE_H */
