/* set.h -- C ABI of libset: stream-event-triggered (SET) dispatch of CUDA-graph pipelines on one B200.
 *
 * Source of the method: arxiv/paper_2606_05495 ("SET: Stream-Event-Triggered Scheduling for Efficient
 * CUDA Graph Pipelines"), cited below as PAPER.md:<line> (+ section / algorithm).  The four main calls
 * follow the paper's statement of the problem (§4; §4.2) in the shape
 * BASELINE.json:north_star names: set_create / set_register_pipeline / set_submit / set_drain.
 *
 * A *job* is one pass  H2D copies -> stage kernels -> D2H copies  ("memcpy H2D, kernels,
 * memcpy D2H"; "Job-as-Graph") over caller-owned host memory.  Jobs are independent.
 * A *slot* is the paper's worker W_i = (stream S_i, graph executable G_i, device buffers M_i)
 * (PAPER.md:110); here slot w runs on stream  w mod num_streams  and there are max_inflight slots, so a
 * stream carries max_inflight/num_streams jobs back to back.
 *
 * Environment (read once, at set_create / set_create_ex):
 *   SET_DRIVER_LOCK=1       take one mutex around every graph update and graph launch.  Only for runs under Nsight
 *                           Compute 2025.2, whose injection library is not safe against one thread updating a graph
 *                           executable while another launches one (profiles/r1_ncu.md).  Never set for timing.
 *                           Turned on by itself when the process runs under a CUDA injection library (CUDA_INJECTION64_PATH
 *                           or an NV_NSIGHT_INJECTION_* / NV_COMPUTE_PROFILER_* variable is set); SET_DRIVER_LOCK=0 overrides.
 *   SET_COPY_MAX_BLOCKS=n   blocks of an SM copy node that READS pinned host memory (default 64 / CUDA streams, between 2 and 8:
 *                           about 512 KB in flight over all streams saturates the link; more delays the GPU's own command
 *                           fetches over the same link, DESIGN.md sections 5d and 11).
 *   SET_FUSE_SIGNAL=0       keep the completion signal a node of its own even where the job has a single SM copy-out node that
 *                           could carry it (for A/B measurements; read at set_register_pipeline).
 *   SET_FORWARD_OUT=0       turn output-address forwarding off (read at set_register_pipeline; for A/B measurements).  By default,
 *                           where a job graph has an SM copy-in node and SM copy-out nodes, the copy-in node carries the job's
 *                           host_out address into a per-slot device word and the copy-out nodes take their destination from
 *                           there, so that binding a job updates ONE graph node instead of two.
 *
 * Conventions
 *   - Plain C, opaque handle, no exceptions cross the ABI, the library never aborts the process.
 *   - Every pointer argument says HOST or DEVICE.  No torch / C++ types appear in any signature.
 *   - Every call returns set_status (0 = SET_OK, negative = error) unless stated otherwise.
 *   - Errors are sticky: after the first failure every later call on the handle (except
 *     set_last_error, set_get_stats, set_destroy) returns the same failing status, and set_drain
 *     still returns (it never hangs on a failed context).
 *   - Thread safety: set_submit* may be called from several threads at once (Algorithm 1's
 *     compare-exchange on c_next implies concurrent claimants); all other calls are
 *     single-caller and must not race with each other.
 */
#ifndef SET_H
#define SET_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct set_ctx set_ctx;
typedef int32_t set_status;

#define SET_OK            0
#define SET_ERR_INVALID  (-1) /* bad argument (NULL, out of range, malformed descriptor)          */
#define SET_ERR_CUDA     (-2) /* a CUDA runtime/driver call failed; text in set_last_error()       */
#define SET_ERR_NOMEM    (-3) /* host or device allocation failed                                  */
#define SET_ERR_STATE    (-4) /* call out of order (submit before register, register twice, ...)   */
#define SET_ERR_SIZE     (-5) /* a per-job size computed from dims exceeds a registered buffer     */
#define SET_ERR_BUSY     (-6) /* set_try_submit_dims: no executable is free right now (not an error state)   */

#define SET_MAX_STAGES  16
#define SET_MAX_BUFFERS  8
#define SET_MAX_ARGS    12
#define SET_MAX_DIMS     4

/* ------------------------------------------------------------------------------------------------
 * Size expressions: the "placeholders" of PAPER.md:102 that vary per job.
 *   value(dims) = fixed + per_unit * PROD_{i : dim_mask bit i set} dims[i]
 * dims[0..3] are the four uint32 passed to set_submit_dims (all 1 for set_submit).
 * ---------------------------------------------------------------------------------------------- */
typedef struct set_size_expr {
    uint64_t fixed;
    uint64_t per_unit;
    uint32_t dim_mask;
    uint32_t reserved;
} set_size_expr;

/* How each grid dimension of a stage is derived: grid = max(1, ceil(value(count) / divisor)). */
typedef struct set_grid_rule {
    set_size_expr count;
    uint32_t divisor; /* >= 1 */
    uint32_t reserved;
} set_grid_rule;

/* Kernel argument kinds.  Arguments are passed to the kernel in list order. */
#define SET_ARG_BUFFER  0 /* DEVICE pointer: slot buffer `index` + value(offset)                   */
#define SET_ARG_IMM32   1 /* 4-byte immediate (low 32 bits of imm)                                 */
#define SET_ARG_IMM64   2 /* 8-byte immediate                                                      */
#define SET_ARG_DIM     3 /* uint32 = dims[index] of the job                                       */
#define SET_ARG_COND    5 /* 8-byte cudaGraphConditionalHandle of the enclosing loop (SET_STAGE_LOOP_BEGIN)  */
#define SET_ARG_TMAP2D  4 /* 128-byte CUtensorMap (by value, __grid_constant__) over a 2-D row-major
                             region of slot buffer `index` starting at value(offset); see tmap     */

#define SET_SWIZZLE_NONE 0
#define SET_SWIZZLE_64B  2
#define SET_SWIZZLE_128B 3

typedef struct set_tmap2d {
    uint32_t elem_bytes;   /* 2 (bf16) or 4 (fp32) or 1                                            */
    uint32_t swizzle;      /* SET_SWIZZLE_*                                                        */
    uint64_t inner;        /* elements along the contiguous dimension                              */
    uint64_t outer;        /* rows                                                                 */
    uint64_t pitch_bytes;  /* byte stride between rows (multiple of 16)                            */
    uint32_t box_inner;    /* TMA box, elements                                                    */
    uint32_t box_outer;
} set_tmap2d;

typedef struct set_arg_desc {
    int32_t kind;          /* SET_ARG_*                                                            */
    int32_t index;         /* BUFFER/TMAP2D: buffer index; DIM: dims index                         */
    set_size_expr offset;  /* BUFFER/TMAP2D: byte offset inside the buffer                         */
    uint64_t imm;          /* IMM32 / IMM64 payload                                                */
    set_tmap2d tmap;       /* TMAP2D only                                                          */
} set_arg_desc;

#define SET_STAGE_LOOP_BEGIN 2u /* this stage is the first of a data-dependent loop: the stages from here to the next
                                   SET_STAGE_LOOP_END (inclusive) become the body of a conditional WHILE node of the job graph
                                   (a workload whose iteration count depends on the data does not fit a fixed
                                   graph).  The loop is entered unconditionally; a kernel of the body ends it by calling
                                   cudaGraphSetConditional(handle, 0) with the handle it receives as a SET_ARG_COND argument.
                                   A pipeline with a loop is bound to its slot for good (CUDA cannot re-point the nodes of a
                                   loop body one by one): the kernels of the body may not take SET_ARG_DIM arguments or dim-dependent
                                   offsets / grids (per-job sizes travel in the job's device image instead), a job is never
                                   retargeted to another slot's executable (a thief without a free executable of its own
                                   puts the job back), and SET_MODE_PLAIN_STREAMS is refused.  One loop per pipeline.
                                   The body needs at least 3 stages: a two-node body failed about once in 10^5 jobs on this
                                   driver (cudaErrorLaunchFailure, the context is lost) and is refused with SET_ERR_INVALID.
                                   In SET_MODE_SET such a pipeline runs one job at a time on each of at most 8 CUDA streams
                                   (the largest divisor of num_streams that is <= 8), whatever max_inflight and
                                   streams_per_lane say: more WHILE graphs in flight than that fail now and then on this
                                   driver, and a WHILE graph queued behind a running one slows both.      */
#define SET_STAGE_LOOP_END   4u
#define SET_STAGE_PDL 1u   /* connect this stage to the node before it (the previous stage; for the first stage,
                              an SM copy node) with a programmatic-dependent-launch edge.  By setting the flag the
                              caller asserts that the kernel executes griddepcontrol.wait before it reads or writes
                              job data; every built-in kernel does (the tcgen05 GEMM after its barrier / TMEM set-up,
                              before its first TMA load).  A kernel that also executes griddepcontrol.launch_dependents
                              early lets the NEXT node's blocks become resident while it still runs: the built-in kernels
                              with a handful of blocks do, those whose grid covers a frame do not (their dependents
                              would only sit on SM resources).  Ignored where the predecessor is a copy-engine node.  */

/* One stage = one kernel node of the job graph ("nodes are initialized with the target
 * function, input arguments, grid and block dimensions").  Stages run in list order. */
typedef struct set_stage_desc {
    const void *func;      /* HOST address of the __global__ function's host stub (what
                              cudaLaunchKernel takes), e.g. from set_builtin_kernel()              */
    set_grid_rule grid[3];
    uint32_t block[3];
    uint32_t smem_bytes;   /* dynamic shared memory                                                */
    uint32_t flags;        /* SET_STAGE_*                                                          */
    int32_t num_args;
    int32_t reserved;
    set_arg_desc args[SET_MAX_ARGS];
} set_stage_desc;

#define SET_BUF_ZERO 1u    /* zero [zero_offset, zero_offset+zero_bytes) on the device at the start
                              of every job (a memset node ahead of the first stage)                */

/* One device buffer of the slot's memory set M_w ("pre-allocated memory slots",
 * PAPER.md:110 "dedicated set of device-side buffers M_i"), plus at most one H2D and one D2H copy.
 * All H2D copies precede the first stage, all D2H copies follow the last one. */
typedef struct set_buffer_desc {
    uint64_t bytes;             /* device bytes per slot (capacity; per-job sizes must fit)        */
    uint32_t flags;             /* SET_BUF_*                                                       */
    uint32_t reserved;
    set_size_expr h2d_bytes;    /* 0 => no H2D for this buffer                                     */
    set_size_expr h2d_host_off; /* byte offset in the job's host_in                                */
    set_size_expr h2d_dev_off;  /* byte offset in this buffer                                      */
    set_size_expr d2h_bytes;    /* 0 => no D2H for this buffer                                     */
    set_size_expr d2h_host_off; /* byte offset in the job's host_out                               */
    set_size_expr d2h_dev_off;
    set_size_expr zero_off;     /* SET_BUF_ZERO range                                              */
    set_size_expr zero_bytes;
} set_buffer_desc;

/* Scheduling models.  SET is the product; the others are the in-run baselines of BASELINE.md §5 /
 * PAPER.md:224-229 and share buffers, graphs and kernels with it, not the scheduler. */
#define SET_MODE_SET           0 /* Algorithms 1-3                               */
#define SET_MODE_PLAIN_STREAMS 1 /* cudaMemcpyAsync + <<<>>> per job on stream j mod S (PAPER.md:226
                                    synchronous model, spread over the stream pool)                */
#define SET_MODE_BATCH_SYNC    2 /* static batching: b graphs on fixed streams, host sync after
                                    every batch                        */
#define SET_MODE_SINGLE_GRAPH  3 /* graph model: one exec replayed on one stream    */
#define SET_MODE_MUTEX_QUEUE   4 /* queue model: one global queue behind a mutex, O(b) completion
                                    queries by the host                */

#define SET_IO_HOST   0 /* host_in / host_out are HOST pointers (pinned: DMA'd in place; pageable:
                           staged through the library's pinned ring)                               */
#define SET_IO_DEVICE 1 /* host_in / host_out are DEVICE pointers: the copy nodes become D2D.  Used
                           to time the path with inputs already resident in HBM.                   */

#define SET_STEAL_SWAP     0 /* a stolen job is re-bound onto an exec already tied to the thief's
                                M_w (only the host pointers change)                                */
#define SET_STEAL_RETARGET 1 /* PAPER.md:122 literally: the victim's exec is retargeted to the
                                thief's buffers (every node updated) and migrates with the job     */

#define SET_CB_DEFAULT       0 /* the library's choice: SET_CB_FLAG_POLL      */
#define SET_CB_NOTIFY_STREAM 1 /* event chaining: cudaEventRecord on S_w, cudaStreamWaitEvent +
                                  cudaLaunchHostFunc on a per-stream notify stream                 */
#define SET_CB_WORK_STREAM   2 /* PAPER.md:203 literally: cudaLaunchHostFunc on S_w itself         */
#define SET_CB_FLAG_POLL     3 /* the job graph ends in a one-thread kernel node that stores a word to
                                  pinned host memory; the dispatcher thread watches the words of the
                                  in-flight slots and runs Algorithm 3 itself (no driver callback
                                  thread, no extra API call per job; measured 8x lower completion
                                  latency than cudaLaunchHostFunc on B200, profiles/)             */

#define SET_CB_HOST_NODE     4 /* the job graph ends in a host node (cudaGraphAddHostNode) that runs Algorithm 3 on the
                                  driver's callback thread: no API call per job beyond cudaGraphLaunch, but the
                                  stream waits for the host round trip like SET_CB_WORK_STREAM                */

typedef struct set_config {
    uint32_t struct_bytes;    /* = sizeof(set_config), for forward compatibility                   */
    int32_t num_streams;      /* S >= 1                                                            */
    int32_t max_inflight;     /* b >= 1: launched-but-not-completed jobs             */
    int32_t mode;             /* SET_MODE_*                                                        */
    int32_t io;               /* SET_IO_*                                                          */
    int32_t queue_capacity;   /* q >= 1 prepared jobs per slot queue Q_w; 0 => default (2)         */
    int32_t num_dispatchers;  /* dispatcher threads; 0 => default (1)                              */
    int32_t steal_policy;     /* SET_STEAL_*                                                       */
    int32_t callback_mode;    /* SET_CB_*                                                          */
    int32_t device;           /* CUDA device ordinal; -1 => current device                         */
    int32_t spin_us;          /* dispatcher/drain spin time before sleeping; 0 => default (50)     */
    int32_t sm_copy_max_bytes;/* H2D/D2H copies of up to this many bytes become kernel nodes
                                 (SET_K_COPY: the SMs read/write pinned host memory over the link) instead of
                                 copy-engine memcpy nodes; a copy whose size depends on the job's dims counts with the
                                 capacity of its buffer; 0 => default (262144), -1 => never.   */
    int32_t timestamps;       /* 1: every job graph gets two extra one-thread kernel nodes that store the GPU's
                                 %globaltimer when the graph starts (a root node beside the first copy) and when it
                                 ends (the completion-signal node, or a last node of its own): the device-side gap
                                 between consecutive jobs of a stream, measured at full speed without a profiler
                                 attached; read with set_get_gap_stats.  0 (default): no such nodes.            */
    int32_t completion_fence; /* SET_CB_FLAG_POLL: how the signal node publishes the slot's word.  SET_FENCE_DEFAULT (0) =
                                 the library's choice, SET_FENCE_SYSTEM; SET_FENCE_SYSTEM (1) = fence.acq_rel.sys before
                                 the store (release at system scope: the job's D2H output, written by an earlier grid, is
                                 ordered before the word by the PTX memory model); SET_FENCE_NONE (2) = plain volatile
                                 store, relying on grid completion alone.  UNSAFE, a measurement arm only: about 10 % faster,
                                 not guaranteed by the model, and caught on B200 with several CUDA streams per lane -- about
                                 one completion in 30,000 is seen before its output (profiles/r2_signal_soak.md).  Outputs are
                                 still complete once set_drain has returned.  DESIGN.md 5a.                          */
    void *const *streams;     /* HOST array of num_streams cudaStream_t owned by the caller (e.g.
                                 torch.cuda.Stream.cuda_stream), or NULL: the library creates them */
    void *device_arena;       /* DEVICE memory owned by the caller for all slot buffers, or NULL   */
    uint64_t device_arena_bytes;
    int32_t streams_per_lane; /* CUDA streams behind each of the num_streams logical streams ("lanes"): slot w runs on
                                 lane w mod S, CUDA stream (w / S) mod streams_per_lane of that lane, so consecutive jobs
                                 of a lane overlap (job k+1's copy-in runs beside job k's kernels and tail) instead of
                                 queueing behind each other's last node.  The paper's worker owns a stream of its own
                                 (PAPER.md:110), which is streams_per_lane = max_inflight / num_streams; larger values are
                                 clamped to that.  0 => default: with SET_IO_HOST as many as the slots allow up to 32 CUDA
                                 streams in all, with SET_IO_DEVICE 1 (DESIGN.md 5b gives the measurements).  Forced to 1
                                 when the caller supplies `streams`.  The in-run baseline models use the same streams.  */
    int32_t completion_thread;/* SET_CB_FLAG_POLL: 1 = a thread of its own watches the completion words and runs Algorithm 3, the
                                 dispatcher(s) only find and launch jobs; 2 = the dispatcher(s) poll between launches;
                                 0 => default (1 from max_inflight = 16 up: +6-10 % on config 1 end to end where the host
                                 is slow; 2 below: the hand-off costs a latency-bound config 6 %).  DESIGN.md 5d.   */
    int32_t bind_at_launch;   /* 1 = set_submit only checks the job and queues its description; the executable is updated on the
                                 dispatcher thread right before it is launched (the JIT update of PAPER.md:122 for every job), so
                                 that all driver calls of a job come from one thread; 2 = set_submit updates the executable
                                 (Algorithm 1 literally); 0 => default (2).  DESIGN.md 5d.                            */
    uint32_t debug_sentinel;  /* test hook: non-zero => at the moment a job's completion is observed (before the slot is
                                 released) the first and last 32-bit word of every D2H region of its host_out are compared
                                 with this value; a match means the completion overtook the output, counted in
                                 set_stats.early_completions.  The caller pre-fills host_out with the value.  0 = off.  */
} set_config;

#define SET_FENCE_DEFAULT 0
#define SET_FENCE_SYSTEM  1
#define SET_FENCE_NONE    2

typedef struct set_stats {
    uint64_t submitted;        /* jobs accepted by set_submit*                                     */
    uint64_t completed;        /* c_done of Algorithm 3                                            */
    uint64_t launched;         /* graph launches (or per-job launch sequences in baseline modes)   */
    uint64_t steals;           /* jobs taken from another slot's queue (Alg. 2 l.12-16)            */
    uint64_t full_rebinds;     /* exec updates that touched every node (device pointers / dims)    */
    uint64_t host_rebinds;     /* exec updates that touched only the host-pointer copy nodes       */
    uint64_t staged_jobs;      /* jobs whose pageable buffers went through the pinned ring         */
    uint64_t submit_stalls;    /* times set_submit had to wait for a free queue entry              */
    uint64_t dispatcher_sleeps;/* times a dispatcher blocked in the kernel (futex)                 */
    uint64_t kernel_nodes;     /* kernel launches issued (graph kernel nodes count once per launch)*/
    uint64_t ns_submit;        /* host ns inside set_submit* (claim + bind + push)                 */
    uint64_t ns_bind;          /* host ns inside exec parameter updates                            */
    uint64_t ns_launch;        /* host ns inside launch + event chaining                           */
    uint64_t ns_callback;      /* host ns inside completion callbacks                              */
    uint64_t ns_sync;          /* host ns blocked in batch/stream synchronisation (baselines)      */
    uint64_t max_inflight_seen;/* high-water mark of launched-not-completed jobs                   */
    uint64_t signal_nodes;     /* completion-signal kernel launches (SET_CB_FLAG_POLL: one per job)*/
    uint64_t copy_nodes;       /* SET_K_COPY kernel launches (copies done by the SMs)                 */
    uint64_t early_completions;/* set_config.debug_sentinel: jobs whose output still held the sentinel when their completion
                                  was observed (must stay 0)                                             */
    uint64_t cuda_streams;     /* CUDA streams jobs run on: num_streams * streams_per_lane, or at most 8 once a pipeline with a
                                  loop is registered (SET_STAGE_LOOP_BEGIN says why) (not a counter)     */
} set_stats;

/* ---------------------------------------------------------------------------------------------- *
 * A1  set_create -- PAPER.md:116 "Initialization": create the stream pool, b = max_inflight slots,
 * the free-worker pool W_pool holding every slot id and the per-slot job queues Q_w
 * (PAPER.md:112); spawn the dispatcher thread(s).  No device memory is allocated yet.
 *   num_streams, max_inflight : >= 1.  max_inflight is rounded up to a multiple of num_streams.
 *   out : HOST, receives the handle.  Ownership: caller, release with set_destroy.
 * Errors: SET_ERR_INVALID, SET_ERR_CUDA (no device), SET_ERR_NOMEM.  *out is NULL on failure.
 * set_create(S, b, out) == set_create_ex with mode SET, io HOST, defaults elsewhere.
 */
set_status set_create(int num_streams, int max_inflight, set_ctx **out);
set_status set_create_ex(const set_config *cfg, set_ctx **out);

/* A2  set_register_pipeline -- PAPER.md:102 (job-as-graph with placeholders), PAPER.md:104 (memory
 * slots), PAPER.md:110 (G_i bound only to M_i).  For every slot: allocate the device buffers, build
 * the DAG  [memset] -> H2D copy nodes -> kernel nodes in list order -> D2H copy nodes  by explicit
 * construction, instantiate queue_capacity+1 graph executables and bind them to the slot's buffers.
 *   stages : HOST array[num_stages], 1..SET_MAX_STAGES.  bufs : HOST array[num_bufs], 1..SET_MAX_BUFFERS.
 *   Descriptors are copied; the caller may free them on return.  Kernel images must stay loaded.
 * One pipeline per context; a second call returns SET_ERR_STATE.
 * Errors: SET_ERR_INVALID (malformed descriptor), SET_ERR_NOMEM, SET_ERR_CUDA.
 */
set_status set_register_pipeline(set_ctx *ctx, const set_stage_desc *stages, int num_stages,
                                 const set_buffer_desc *bufs, int num_bufs);

/* A3  set_submit -- Algorithm 1 and PAPER.md:118: claim the job, pick a queue with
 * a free entry starting at job ticket mod b, update the graph executable's copy nodes to host_in /
 * host_out (UpdateGraphParams) and push it to Q_i.  Blocks (back-pressure) while every queue is full.
 *   job_id   : caller's tag, reported back nowhere except stats/tracing; need not be unique.
 *   host_in  : HOST (or DEVICE under SET_IO_DEVICE), read-only to the library.  Layout = the byte image
 *              the pipeline's h2d_host_off / h2d_bytes describe.  Must stay valid and unmodified
 *              until set_drain returns.
 *   host_out : HOST (or DEVICE), written by DMA.  Contents are defined after set_drain returns SET_OK.
 *   dims     : HOST array[4] of per-job dimensions for size expressions (set_submit: all 1).
 * Pinned pointers (set_host_alloc, cudaHostAlloc, torch pin_memory) are DMA'd in place; pageable
 * pointers are copied through the library's pinned staging ring.
 * Errors: SET_ERR_STATE (no pipeline), SET_ERR_SIZE (dims overflow a buffer), sticky errors.
 */
set_status set_submit(set_ctx *ctx, uint64_t job_id, const void *host_in, void *host_out);
set_status set_submit_dims(set_ctx *ctx, uint64_t job_id, const void *host_in, void *host_out,
                           const uint32_t dims[SET_MAX_DIMS]);
/* set_submit_dims that never blocks: SET_ERR_BUSY if no executable is free right now (nothing was queued, the context is
 * unchanged and stays usable); SET_MODE_SET only (SET_ERR_STATE otherwise).  The building block of set_multi_submit_dims. */
set_status set_try_submit_dims(set_ctx *ctx, uint64_t job_id, const void *host_in, void *host_out,
                               const uint32_t dims[SET_MAX_DIMS]);
/* n submissions in one call (same semantics as n calls in order).  host_ins/host_outs: HOST arrays of
 * n pointers; dims: HOST array[n][4] or NULL; job_ids: HOST array[n] or NULL (then first_id + i). */
set_status set_submit_batch(set_ctx *ctx, int64_t n, uint64_t first_id, const uint64_t *job_ids,
                            const void *const *host_ins, void *const *host_outs, const uint32_t *dims);

/* A8  set_drain -- implied by the done counter of Algorithm 3: block until every
 * submitted job has completed (c_done == c_submitted), then surface the sticky error if any.
 * After SET_OK every host_out is fully written.  The context stays usable for more submissions. */
set_status set_drain(set_ctx *ctx);

/* Stop the dispatcher(s), drain, free every library-owned resource.  NULL is allowed. */
set_status set_destroy(set_ctx *ctx);

/* Pinned host memory from the context's allocator (cudaHostAlloc, portable).  Returns HOST pointer or
 * NULL.  Ownership: caller; release with set_host_free before set_destroy (set_destroy frees leftovers). */
void *set_host_alloc(set_ctx *ctx, size_t bytes);
void set_host_free(set_ctx *ctx, void *p);

/* Tell the library that [p, p + bytes) is pinned HOST memory the caller owns (cudaHostAlloc / cudaHostRegister / torch
 * pin_memory) so that jobs in it skip the per-job driver query.  The range is checked once (SET_ERR_INVALID if it is
 * not pinned, or if an SM copy could not dereference it on the device).  The caller must call set_host_unregister
 * before freeing or unpinning the memory: the library caches only ranges it was told about (its own set_host_alloc
 * blocks and these); any other pointer is queried at every submit. */
set_status set_host_register(set_ctx *ctx, const void *p, size_t bytes);
set_status set_host_unregister(set_ctx *ctx, const void *p);

/* Counters and per-phase host time since create (or since set_reset_stats). out: HOST. */
set_status set_get_stats(set_ctx *ctx, set_stats *out);
set_status set_reset_stats(set_ctx *ctx);

/* Device-side timing of the jobs completed since create / set_reset_stats, from the timestamp nodes of
 * set_config.timestamps = 1 (all zero otherwise).  A gap is  start(job k+1) - end(job k)  of two jobs that ran
 * one after the other on the same stream (negative differences count as 0): the idle "white space" between
 * jobs of PAPER.md:15-17 as the GPU saw it.  Collected in SET, batch-synchronous and mutex-queue modes.
 * Single caller, drained context.  out: HOST. */
typedef struct set_gap_stats {
    uint64_t jobs;          /* jobs with both timestamps                                            */
    uint64_t gaps;          /* job pairs                                                            */
    double gap_mean_us, gap_p50_us, gap_p99_us, gap_max_us;
    double job_mean_us;     /* mean of end - start of one job (its chain on the device)             */
    double span_us;         /* last end - first start over all jobs                                 */
    double stream_busy_frac;/* sum of job durations / (span * CUDA streams): how full the streams were */
    double busy_union_us;   /* |union over all streams of the jobs' [start, end] intervals|: time during which the
                               GPU had at least one job in progress                                  */
    double idle_frac;       /* 1 - busy_union_us / span_us: the timeline's white space, the
                               t_schedule / T_measured of PAPER.md:81-90, :253 under reading S12, at job granularity */
    double idle_gaps;       /* number of intervals inside the span during which NO job was in progress on any stream */
    double idle_gap_mean_us;/* their mean length: the device-wide gap between jobs (0 if there is none)             */
} set_gap_stats;
set_status set_get_gap_stats(set_ctx *ctx, set_gap_stats *out);

/* HOST, NUL-terminated text of the first error on this context ("" if none).  Valid until destroy. */
const char *set_last_error(set_ctx *ctx);

/* Number of slots b actually created, streams S, execs per slot (q+1). out_*: HOST, may be NULL. */
set_status set_get_geometry(set_ctx *ctx, int *out_slots, int *out_streams, int *out_execs_per_slot);

/* Time stage `stage` alone on slot 0's buffers and stream: a graph holding a chain of `iters` launches of the
 * stage's kernel (no host launch cost between them), run once or more for warm-up (`warmup` > 0) and then once
 * bracketed by CUDA events on that stream; dims as in set_submit_dims (NULL => all 1).  The launches are chained by
 * plain edges, or by programmatic edges if the stage was registered with SET_STAGE_PDL (what the kernel costs behind
 * another kernel of such a job graph: the next launch is already resident while this one drains).
 * out_avg_us: HOST, average microseconds per launch.  Requires a drained context. */
set_status set_time_stage(set_ctx *ctx, int stage, const uint32_t *dims, int warmup, int iters,
                          float *out_avg_us);

/* ---------------------------------------------------------------------------------------------- *
 * Built-in stage kernels (hand-written sm_100a CUDA, csrc/kernels/) and the five pipelines of
 * BASELINE.json:configs[0..4].  Operation definitions: DESIGN.md §"Stage kernels".
 */
#define SET_K_SCAN_I32        1  /* (const int32* in, int32* out, uint32 n)  inclusive prefix sum, 1 block of 1024 */
#define SET_K_HIST_MOD64      2  /* (const int32* in, uint32* hist, uint32 n) 64 bins of v mod 64, 1 block of 256 */
#define SET_K_AFFINE_F32      3  /* (const float* x, float* y, uint32 n)  y = fl(fl(2.5x)+0.1)               */
#define SET_K_ADD_BIAS_F32    4  /* (float* y, const float* bias, uint32 n)  y = fl(y + bias)                */
#define SET_K_RELU_F32        5  /* (float* y, uint32 n)  y = max(y,0)                                       */
#define SET_K_SQUARE_F32      6  /* (float* y, uint32 n)  y = fl(y*y)                                        */
#define SET_K_BLOCK_SUM_F32   7  /* (const float* y, float* out, uint32 n)  out[0] = sum, fixed tree, 1 block */
#define SET_K_JACOBI5_F32     8  /* (const float* u, float* v, uint32 h, uint32 w, uint32 flip)  one sweep, zero
                                    halo; flip = 1 walks the row blocks bottom-up (L2 reuse between sweeps)  */
#define SET_K_GEMM_BIAS_GELU  9  /* (tmapA, tmapB, tmapC, const float* bias, uint32 M, N, K)  tcgen05 + TMA   */
#define SET_K_RGB2GRAY_U8    10  /* (const uint8* rgb, uint8* gray, uint32 w, uint32 h)                      */
#define SET_K_BLUR3X3_U8     11  /* (const uint8* g, uint8* out, uint32 w, uint32 h)  clamp-to-edge          */
#define SET_K_HIST256_U8     12  /* (const uint8* p, uint32* hist, uint32 w, uint32 h)  hist must be zeroed  */
#define SET_K_SPIN           13  /* (uint32* scratch, uint32 ns)  debug delay stage (busy-waits ns)          */
#define SET_K_SIGNAL         14  /* (uint32* flag, uint64* stamp, uint32 fence)  *flag = 1 in mapped pinned HOST memory
                                    (SET_CB_FLAG_POLL), behind fence.acq_rel.sys if fence != 0; stamp != NULL:
                                    *stamp = %globaltimer first                                               */
#define SET_K_STAMP          16  /* (uint64* stamp)  *stamp = %globaltimer (set_config.timestamps)               */
#define SET_K_COPY           15  /* (const void* src, void* dst, uint32 bytes, void** fwd_slot, void* fwd_value)  copy by the
                                    SMs; src / dst may be pinned HOST or DEVICE memory; fwd_slot != NULL: also stores
                                    fwd_value (the job's output address) into that DEVICE word                */
#define SET_K_COPY_OUT       24  /* (const void* src, void* const* dst_slot, uint64 dst_off, uint32 bytes, uint32* flag,
                                    uint64* stamp, uint32 fence)  copy by the SMs to *dst_slot + dst_off: the address the
                                    job's copy-in node forwarded; flag != NULL: the block that finishes last also does what
                                    SET_K_SIGNAL does (the job's completion signal folded into its only copy-out node)   */
#define SET_K_SSSP_SOLO      25  /* (img, out, scratch, maxV)  the whole SSSP job in one block of 1024 threads: K21's
                                    initialisation, K22's relaxation round after round with a block barrier between them,
                                    the round count; distances and frontier flags in 5 maxV bytes (flags padded to a
                                    word) of DYNAMIC shared memory, scratch = work list uint32[maxV].  Launch with grid 1,
                                    block 1024; maxV <= 40000.                                                          */
/* the two paper workloads of SURVEY.md 8(f)4 (readings S5-*, S6-*) */
#define SET_K_SOBEL3X3_U8    17  /* (const uint8* n, uint8* e, uint32 w, uint32 h)  min(255, |gx| + |gy|), clamp-to-edge   */
#define SET_K_MEAN3X3_U8     18  /* (const uint8* e, uint8* m, uint32 w, uint32 h)  3 x 3 sum / 9, clamp-to-edge          */
#define SET_K_THRESHOLD_U8   19  /* (const uint8* m, uint8* t, uint32 w, uint32 h, uint32 thresh)  m >= thresh ? 255 : 0  */
#define SET_K_BLEND_U8       20  /* (const uint8* t, const uint8* n, uint8* out, uint32 w, uint32 h)  (t + n) >> 1        */
#define SET_K_SSSP_INIT      21  /* (const int32* img, int32* out, uint32* scratch, uint32 maxV)  dist = INF, dist[src] = 0,
                                    frontier = {src};  img = [V, E, src, 0][row_ptr V+1][col E][w E]               */
#define SET_K_SSSP_RELAX     22  /* (img, out, scratch, maxV, uint32 sub)  one frontier round, the sub-th of the U a pass
                                    of the loop body holds: atomicMin relaxation of every edge out of the frontier, next
                                    frontier = vertices whose distance got smaller; scratch = flags[2][maxV], ctrl[16] */
#define SET_K_SSSP_CONTROL   23  /* (img, out, scratch, maxV, uint32 U, loop handle)  counts the rounds of this pass that
                                    had a frontier and sets the condition of the enclosing WHILE node: another pass iff
                                    the pass's last round changed some distance                                      */

/* HOST address usable as set_stage_desc.func, or NULL for an unknown id. */
const void *set_builtin_kernel(int kernel_id);

/* Fill stage/buffer descriptors for BASELINE.json:configs[config] (0..4) or one of the two paper workloads (5, 6).
 *   params : HOST array of uint32 or NULL for the BASELINE sizes:
 *     config 0: {n}            config 1: {n}          config 2: {h, w, sweeps[, alternate = 1]}
 *     config 3: {M, N, K}      config 4: {max_w, max_h}  (dims per job = {w, h, 1, 1})
 *     config 5 (SSSP): {maxV, maxE[, U = 4]}  (dims per job = {E, 1, 1, 1}; V, E, src travel in the job
 *               image; U = 2..8 relaxation rounds per pass of the WHILE body, 2 + U stage kernels in all)
 *     config 6 (Sobel chain): {max_w, max_h[, thresh = 64]}  (dims per job = {w, h, 1, 1})
 *   variant: 0 = default.  config 0: 1 = histogram of the INPUT values (reading C0-1 alternative).
 *            config 5: 1 = the whole job as ONE kernel of one block (SET_K_SSSP_SOLO) instead of the WHILE-node pipeline:
 *            same buffers, same output; meant for graphs of a few thousand vertices.
 * *            any config: bit 8 set = append a SET_K_SPIN delay stage that busy-waits dims[3] nanoseconds.
 *   stages/bufs : HOST arrays with room for SET_MAX_STAGES / SET_MAX_BUFFERS entries.
 *   host_in_bytes/host_out_bytes : HOST, may be NULL; maximum byte size of a job's host images.
 */
set_status set_builtin_pipeline(int config, int variant, const uint32_t *params, int num_params,
                                set_stage_desc *stages, int *num_stages,
                                set_buffer_desc *bufs, int *num_bufs,
                                uint64_t *host_in_bytes, uint64_t *host_out_bytes);

/* ---------------------------------------------------------------------------------------------- *
 * Host-only self tests of the lock-free structures (no CUDA call is made; usable without a GPU).
 */
/* Steal-scan order of Algorithm 2 l.8-17: given b queues whose non-emptiness is the
 * bit mask `nonempty` (b <= 64), return the queue FindJob(w) takes from: w if non-empty, else the
 * first (w+k) mod b, k = 1..b-1, that is non-empty, else -1. */
int set_selftest_find_order(int b, int w, uint64_t nonempty);
/* Multi-threaded stress of the bounded MPMC ring used for Q_w, W_pool and the exec free lists:
 * `producers` threads push `items_per_producer` distinct tokens, `consumers` threads pop until all
 * are seen.  Returns 0 if every token was delivered exactly once, else a negative count of errors. */
int64_t set_selftest_ring(int capacity, int producers, int consumers, int64_t items_per_producer);
/* Run Algorithms 1-3 end to end with a simulated device: `completers` host threads stand in for the
 * CUDA driver's callback thread and finish launched jobs after a pseudo-random delay.  Checks: every
 * job completes exactly once, never more than b in flight, no slot runs two jobs at once, a stolen
 * job is bound to the thief's slot.  seed bit 0 selects SET_STEAL_RETARGET, seed bit 1 flag-polled completion
 * (the completers store the slot's word instead of calling Algorithm 3), seed bit 2 a completion thread of its own
 * (set_config.completion_thread), seed bit 3 bind-at-launch (set_config.bind_at_launch).  Returns 0 or a negative error code. */
int64_t set_selftest_scheduler(int num_streams, int max_inflight, int queue_capacity, int num_dispatchers,
                               int submitters, int64_t jobs, uint32_t seed, uint64_t *out_steals);

/* ---------------------------------------------------------------------------------------------- *
 * Several scheduler instances behind one submit call ("one scheduler instance per GPU (own streams, slots,
 * execs); job_id mod n_gpu as home, host-side stealing across instances"; PAPER.md:122 for the retarget-to-thief idea).
 * No collective, no device-to-device traffic: jobs are independent and live in host memory; an instance is a whole set_ctx
 * on the device it was given, and two instances may share a device.  Host buffers must be reachable from every device
 * (set_host_alloc memory is: it is allocated portable).  Unmeasured on more than one GPU.
 *
 * set_multi_create      : cfg as for set_create_ex (cfg->device is ignored), devices: HOST array[num_instances] of CUDA
 *                         ordinals, 1 <= num_instances <= 64.  SET_MODE_SET only.  *out is NULL on failure.
 * set_multi_register_pipeline : the same pipeline on every instance (arguments as set_register_pipeline).
 * set_multi_submit_dims : home = job_id mod num_instances.  If the home instance has no free executable at this instant
 *                         the job goes to the first other instance (home + 1, home + 2, ... cyclically) that has one -- the
 *                         idle instance steals at the host, before anything was bound -- and if none has, the call blocks
 *                         on the home instance (back-pressure).  Thread-safe like set_submit.  dims may be NULL.
 * set_multi_drain       : set_drain of every instance; returns the first failing status.
 * set_multi_instance    : the i-th set_ctx (for set_host_alloc, set_get_stats, set_last_error), NULL if out of range.
 * set_multi_stolen      : jobs that ran on an instance other than their home since creation.
 * set_multi_destroy     : drains and destroys every instance.
 */
typedef struct set_multi set_multi;
set_status set_multi_create(const set_config *cfg, int num_instances, const int *devices, set_multi **out);
set_status set_multi_register_pipeline(set_multi *m, const set_stage_desc *stages, int num_stages,
                                       const set_buffer_desc *bufs, int num_bufs);
set_status set_multi_submit_dims(set_multi *m, uint64_t job_id, const void *host_in, void *host_out,
                                 const uint32_t dims[SET_MAX_DIMS]);
set_status set_multi_drain(set_multi *m);
set_ctx *set_multi_instance(set_multi *m, int i);
uint64_t set_multi_stolen(set_multi *m);
set_status set_multi_destroy(set_multi *m);

/* ---------------------------------------------------------------------------------------------- *
 * An entry point that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid allocation).
 *
 * set_sssp_noalloc: one SSSP job -- the computation of builtin config 5 ("Bellman-Ford graph traversal with
 * frontier-based relaxation"; readings S5-1..S5-4) -- as ONE kernel launch on `stream`, without a set_ctx.
 *   dev_image    : DEVICE, int32 [V, E, src, 0][row_ptr V+1][col E][w E], 4-byte aligned (the job image of config 5);
 *                  read only; the caller keeps it alive and unchanged until the launch has finished on `stream`
 *   dev_out      : DEVICE, int32 [dist V][rounds, 0, 0, 0]: written by the kernel; dist[] is the unique result
 *                  (unreachable = 2^31 - 1), rounds counts the relaxation rounds that had a frontier
 *   num_vertices : V of the image (the kernel reads min(image V, num_vertices) vertices); 0 = do the per-device set-up
 *                  only and launch nothing (call this once per device before a graph capture)
 *   stream       : a cudaStream_t passed as a plain pointer (NULL = the default stream)
 * The kernel's scratch (its work list of frontier vertices, SET_NOALLOC_MAX_VERTICES uint32 = 64 KiB) is a file-scope static
 * __device__ array: every GPU that loads the library holds it until the process exits.  The call makes no cudaMalloc, cudaFree or
 * other allocating call; the first call on a device resolves the array's device address (cudaGetSymbolAddress).  It is
 * asynchronous: the result is in dev_out once `stream` has reached the launch.
 * EVERY call on a device shares the one array, and it keeps the last call's contents: the kernel writes every entry it
 * reads before reading it, so calls one after the other -- on one stream, or ordered by events -- are independent, but
 * two calls that OVERLAP on the GPU (different streams, no ordering) race on it and give wrong distances.
 * Errors: SET_ERR_SIZE if num_vertices > SET_NOALLOC_MAX_VERTICES (nothing is launched), SET_ERR_INVALID (NULL
 * pointers), SET_ERR_CUDA (no device, failed launch); the text is in set_noalloc_last_error() (per thread, valid until
 * that thread's next call).  One block runs the job: a latency path, not a throughput one.
 */
#define SET_NOALLOC_MAX_VERTICES 16384
set_status set_sssp_noalloc(const void *dev_image, void *dev_out, uint32_t num_vertices, void *stream);
const char *set_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SET_H */
