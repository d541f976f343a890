// set_cuda.cpp -- CUDA backend and C ABI of libset (include/set.h).
//
// Layers L1 (job-as-graph + memory slots) and the CUDA half of L2 (GraphLaunch, AddCallback,
// UpdateGraphParams of Algorithms 1-2).  The lock-free scheduling logic itself is in
// set_core.hpp.  Also holds the in-run baseline models of PAPER.md:224-229 (they share buffers, graphs and
// kernels with SET, not the scheduler).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <condition_variable>
#include <deque>
#include <memory>
#include <mutex>
#include <thread>
#include <vector>

#include "../../include/set.h"
#include "set_core.hpp"

using namespace setrt;

#define SET_COPY_BYTES_PER_BLOCK 8192u  // kernels/kernels.h kCopyBytesPerBlock (SET_K_COPY: 256 threads x 2 x 16 B)


namespace {

inline uint64_t eval(const set_size_expr& e, const uint32_t* dims) {
    uint64_t prod = 1;
    for (int i = 0; i < SET_MAX_DIMS; ++i)
        if (e.dim_mask >> i & 1) prod *= dims[i];
    return e.fixed + e.per_unit * prod;
}
inline bool expr_is_zero(const set_size_expr& e) { return e.fixed == 0 && e.per_unit == 0; }

struct SpinLock {
    std::atomic_flag f = ATOMIC_FLAG_INIT;
    void lock() {
        while (f.test_and_set(std::memory_order_acquire)) cpu_relax();
    }
    void unlock() { f.clear(std::memory_order_release); }
};

struct ArgPack {
    alignas(64) unsigned char store[SET_MAX_ARGS][128];
    void* ptrs[SET_MAX_ARGS];
};

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct SlotMem {
    void* buf[SET_MAX_BUFFERS] = {};
    cudaEvent_t done = nullptr;   // event chaining: recorded behind the slot's graph on its work stream
    cudaEvent_t t0 = nullptr;     // plain-stream baseline / timing helpers
    bool used = false;
};

struct ExecState {
    cudaGraphExec_t exec = nullptr;
    int bound_slot = -1;
    const void* in = nullptr;  // what the copy nodes currently point at
    void* out = nullptr;
    uint32_t dims[4] = {1, 1, 1, 1};
    // pageable staging (lazily allocated pinned blocks tied to this exec)
    void* stage_in = nullptr;
    void* stage_out = nullptr;
    bool staged = false;
    void* user_out = nullptr;
    uint64_t out_bytes = 0;
};

struct PinnedRange {
    uintptr_t lo, hi;
};

}  // namespace

constexpr int kMaxLoopStreams = 8;     // WHILE graphs in flight at once (set_register_pipeline says why)
constexpr int kMinLoopBodyStages = 3;  // kernel nodes in a WHILE body (set_register_pipeline says why)

struct set_ctx final : public Backend {
    set_config cfg{};
    int S = 0, b = 0, q = 0, epp = 0, device = 0;
    int L = 1, H = 0;  // set_config.streams_per_lane and the number of CUDA streams H = S * L; slot w runs on streams[w % Hw]
    int Hw = 0;        // streams in use: H, or for a pipeline with a loop at most kMaxLoopStreams of them (see set_register_pipeline)
    std::vector<cudaStream_t> streams, notify;
    bool own_streams = false;
    std::unique_ptr<SpinLock[]> stream_locks;

    bool registered = false;
    std::vector<set_stage_desc> stages;
    std::vector<set_buffer_desc> bufs;
    uint64_t in_extent_unit = 0, out_extent_unit = 0;

    std::vector<SlotMem> slots;
    std::vector<ExecState> execs;
    std::vector<void*> owned_dev;
    // One job graph and the handles of its nodes.  Ordinarily there is ONE template, built on slot 0's buffers, and every
    // executable is instantiated from it and re-bound to its slot node by node.  A graph that holds a conditional node can be
    // instantiated only ONCE (a second cudaGraphInstantiate returns cudaErrorNotSupported, CUDA 12.9), so a pipeline with a
    // data-dependent loop (SET_STAGE_LOOP_BEGIN) gets one graph PER EXECUTABLE, built directly on its slot's buffers -- and
    // its executables never leave their slot.
    struct NodeSet {
        cudaGraph_t graph = nullptr;
        std::vector<cudaGraphNode_t> kern_nodes;
        cudaGraphNode_t memset_nodes[SET_MAX_BUFFERS] = {}, h2d_nodes[SET_MAX_BUFFERS] = {}, d2h_nodes[SET_MAX_BUFFERS] = {};
        cudaGraphNode_t signal_node = nullptr;  // SET_CB_FLAG_POLL: last node, stores the slot's completion word
        cudaGraphNode_t host_node = nullptr;    // SET_CB_HOST_NODE: last node, runs Algorithm 3 on the driver's callback thread
        cudaGraphNode_t stamp_start_node = nullptr, stamp_end_node = nullptr;
        cudaGraphNode_t loop_node = nullptr;    // the conditional WHILE node, if the pipeline has a loop
    };
    std::vector<NodeSet> nsets;
    bool slot_graphs = false;                  // the pipeline has a loop: nsets[e] belongs to executable e (slot e / epp)
    std::vector<char> stage_in_loop;           // per stage: inside the WHILE body
    bool has_signal = false, has_host_node = false;
    NodeSet& nodes_of_exec(int exec) { return nsets[slot_graphs ? (size_t)exec : 0]; }
    // set_config.timestamps: per slot one 64-byte line of mapped pinned memory, [0] = %globaltimer at graph start, [1] = at end
    bool stamps = false;
    unsigned long long* ts_host = nullptr;
    unsigned long long* ts_dev = nullptr;
    struct StampRec {
        uint32_t stream;
        uint64_t start, end;
    };
    SpinLock stamp_lock;
    std::vector<StampRec> stamp_recs;  // one per completed job, reduced by set_get_gap_stats
    // SM copies (set_config.sm_copy_max_bytes): h2d_nodes[i] / d2h_nodes[i] are SET_K_COPY kernel nodes where set
    bool h2d_sm[SET_MAX_BUFFERS] = {}, d2h_sm[SET_MAX_BUFFERS] = {};
    int n_sm_copies = 0;
    bool pdl = false;                          // some stage asked for SET_STAGE_PDL: kernel-to-kernel edges are programmatic
    uint32_t* flags_host = nullptr;            // b words, kFlagStride apart, mapped pinned host memory
    uint32_t* flags_dev = nullptr;             // the device's address of the same memory
    bool flag_poll = false;
    void* ph_in = nullptr;   // placeholder operands the template graph is built with
    void* ph_out = nullptr;

    std::unique_ptr<Scheduler> sched;
    struct CbArg {
        set_ctx* ctx;
        int slot;
    };
    std::vector<CbArg> cbargs;

    // counters owned by the backend
    std::atomic<uint64_t> full_rebinds{0}, host_rebinds{0}, staged_jobs{0}, ns_bind{0}, ns_sync{0}, kernel_nodes{0}, signal_nodes{0}, copy_nodes{0},
        early_completions{0};
    std::atomic<uint64_t> base_submitted{0}, base_completed{0}, base_launched{0}, base_ns_submit{0}, base_ns_launch{0};

    // sticky error
    std::atomic<int> err{0};
    std::mutex errmu;
    char errmsg[512] = {0};

    // host allocations and the pinned-range cache
    std::mutex hostmu;
    std::vector<std::pair<void*, size_t>> host_allocs;
    SpinLock range_lock;
    std::vector<PinnedRange> pinned_ranges;

    PFN_encodeTiled encode_tiled = nullptr;

    // SET_DRIVER_LOCK=1 (environment, read at create): every graph update and graph launch takes this one lock.
    // Only for runs under Nsight Compute 2025.2, whose injection library double-frees when one thread updates a
    // graph executable while another thread is inside cudaGraphLaunch (profiles/r1_ncu.md); never set for timing.
    uint32_t copy_max_blocks = 0;  // SET_COPY_MAX_BLOCKS (environment): blocks per SM copy that reads host memory; 0 = default (8)
    bool driver_lock = false;
    std::mutex driver_mu;

    // baseline state (single caller thread)
    std::vector<JobDesc> batch;
    uint64_t base_ticket = 0;
    // SET_MODE_MUTEX_QUEUE: one global issue queue behind a mutex; a worker thread scans all
    // b slots every round (O(b) cudaEventQuery calls), and feeds each free slot from the queue.
    std::mutex mq_mu;
    std::condition_variable mq_cv;
    std::deque<JobDesc> mq_queue;
    std::thread mq_thread;
    std::atomic<bool> mq_stop{false};
    std::atomic<uint64_t> mq_queries{0};
    void mq_loop();

    // ------------------------------------------------------------------ errors
    int fail(int code, const char* fmt, ...) {
        int zero = 0;
        if (err.compare_exchange_strong(zero, code)) {
            std::lock_guard<std::mutex> g(errmu);
            va_list ap;
            va_start(ap, fmt);
            vsnprintf(errmsg, sizeof(errmsg), fmt, ap);
            va_end(ap);
        }
        if (sched) sched->set_error(code);
        return code;
    }
    int cuda_fail(cudaError_t e, const char* what, int line) {
        return fail(SET_ERR_CUDA, "%s failed at set_cuda.cpp:%d: %s (%s)", what, line, cudaGetErrorName(e),
                    cudaGetErrorString(e));
    }

    void bind_thread() {
        static thread_local int bound = -1;
        if (bound != device) {
            cudaSetDevice(device);
            bound = device;
        }
    }

    // ------------------------------------------------------------------ Backend interface
    int bind(int exec, int slot, JobDesc& job, bool* pinned_to_exec) override;
    int launch(int exec, int slot, const JobDesc& job) override;
    int validate(const JobDesc& job) override { return check_sizes(job.dims); }
    void finish(int exec, int slot, const JobDesc& job) override;
    int poll() override;
    volatile uint32_t* done_flags() override { return flag_poll ? flags_host : nullptr; }

    int build_args(const set_stage_desc& st, int slot, const uint32_t* dims, ArgPack& ap, dim3& grid, unsigned long long cond = 0);
    // SET_K_COPY node parameters for buffer i of `slot`: H2D (host_or_dev = job input) or D2H (job output)
    struct CopyArgs {
        const void* src;
        void* dst;
        uint32_t bytes;
        void** fwd_slot;               // SET_K_COPY: where the copy-in node leaves the job's output address (or NULL)
        void* fwd_value;
        unsigned long long dst_off;    // SET_K_COPY_OUT: byte offset behind the forwarded address
        uint32_t* sig_flag;            // SET_K_COPY_OUT with the completion signal folded in (else NULL)
        unsigned long long* sig_stamp;
        uint32_t sig_fence;
        void* ptrs[7];
        cudaKernelNodeParams kp;
    };
    // `host` is the job's input (to_device) or output image; `fwd_out` the job's output image, forwarded by copy-in node fwd_buf
    void copy_params(CopyArgs& ca, int slot, int i, bool to_device, const void* host, const uint32_t* dims, const void* fwd_out = nullptr);
    // Output-address forwarding: SM copy-out nodes take their destination from a per-slot device word that the
    // job's first SM copy-in node fills, so a job in the steady state costs one graph-node update, not two.
    int fwd_buf = -1;                  // buffer whose H2D SM-copy node forwards; -1 = off
    bool d2h_ind[SET_MAX_BUFFERS] = {};
    void** fwd_dev = nullptr;          // per slot two 8-byte device words: the forwarded address, the copy-out blocks' ticket counter
    int fused_signal_buf = -1;         // the job's ONLY copy-out node is this buffer's SM copy and also stores the completion word
    int check_sizes(const uint32_t* dims);
    bool is_pinned(const void* p);
    void add_pinned_range(const void* p, size_t n);
    int build_graph(int slot, int set_index);
    int plain_job(int slot, const JobDesc& job);
    int baseline_submit(const JobDesc& job);
    int baseline_flush();
    int baseline_drain();
};

#define CK(call)                                                         \
    do {                                                                 \
        cudaError_t _e = (call);                                         \
        if (_e != cudaSuccess) return cuda_fail(_e, #call, __LINE__);    \
    } while (0)

// ---------------------------------------------------------------------------------------------------------
// kernel arguments: placeholders -> concrete values for (slot, dims)
// ---------------------------------------------------------------------------------------------------------
int set_ctx::build_args(const set_stage_desc& st, int slot, const uint32_t* dims, ArgPack& ap, dim3& grid, unsigned long long cond) {
    for (int a = 0; a < st.num_args; ++a) {
        const set_arg_desc& d = st.args[a];
        ap.ptrs[a] = ap.store[a];
        switch (d.kind) {
            case SET_ARG_BUFFER: {
                char* p = (char*)slots[slot].buf[d.index] + eval(d.offset, dims);
                memcpy(ap.store[a], &p, sizeof(p));
                break;
            }
            case SET_ARG_IMM32: {
                uint32_t v = (uint32_t)d.imm;
                memcpy(ap.store[a], &v, 4);
                break;
            }
            case SET_ARG_IMM64:
                memcpy(ap.store[a], &d.imm, 8);
                break;
            case SET_ARG_DIM:
                memcpy(ap.store[a], &dims[d.index], 4);
                break;
            case SET_ARG_COND:  // cudaGraphConditionalHandle of the enclosing loop (0 outside a job graph)
                memcpy(ap.store[a], &cond, 8);
                break;
            case SET_ARG_TMAP2D: {
                if (!encode_tiled) return fail(SET_ERR_CUDA, "cuTensorMapEncodeTiled entry point unavailable");
                const set_tmap2d& t = d.tmap;
                CUtensorMapDataType dt = t.elem_bytes == 2   ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                         : t.elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                                             : CU_TENSOR_MAP_DATA_TYPE_UINT8;
                cuuint64_t gdim[2] = {t.inner, t.outer};
                cuuint64_t gstride[1] = {t.pitch_bytes};
                cuuint32_t box[2] = {t.box_inner, t.box_outer};
                cuuint32_t estr[2] = {1, 1};
                CUtensorMapSwizzle sw = t.swizzle == SET_SWIZZLE_128B  ? CU_TENSOR_MAP_SWIZZLE_128B
                                        : t.swizzle == SET_SWIZZLE_64B ? CU_TENSOR_MAP_SWIZZLE_64B
                                                                       : CU_TENSOR_MAP_SWIZZLE_NONE;
                char* base = (char*)slots[slot].buf[d.index] + eval(d.offset, dims);
                CUresult r = encode_tiled((CUtensorMap*)ap.store[a], dt, 2, base, gdim, gstride, box, estr,
                                          CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS) return fail(SET_ERR_CUDA, "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
                break;
            }
            default:
                return fail(SET_ERR_INVALID, "unknown argument kind %d", d.kind);
        }
    }
    unsigned g[3];
    for (int i = 0; i < 3; ++i) {
        uint64_t c = eval(st.grid[i].count, dims);
        uint64_t dv = st.grid[i].divisor ? st.grid[i].divisor : 1;
        uint64_t v = (c + dv - 1) / dv;
        g[i] = (unsigned)(v ? v : 1);
    }
    grid = dim3(g[0], g[1], g[2]);
    return 0;
}

void set_ctx::copy_params(CopyArgs& ca, int slot, int i, bool to_device, const void* host, const uint32_t* dims, const void* fwd_out) {
    const set_buffer_desc& bd = bufs[i];
    ca.kp = cudaKernelNodeParams{};
    ca.fwd_slot = nullptr;
    ca.fwd_value = nullptr;
    ca.dst_off = 0;
    if (to_device) {
        ca.src = (const char*)host + eval(bd.h2d_host_off, dims);
        ca.dst = (char*)slots[slot].buf[i] + eval(bd.h2d_dev_off, dims);
        ca.bytes = (uint32_t)eval(bd.h2d_bytes, dims);
        if (i == fwd_buf) {
            ca.fwd_slot = fwd_dev + 2 * (size_t)slot;
            ca.fwd_value = const_cast<void*>(fwd_out);
        }
    } else {
        ca.src = (const char*)slots[slot].buf[i] + eval(bd.d2h_dev_off, dims);
        ca.dst = (char*)host + eval(bd.d2h_host_off, dims);
        ca.bytes = (uint32_t)eval(bd.d2h_bytes, dims);
        ca.dst_off = eval(bd.d2h_host_off, dims);
    }
    if (!to_device && d2h_ind[i]) {  // (src, dst_slot, dst_off, bytes, flag, stamp, fence)
        ca.fwd_slot = fwd_dev + 2 * (size_t)slot;
        const bool sig = i == fused_signal_buf;
        ca.sig_flag = sig ? flags_dev + (size_t)slot * kFlagStride : nullptr;
        ca.sig_stamp = sig && stamps ? ts_dev + (size_t)slot * 8 + 1 : nullptr;
        ca.sig_fence = cfg.completion_fence == SET_FENCE_SYSTEM ? 1u : 0u;
        ca.ptrs[0] = &ca.src;
        ca.ptrs[1] = &ca.fwd_slot;
        ca.ptrs[2] = &ca.dst_off;
        ca.ptrs[3] = &ca.bytes;
        ca.ptrs[4] = &ca.sig_flag;
        ca.ptrs[5] = &ca.sig_stamp;
        ca.ptrs[6] = &ca.sig_fence;
        ca.kp.func = const_cast<void*>(set_builtin_kernel(SET_K_COPY_OUT));
    } else {                         // (src, dst, bytes, fwd_slot, fwd_value)
        ca.ptrs[0] = &ca.src;
        ca.ptrs[1] = &ca.dst;
        ca.ptrs[2] = &ca.bytes;
        ca.ptrs[3] = &ca.fwd_slot;
        ca.ptrs[4] = &ca.fwd_value;
        ca.kp.func = const_cast<void*>(set_builtin_kernel(SET_K_COPY));
    }
    uint32_t pieces = (ca.bytes + SET_COPY_BYTES_PER_BLOCK - 1) / SET_COPY_BYTES_PER_BLOCK;
    // Reads of pinned host memory share the link with the GPU's own fetches of launch commands: streams that each put 128 KB of
    // reads in flight at once delay the start of every stream's next graph, and the link is saturated by about 512 KB in
    // flight over all streams.  So a copy that reads host memory gets 64 / (CUDA streams) blocks of 8 KB, between 2 and 8 (the
    // kernel strides over the rest).  Measured, config 1 end to end (profiles/r2_probes.md): 32 streams -- 1 / 2 / 3 / 4 / 8 / 16
    // blocks give 367 / 380 / 373 / 353 / 325 / 303 K jobs/s (380 K is the duplex link bound); 8 streams -- 1 / 2 / 3 / 8 blocks
    // give 163 / 194 / 203 / 219 K.  Stores to host memory and HBM-to-HBM copies are not capped.
    if (to_device && cfg.io == SET_IO_HOST) {
        const uint32_t cap = copy_max_blocks ? copy_max_blocks : (uint32_t)std::min(8, std::max(2, 64 / std::max(1, H)));
        if (pieces > cap) pieces = cap;
    }
    ca.kp.gridDim = dim3(pieces ? pieces : 1);
    ca.kp.blockDim = dim3(256);
    ca.kp.kernelParams = ca.ptrs;
}

int set_ctx::check_sizes(const uint32_t* dims) {
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (eval(bd.h2d_dev_off, dims) + eval(bd.h2d_bytes, dims) > bd.bytes) return SET_ERR_SIZE;
        if (eval(bd.d2h_dev_off, dims) + eval(bd.d2h_bytes, dims) > bd.bytes) return SET_ERR_SIZE;
        if ((bd.flags & SET_BUF_ZERO) && eval(bd.zero_off, dims) + eval(bd.zero_bytes, dims) > bd.bytes) return SET_ERR_SIZE;
    }
    for (auto& st : stages)
        for (int a = 0; a < st.num_args; ++a)
            if ((st.args[a].kind == SET_ARG_BUFFER || st.args[a].kind == SET_ARG_TMAP2D) &&
                eval(st.args[a].offset, dims) > bufs[st.args[a].index].bytes)
                return SET_ERR_SIZE;
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// pinned-memory test: known ranges first, one driver query per unknown allocation
// ---------------------------------------------------------------------------------------------------------
// pinned_ranges is kept sorted by start address (ranges never overlap: they are whole allocations), so the test is a
// binary search however many buffers the caller has allocated
void set_ctx::add_pinned_range(const void* p, size_t n) {
    PinnedRange r{(uintptr_t)p, (uintptr_t)p + n};
    range_lock.lock();
    auto it = std::upper_bound(pinned_ranges.begin(), pinned_ranges.end(), r.lo,
                               [](uintptr_t a, const PinnedRange& b) { return a < b.lo; });
    pinned_ranges.insert(it, r);
    range_lock.unlock();
}

bool set_ctx::is_pinned(const void* p) {
    uintptr_t a = (uintptr_t)p;
    range_lock.lock();
    auto it = std::upper_bound(pinned_ranges.begin(), pinned_ranges.end(), a,
                               [](uintptr_t x, const PinnedRange& b) { return x < b.lo; });
    bool hit = it != pinned_ranges.begin() && a < (it - 1)->hi;
    range_lock.unlock();
    if (hit) return true;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    if (at.type != cudaMemoryTypeHost) return false;
    // SM copies dereference the caller's pointer on the device: registered memory whose device alias differs (or
    // that is not mapped at all) goes through the library's own pinned staging blocks like pageable memory
    if (n_sm_copies && at.devicePointer != p) return false;
    // Not cached: the library does not own this memory and cannot see it being freed (a stale entry would later send
    // an SM copy into pageable memory).  Callers with their own pinned buffers declare them with set_host_register.
    return true;
}

// ---------------------------------------------------------------------------------------------------------
// A2: job-as-graph.  [memset] / H2D roots -> kernel chain -> D2H leaves, built by explicit construction
// with slot 0's buffers and placeholder host operands; every exec is then re-bound.
// ---------------------------------------------------------------------------------------------------------
static void CUDART_CB set_completion_cb(void* arg);

int set_ctx::build_graph(int slot, int set_index) {
    NodeSet& g = nsets[(size_t)set_index];
    const uint32_t unit[4] = {1, 1, 1, 1};
    cudaMemcpyKind kin = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    cudaMemcpyKind kout = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    // dependency helper: a programmatic (PDL) edge where both ends are kernel nodes and the pipeline asked for it
    auto depend_in = [&](cudaGraph_t gr, cudaGraphNode_t from, cudaGraphNode_t to, bool programmatic) -> cudaError_t {
        if (!programmatic) return cudaGraphAddDependencies(gr, &from, &to, 1);
        cudaGraphEdgeData ed{};
        ed.from_port = cudaGraphKernelNodePortProgrammatic;
        ed.to_port = 0;
        ed.type = cudaGraphDependencyTypeProgrammatic;
        return cudaGraphAddDependencies_v2(gr, &from, &to, &ed, 1);
    };
    auto depend = [&](cudaGraphNode_t from, cudaGraphNode_t to, bool programmatic) { return depend_in(g.graph, from, to, programmatic); };
    CK(cudaGraphCreate(&g.graph, 0));
    std::vector<cudaGraphNode_t> roots;
    std::vector<bool> root_is_kernel;
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (bd.flags & SET_BUF_ZERO) {
            cudaMemsetParams mp{};
            mp.dst = (char*)slots[slot].buf[i] + eval(bd.zero_off, unit);
            mp.elementSize = 1;
            mp.width = eval(bd.zero_bytes, unit);
            mp.height = 1;
            mp.value = 0;
            CK(cudaGraphAddMemsetNode(&g.memset_nodes[i], g.graph, nullptr, 0, &mp));
            roots.push_back(g.memset_nodes[i]);
            root_is_kernel.push_back(false);
        }
        if (!expr_is_zero(bd.h2d_bytes)) {
            if (h2d_sm[i]) {
                CopyArgs ca;
                copy_params(ca, slot, (int)i, true, ph_in, unit, ph_out);
                CK(cudaGraphAddKernelNode(&g.h2d_nodes[i], g.graph, nullptr, 0, &ca.kp));
            } else {
                CK(cudaGraphAddMemcpyNode1D(&g.h2d_nodes[i], g.graph, nullptr, 0, (char*)slots[slot].buf[i] + eval(bd.h2d_dev_off, unit),
                                            (char*)ph_in + eval(bd.h2d_host_off, unit), eval(bd.h2d_bytes, unit), kin));
            }
            roots.push_back(g.h2d_nodes[i]);
            root_is_kernel.push_back(h2d_sm[i]);
        }
    }
    if (stamps) {  // a root of its own, beside the first copies: runs when the graph starts, nothing waits for it
        unsigned long long* p = ts_dev + (size_t)slot * 8;
        void* args[1] = {&p};
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void*>(set_builtin_kernel(SET_K_STAMP));
        kp.gridDim = dim3(1);
        kp.blockDim = dim3(1);
        kp.kernelParams = args;
        CK(cudaGraphAddKernelNode(&g.stamp_start_node, g.graph, nullptr, 0, &kp));
    }
    g.kern_nodes.assign(stages.size(), nullptr);
    cudaGraphNode_t prev = nullptr;       // last node of the top-level chain
    cudaGraph_t body = nullptr;           // body graph of the loop being filled, if any
    cudaGraphNode_t body_prev = nullptr;
    cudaGraphConditionalHandle cond = 0;
    // first node of the top-level chain hangs off every root; a kernel may have at most one programmatic predecessor worth
    // having: use it only for a lone SM-copy root
    auto attach_top = [&](cudaGraphNode_t node, bool node_is_kernel, bool want_pdl) -> int {
        if (!prev) {
            for (size_t r = 0; r < roots.size(); ++r)
                CK(depend(roots[r], node, node_is_kernel && want_pdl && roots.size() == 1 && root_is_kernel[r]));
        } else {
            CK(depend(prev, node, node_is_kernel && want_pdl && prev != g.loop_node));
        }
        prev = node;
        return 0;
    };
    for (size_t s = 0; s < stages.size(); ++s) {
        const set_stage_desc& st = stages[s];
        if (st.flags & SET_STAGE_LOOP_BEGIN) {
            // PAPER.md:220 / SURVEY.md 8(f)4: the iteration count depends on the data, so the stages up to SET_STAGE_LOOP_END
            // become the body of a conditional WHILE node; the body's control kernel sets the condition on the device.
            CK(cudaGraphConditionalHandleCreate(&cond, g.graph, 1, cudaGraphCondAssignDefault));
            cudaGraphNodeParams np{};
            np.type = cudaGraphNodeTypeConditional;
            np.conditional.handle = cond;
            np.conditional.type = cudaGraphCondTypeWhile;
            np.conditional.size = 1;
            CK(cudaGraphAddNode(&g.loop_node, g.graph, nullptr, 0, &np));
            if (int rc = attach_top(g.loop_node, false, false)) return rc;
            body = np.conditional.phGraph_out[0];
            body_prev = nullptr;
        }
        ArgPack ap;
        dim3 grid;
        if (int rc = build_args(st, slot, unit, ap, grid, (unsigned long long)cond)) return rc;
        if (st.smem_bytes > 48 * 1024)
            CK(cudaFuncSetAttribute(st.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)st.smem_bytes));
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void*>(st.func);
        kp.gridDim = grid;
        kp.blockDim = dim3(st.block[0], st.block[1] ? st.block[1] : 1, st.block[2] ? st.block[2] : 1);
        kp.sharedMemBytes = st.smem_bytes;
        kp.kernelParams = ap.ptrs;
        const bool want_pdl = (st.flags & SET_STAGE_PDL) != 0;
        if (body) {
            CK(cudaGraphAddKernelNode(&g.kern_nodes[s], body, nullptr, 0, &kp));
            // always a plain edge inside a loop body: with a programmatic edge between the relaxation and the control kernel
            // 16 or more concurrent WHILE graphs ended in cudaErrorLaunchFailure on B200 (CUDA 12.9); SET_STAGE_PDL is ignored here
            if (body_prev) CK(depend_in(body, body_prev, g.kern_nodes[s], false));
            (void)want_pdl;
            body_prev = g.kern_nodes[s];
            if (st.flags & SET_STAGE_LOOP_END) body = nullptr;
        } else {
            CK(cudaGraphAddKernelNode(&g.kern_nodes[s], g.graph, nullptr, 0, &kp));
            if (int rc = attach_top(g.kern_nodes[s], true, want_pdl)) return rc;
        }
    }
    const bool prev_is_kernel = prev != g.loop_node;
    std::vector<cudaGraphNode_t> leaves;
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (!expr_is_zero(bd.d2h_bytes)) {
            if (d2h_sm[i]) {
                CopyArgs ca;
                copy_params(ca, slot, (int)i, false, ph_out, unit);
                CK(cudaGraphAddKernelNode(&g.d2h_nodes[i], g.graph, nullptr, 0, &ca.kp));
                CK(depend(prev, g.d2h_nodes[i], pdl && prev_is_kernel));
            } else {
                CK(cudaGraphAddMemcpyNode1D(&g.d2h_nodes[i], g.graph, &prev, 1, (char*)ph_out + eval(bd.d2h_host_off, unit),
                                            (char*)slots[slot].buf[i] + eval(bd.d2h_dev_off, unit), eval(bd.d2h_bytes, unit), kout));
            }
            leaves.push_back(g.d2h_nodes[i]);
        }
    }
    if (flag_poll && fused_signal_buf >= 0) {
        // the job's only copy-out node stores the completion word itself (K24); the start stamp only has to have run before it
        if (stamps) CK(depend(g.stamp_start_node, g.d2h_nodes[fused_signal_buf], false));
    } else if (flag_poll) {  // completion signal: runs after every D2H copy of the job has finished (kernels.cu K14)
        std::vector<bool> leaf_is_kernel;
        for (size_t i = 0; i < bufs.size(); ++i)
            if (!expr_is_zero(bufs[i].d2h_bytes)) leaf_is_kernel.push_back(d2h_sm[i]);
        if (leaves.empty()) {
            leaves.push_back(prev);
            leaf_is_kernel.push_back(prev_is_kernel);
        }
        uint32_t* flag = flags_dev + (size_t)slot * kFlagStride;
        unsigned long long* stamp = stamps ? ts_dev + (size_t)slot * 8 + 1 : nullptr;
        uint32_t fence = cfg.completion_fence == SET_FENCE_SYSTEM ? 1u : 0u;
        void* args[3] = {&flag, &stamp, &fence};
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void*>(set_builtin_kernel(SET_K_SIGNAL));
        kp.gridDim = dim3(1);
        kp.blockDim = dim3(1);
        kp.kernelParams = args;
        CK(cudaGraphAddKernelNode(&g.signal_node, g.graph, nullptr, 0, &kp));
        for (size_t l = 0; l < leaves.size(); ++l) CK(depend(leaves[l], g.signal_node, pdl && leaves.size() == 1 && leaf_is_kernel[l]));
        // the start stamp is a root nothing else waits for; this edge only makes sure it has run before the end stamp
        if (stamps) CK(depend(g.stamp_start_node, g.signal_node, false));
        has_signal = true;
    } else if (stamps) {  // no signal node in this mode: the end timestamp gets a last node of its own
        if (leaves.empty()) leaves.push_back(prev);
        unsigned long long* p = ts_dev + (size_t)slot * 8 + 1;
        void* args[1] = {&p};
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void*>(set_builtin_kernel(SET_K_STAMP));
        kp.gridDim = dim3(1);
        kp.blockDim = dim3(1);
        kp.kernelParams = args;
        leaves.push_back(g.stamp_start_node);  // not on the critical path: it only has to have run before the end stamp
        CK(cudaGraphAddKernelNode(&g.stamp_end_node, g.graph, leaves.data(), leaves.size(), &kp));
        leaves.assign(1, g.stamp_end_node);
    }
    if (cfg.mode == SET_MODE_SET && cfg.callback_mode == SET_CB_HOST_NODE) {
        if (leaves.empty()) leaves.push_back(prev);
        cudaHostNodeParams hp{};
        hp.fn = set_completion_cb;
        hp.userData = &cbargs[slot];
        CK(cudaGraphAddHostNode(&g.host_node, g.graph, leaves.data(), leaves.size(), &hp));
        has_host_node = true;
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// UpdateGraphParams(J, i)  (Alg. 1 l.4 / Alg. 2 l.20)
// Host-pointer copy nodes change for every job; kernel/memset nodes and the device side of the copies change
// only when the exec moves to another slot's memory or the job's dims differ from the exec's last dims.
// ---------------------------------------------------------------------------------------------------------
int set_ctx::bind(int exec, int slot, JobDesc& job, bool* pinned_to_exec) {
    uint64_t t0 = now_ns();
    bind_thread();
    std::unique_lock<std::mutex> dl(driver_mu, std::defer_lock);
    if (driver_lock) dl.lock();
    ExecState& es = execs[exec];
    NodeSet& g = nodes_of_exec(exec);
    bool dims_changed = memcmp(es.dims, job.dims, sizeof(es.dims)) != 0;
    bool full = es.bound_slot != slot || dims_changed;
    if (slot_graphs && es.bound_slot != slot)
        return fail(SET_ERR_STATE, "an executable of a pipeline with a loop cannot move from slot %d to slot %d", es.bound_slot, slot);
    if (dims_changed)
        if (int rc = check_sizes(job.dims)) return rc;

    const void* in = job.in;
    void* out = job.out;
    *pinned_to_exec = false;
    if (cfg.io == SET_IO_HOST && !es.staged /* a retarget keeps the staging it already has */) {
        bool pin_in = is_pinned(in), pin_out = is_pinned(out);
        if (!pin_in || !pin_out) {
            // pageable caller memory: go through this exec's pinned staging blocks (per-stream pinned ring)
            uint64_t in_bytes = 0, out_bytes = 0;
            for (auto& bd : bufs) {
                if (!expr_is_zero(bd.h2d_bytes)) in_bytes = std::max(in_bytes, eval(bd.h2d_host_off, job.dims) + eval(bd.h2d_bytes, job.dims));
                if (!expr_is_zero(bd.d2h_bytes)) out_bytes = std::max(out_bytes, eval(bd.d2h_host_off, job.dims) + eval(bd.d2h_bytes, job.dims));
            }
            uint64_t cap_in = 0, cap_out = 0;  // capacity: the buffers bound every per-job size
            for (auto& bd : bufs) {
                if (!expr_is_zero(bd.h2d_bytes)) cap_in += bd.bytes;
                if (!expr_is_zero(bd.d2h_bytes)) cap_out += bd.bytes;
            }
            if (!es.stage_in) {
                CK(cudaHostAlloc(&es.stage_in, std::max<uint64_t>(cap_in, in_bytes), cudaHostAllocPortable));
                CK(cudaHostAlloc(&es.stage_out, std::max<uint64_t>(cap_out, out_bytes), cudaHostAllocPortable));
            }
            memcpy(es.stage_in, in, in_bytes);
            es.staged = true;
            es.user_out = out;
            es.out_bytes = out_bytes;
            staged_jobs.fetch_add(1, std::memory_order_relaxed);
        }
    }
    if (es.staged) {
        in = es.stage_in;
        out = es.stage_out;
        *pinned_to_exec = true;
    }

    cudaMemcpyKind kin = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    cudaMemcpyKind kout = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (full) {
        for (size_t s = 0; s < stages.size(); ++s) {
            // nodes inside a loop body cannot be re-pointed one by one; register made sure they do not depend on the job
            if (slot_graphs && stage_in_loop[s]) continue;
            ArgPack ap;
            dim3 grid;
            if (int rc = build_args(stages[s], slot, job.dims, ap, grid)) return rc;
            cudaKernelNodeParams kp{};
            kp.func = const_cast<void*>(stages[s].func);
            kp.gridDim = grid;
            kp.blockDim = dim3(stages[s].block[0], stages[s].block[1] ? stages[s].block[1] : 1,
                               stages[s].block[2] ? stages[s].block[2] : 1);
            kp.sharedMemBytes = stages[s].smem_bytes;
            kp.kernelParams = ap.ptrs;
            CK(cudaGraphExecKernelNodeSetParams(es.exec, g.kern_nodes[s], &kp));
        }
        for (size_t i = 0; i < bufs.size(); ++i)
            if (bufs[i].flags & SET_BUF_ZERO) {
                cudaMemsetParams mp{};
                mp.dst = (char*)slots[slot].buf[i] + eval(bufs[i].zero_off, job.dims);
                mp.elementSize = 1;
                mp.width = eval(bufs[i].zero_bytes, job.dims);
                mp.height = 1;
                CK(cudaGraphExecMemsetNodeSetParams(es.exec, g.memset_nodes[i], &mp));
            }
        if (g.signal_node && es.bound_slot != slot) {
            uint32_t* flag = flags_dev + (size_t)slot * kFlagStride;
            unsigned long long* stamp = stamps ? ts_dev + (size_t)slot * 8 + 1 : nullptr;
            uint32_t fence = cfg.completion_fence == SET_FENCE_SYSTEM ? 1u : 0u;
            void* args[3] = {&flag, &stamp, &fence};
            cudaKernelNodeParams kp{};
            kp.func = const_cast<void*>(set_builtin_kernel(SET_K_SIGNAL));
            kp.gridDim = dim3(1);
            kp.blockDim = dim3(1);
            kp.kernelParams = args;
            CK(cudaGraphExecKernelNodeSetParams(es.exec, g.signal_node, &kp));
        }
        if (stamps && es.bound_slot != slot) {
            unsigned long long* p0 = ts_dev + (size_t)slot * 8;
            unsigned long long* p1 = p0 + 1;
            cudaKernelNodeParams kp{};
            kp.func = const_cast<void*>(set_builtin_kernel(SET_K_STAMP));
            kp.gridDim = dim3(1);
            kp.blockDim = dim3(1);
            void* a0[1] = {&p0};
            kp.kernelParams = a0;
            CK(cudaGraphExecKernelNodeSetParams(es.exec, g.stamp_start_node, &kp));
            if (g.stamp_end_node) {
                void* a1[1] = {&p1};
                kp.kernelParams = a1;
                CK(cudaGraphExecKernelNodeSetParams(es.exec, g.stamp_end_node, &kp));
            }
        }
        if (g.host_node && es.bound_slot != slot) {
            cudaHostNodeParams hp{};
            hp.fn = set_completion_cb;
            hp.userData = &cbargs[slot];
            CK(cudaGraphExecHostNodeSetParams(es.exec, g.host_node, &hp));
        }
        full_rebinds.fetch_add(1, std::memory_order_relaxed);
    } else {
        host_rebinds.fetch_add(1, std::memory_order_relaxed);
    }
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (!expr_is_zero(bd.h2d_bytes) && (full || es.in != in || ((int)i == fwd_buf && es.out != out))) {
            if (h2d_sm[i]) {
                CopyArgs ca;
                copy_params(ca, slot, (int)i, true, in, job.dims, out);
                CK(cudaGraphExecKernelNodeSetParams(es.exec, g.h2d_nodes[i], &ca.kp));
            } else {
                CK(cudaGraphExecMemcpyNodeSetParams1D(es.exec, g.h2d_nodes[i], (char*)slots[slot].buf[i] + eval(bd.h2d_dev_off, job.dims),
                                                      (const char*)in + eval(bd.h2d_host_off, job.dims), eval(bd.h2d_bytes, job.dims), kin));
            }
        }
        if (!expr_is_zero(bd.d2h_bytes) && (full || (es.out != out && !d2h_ind[i]))) {  // a forwarded destination needs no update
            if (d2h_sm[i]) {
                CopyArgs ca;
                copy_params(ca, slot, (int)i, false, out, job.dims);
                CK(cudaGraphExecKernelNodeSetParams(es.exec, g.d2h_nodes[i], &ca.kp));
            } else {
                CK(cudaGraphExecMemcpyNodeSetParams1D(es.exec, g.d2h_nodes[i], (char*)out + eval(bd.d2h_host_off, job.dims),
                                                      (char*)slots[slot].buf[i] + eval(bd.d2h_dev_off, job.dims), eval(bd.d2h_bytes, job.dims), kout));
            }
        }
    }
    es.bound_slot = slot;
    es.in = in;
    es.out = out;
    memcpy(es.dims, job.dims, sizeof(es.dims));
    ns_bind.fetch_add(now_ns() - t0, std::memory_order_relaxed);
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// GraphLaunch + AddCallback (Alg. 2 l.21-22) with event chaining (A6): the completion event is recorded
// behind the graph on the work stream; a per-stream notify stream waits on it and runs the host function,
// so the work stream itself never stalls on the host round trip (PAPER.md:203 puts the callback "at the end
// of the stream"; SET_CB_WORK_STREAM keeps that literal placement for comparison).
// ---------------------------------------------------------------------------------------------------------
static void CUDART_CB set_completion_cb(void* arg) {
    auto* a = static_cast<set_ctx::CbArg*>(arg);
    a->ctx->sched->on_complete(a->slot);  // Algorithm 3
}

int set_ctx::launch(int exec, int slot, const JobDesc&) {
    bind_thread();
    int s = slot % Hw;
    std::unique_lock<std::mutex> dl(driver_mu, std::defer_lock);
    if (driver_lock) dl.lock();
    SpinLock& lk = stream_locks[s];
    lk.lock();
    cudaError_t e = cudaGraphLaunch(execs[exec].exec, streams[s]);
    if (e == cudaSuccess && !flag_poll && !has_host_node) {
        if (cfg.callback_mode == SET_CB_WORK_STREAM) {
            e = cudaLaunchHostFunc(streams[s], set_completion_cb, &cbargs[slot]);
        } else {
            e = cudaEventRecord(slots[slot].done, streams[s]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(notify[s], slots[slot].done, 0);
            if (e == cudaSuccess) e = cudaLaunchHostFunc(notify[s], set_completion_cb, &cbargs[slot]);
        }
    }
    lk.unlock();
    if (e != cudaSuccess) return cuda_fail(e, "graph launch / event chain", __LINE__);
    kernel_nodes.fetch_add(stages.size(), std::memory_order_relaxed);
    if (n_sm_copies) copy_nodes.fetch_add((uint64_t)n_sm_copies, std::memory_order_relaxed);
    if (has_signal) signal_nodes.fetch_add(1, std::memory_order_relaxed);
    return 0;
}

int set_ctx::poll() {
    bind_thread();
    for (int s = 0; s < H; ++s) {
        cudaError_t e = cudaStreamQuery(streams[s]);
        if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(e, "asynchronous failure on a work stream", __LINE__);
    }
    return 0;
}

void set_ctx::finish(int exec, int slot, const JobDesc&) {
    if (stamps) {
        StampRec r{(uint32_t)(slot % Hw), __atomic_load_n(&ts_host[(size_t)slot * 8], __ATOMIC_ACQUIRE),
                   __atomic_load_n(&ts_host[(size_t)slot * 8 + 1], __ATOMIC_ACQUIRE)};
        // The signal thread stores the end stamp and then the completion word, unfenced: the two stores may reach host
        // memory in either order (seen on B200, rarely -- the reason the job's OUTPUT is never written by
        // the grid that stores the word).  An end stamp older than the start stamp is the previous job's: wait for ours.
        for (uint64_t t0 = now_ns(); r.end < r.start && now_ns() - t0 < 200000;)
            r.end = __atomic_load_n(&ts_host[(size_t)slot * 8 + 1], __ATOMIC_ACQUIRE);
        if (r.start != 0 && r.end >= r.start) {
            stamp_lock.lock();
            if (stamp_recs.size() < (1u << 22)) stamp_recs.push_back(r);
            stamp_lock.unlock();
        }
    }
    ExecState& es = execs[exec];
    if (cfg.debug_sentinel && cfg.io == SET_IO_HOST && es.out) {
        // test hook (set.h debug_sentinel): this is the moment the job's completion was observed and the slot is about to
        // be released.  The caller pre-filled host_out with the sentinel; a D2H region whose first or last word still
        // holds it means the completion overtook the output.
        bool early = false;
        for (size_t i = 0; i < bufs.size(); ++i) {
            const uint64_t n = eval(bufs[i].d2h_bytes, es.dims);
            if (n < 4) continue;
            const char* base = (const char*)es.out + eval(bufs[i].d2h_host_off, es.dims);
            uint32_t first, last;  // host_out need not be 4-byte aligned
            memcpy(&first, const_cast<const char*>(static_cast<const volatile char*>(base)), 4);
            memcpy(&last, const_cast<const char*>(static_cast<const volatile char*>(base + ((n - 4) & ~3ull))), 4);
            early = early || first == cfg.debug_sentinel || last == cfg.debug_sentinel;
        }
        if (early) early_completions.fetch_add(1, std::memory_order_relaxed);
    }
    if (es.staged) {  // staged D2H: pinned ring -> caller's pageable memory, on the callback thread
        memcpy(es.user_out, es.stage_out, es.out_bytes);
        es.staged = false;
        es.in = nullptr;  // force the next job's copy nodes to be re-pointed
        es.out = nullptr;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Baseline models.  All run on the caller's thread inside set_submit / set_drain.
// ---------------------------------------------------------------------------------------------------------
int set_ctx::plain_job(int slot, const JobDesc& job) {
    // "Synchronous model": individual copies and kernel launches, no graph
    int s = slot % Hw;
    cudaStream_t st = streams[s];
    SlotMem& sm = slots[slot];
    if (sm.used) {  // buffer reuse guarded by event synchronisation
        uint64_t t0 = now_ns();
        CK(cudaEventSynchronize(sm.done));
        ns_sync.fetch_add(now_ns() - t0, std::memory_order_relaxed);
        base_completed.fetch_add(1, std::memory_order_relaxed);
    }
    cudaMemcpyKind kin = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    cudaMemcpyKind kout = cfg.io == SET_IO_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (bd.flags & SET_BUF_ZERO)
            CK(cudaMemsetAsync((char*)sm.buf[i] + eval(bd.zero_off, job.dims), 0, eval(bd.zero_bytes, job.dims), st));
        if (!expr_is_zero(bd.h2d_bytes)) {
            if (h2d_sm[i]) {  // the same node list as the job graph, launched one by one
                CopyArgs ca;
                copy_params(ca, slot, (int)i, true, job.in, job.dims, job.out);
                CK(cudaLaunchKernel(ca.kp.func, ca.kp.gridDim, ca.kp.blockDim, ca.ptrs, 0, st));
            } else {
                CK(cudaMemcpyAsync((char*)sm.buf[i] + eval(bd.h2d_dev_off, job.dims), (const char*)job.in + eval(bd.h2d_host_off, job.dims),
                                   eval(bd.h2d_bytes, job.dims), kin, st));
            }
        }
    }
    for (auto& sd : stages) {
        ArgPack ap;
        dim3 grid;
        if (int rc = build_args(sd, slot, job.dims, ap, grid)) return rc;
        CK(cudaLaunchKernel(sd.func, grid, dim3(sd.block[0], sd.block[1] ? sd.block[1] : 1, sd.block[2] ? sd.block[2] : 1),
                            ap.ptrs, sd.smem_bytes, st));
    }
    kernel_nodes.fetch_add(stages.size(), std::memory_order_relaxed);
    for (size_t i = 0; i < bufs.size(); ++i) {
        const set_buffer_desc& bd = bufs[i];
        if (!expr_is_zero(bd.d2h_bytes)) {
            if (d2h_sm[i]) {
                CopyArgs ca;
                copy_params(ca, slot, (int)i, false, job.out, job.dims);
                CK(cudaLaunchKernel(ca.kp.func, ca.kp.gridDim, ca.kp.blockDim, ca.ptrs, 0, st));
            } else {
                CK(cudaMemcpyAsync((char*)job.out + eval(bd.d2h_host_off, job.dims), (char*)sm.buf[i] + eval(bd.d2h_dev_off, job.dims),
                                   eval(bd.d2h_bytes, job.dims), kout, st));
            }
        }
    }
    if (n_sm_copies) copy_nodes.fetch_add((uint64_t)n_sm_copies, std::memory_order_relaxed);
    CK(cudaEventRecord(sm.done, st));
    sm.used = true;
    return 0;
}

int set_ctx::baseline_flush() {
    // Static batching: exec i <- job i, fixed stream i mod S, then the host
    // synchronises with every stream before the next batch may touch the buffers.
    if (batch.empty()) return 0;
    uint64_t t0 = now_ns();
    for (size_t i = 0; i < batch.size(); ++i) {
        bool dummy;
        int e = (int)i * epp;
        if (int rc = bind(e, (int)i, batch[i], &dummy)) return rc;
        CK(cudaGraphLaunch(execs[e].exec, streams[i % Hw]));
    }
    base_launched.fetch_add(batch.size(), std::memory_order_relaxed);
    kernel_nodes.fetch_add(stages.size() * batch.size(), std::memory_order_relaxed);
    copy_nodes.fetch_add((uint64_t)n_sm_copies * batch.size(), std::memory_order_relaxed);
    uint64_t t1 = now_ns();
    for (int s = 0; s < H; ++s) CK(cudaStreamSynchronize(streams[s]));
    uint64_t t2 = now_ns();
    for (size_t i = 0; i < batch.size(); ++i) finish((int)i * epp, (int)i, batch[i]);
    base_completed.fetch_add(batch.size(), std::memory_order_relaxed);
    base_ns_launch.fetch_add(t1 - t0, std::memory_order_relaxed);
    ns_sync.fetch_add(t2 - t1, std::memory_order_relaxed);
    batch.clear();
    return 0;
}

int set_ctx::baseline_submit(const JobDesc& job) {
    uint64_t t0 = now_ns();
    int rc = 0;
    bind_thread();
    if (int r = check_sizes(job.dims)) return r;
    switch (cfg.mode) {
        case SET_MODE_PLAIN_STREAMS: {
            if (cfg.io == SET_IO_HOST && (!is_pinned(job.in) || !is_pinned(job.out)))
                return fail(SET_ERR_INVALID, "baseline modes need pinned host buffers");
            int slot = (int)(base_ticket++ % (uint64_t)b);
            rc = plain_job(slot, job);
            base_launched.fetch_add(1, std::memory_order_relaxed);
            break;
        }
        case SET_MODE_BATCH_SYNC:
            batch.push_back(job);
            if ((int)batch.size() == b) rc = baseline_flush();
            break;
        case SET_MODE_SINGLE_GRAPH: {
            // Graph model: one pre-instantiated exec replayed on one stream; stream order alone
            // protects the single buffer set.  Updating an exec whose previous launch is still running is
            // legal in CUDA: the update applies to later launches.
            bool dummy;
            JobDesc j = job;
            rc = bind(0, 0, j, &dummy);
            if (rc == 0) {
                cudaError_t e = cudaGraphLaunch(execs[0].exec, streams[0]);
                if (e != cudaSuccess) rc = cuda_fail(e, "cudaGraphLaunch", __LINE__);
            }
            base_launched.fetch_add(1, std::memory_order_relaxed);
            kernel_nodes.fetch_add(stages.size(), std::memory_order_relaxed);
            copy_nodes.fetch_add((uint64_t)n_sm_copies, std::memory_order_relaxed);
            break;
        }
        case SET_MODE_MUTEX_QUEUE: {
            if (cfg.io == SET_IO_HOST && (!is_pinned(job.in) || !is_pinned(job.out)))
                return fail(SET_ERR_INVALID, "baseline modes need pinned host buffers");
            std::unique_lock<std::mutex> g(mq_mu);
            mq_cv.wait(g, [&] { return (int)mq_queue.size() < b * q || err.load() != 0; });  // bounded like SET's queues
            if (int e = err.load()) return e;
            mq_queue.push_back(job);
            g.unlock();
            mq_cv.notify_all();
            break;
        }
        default:
            return fail(SET_ERR_INVALID, "mode %d not implemented", cfg.mode);
    }
    if (rc == 0) base_submitted.fetch_add(1, std::memory_order_relaxed);
    base_ns_submit.fetch_add(now_ns() - t0, std::memory_order_relaxed);
    return rc;
}

void set_ctx::mq_loop() {
    bind_thread();
    std::vector<char> busy((size_t)b, 0);
    std::vector<JobDesc> running((size_t)b);
    while (!mq_stop.load(std::memory_order_acquire)) {
        bool progressed = false;
        for (int w = 0; w < b; ++w) {  // O(b) host-side completion queries per round
            if (busy[w]) {
                cudaError_t e = cudaEventQuery(slots[w].done);
                mq_queries.fetch_add(1, std::memory_order_relaxed);
                if (e == cudaErrorNotReady) continue;
                if (e != cudaSuccess) cuda_fail(e, "cudaEventQuery", __LINE__);
                finish(w * epp, w, running[w]);
                busy[w] = 0;
                base_completed.fetch_add(1, std::memory_order_release);
                progressed = true;
                mq_cv.notify_all();
            }
            JobDesc j;
            {
                std::lock_guard<std::mutex> g(mq_mu);  // the shared queue's lock, taken for every dispatch
                if (mq_queue.empty()) continue;
                j = mq_queue.front();
                mq_queue.pop_front();
            }
            mq_cv.notify_all();
            uint64_t t0 = now_ns();
            bool dummy;
            int rc = err.load() ? err.load() : bind(w * epp, w, j, &dummy);
            if (rc == 0) {
                cudaError_t e = cudaGraphLaunch(execs[w * epp].exec, streams[w % Hw]);
                if (e == cudaSuccess) e = cudaEventRecord(slots[w].done, streams[w % Hw]);
                if (e != cudaSuccess) rc = cuda_fail(e, "graph launch (queue model)", __LINE__);
            }
            base_ns_launch.fetch_add(now_ns() - t0, std::memory_order_relaxed);
            if (rc != 0) {  // keep the books balanced so that drain returns
                base_completed.fetch_add(1, std::memory_order_release);
                mq_cv.notify_all();
                continue;
            }
            running[w] = j;
            busy[w] = 1;
            base_launched.fetch_add(1, std::memory_order_relaxed);
            kernel_nodes.fetch_add(stages.size(), std::memory_order_relaxed);
            copy_nodes.fetch_add((uint64_t)n_sm_copies, std::memory_order_relaxed);
            progressed = true;
        }
        if (!progressed) {
            bool any = false;
            for (int w = 0; w < b; ++w) any = any || busy[w];
            if (!any) {  // nothing in flight and nothing queued: sleep until a submit arrives
                std::unique_lock<std::mutex> g(mq_mu);
                mq_cv.wait_for(g, std::chrono::milliseconds(1), [&] { return !mq_queue.empty() || mq_stop.load(); });
            } else {
                cpu_relax();
            }
        }
    }
}

int set_ctx::baseline_drain() {
    bind_thread();
    if (cfg.mode == SET_MODE_BATCH_SYNC)
        if (int rc = baseline_flush()) return rc;
    if (cfg.mode == SET_MODE_MUTEX_QUEUE) {
        uint64_t t0 = now_ns();
        std::unique_lock<std::mutex> g(mq_mu);
        while (base_completed.load(std::memory_order_acquire) < base_submitted.load() && err.load() == 0)
            mq_cv.wait_for(g, std::chrono::microseconds(200));
        ns_sync.fetch_add(now_ns() - t0, std::memory_order_relaxed);
        return err.load();
    }
    uint64_t t0 = now_ns();
    for (int s = 0; s < H; ++s) CK(cudaStreamSynchronize(streams[s]));
    ns_sync.fetch_add(now_ns() - t0, std::memory_order_relaxed);
    for (auto& sm : slots) sm.used = false;
    base_completed.store(base_submitted.load());
    return err.load();
}

// =========================================================================================================
// C ABI
// =========================================================================================================
extern "C" {

set_status set_create_ex(const set_config* cfg_in, set_ctx** out) {
    if (!out) return SET_ERR_INVALID;
    *out = nullptr;
    if (!cfg_in || cfg_in->struct_bytes != sizeof(set_config)) return SET_ERR_INVALID;
    set_config cfg = *cfg_in;
    if (cfg.num_streams < 1 || cfg.max_inflight < 1 || cfg.num_streams > 1024 || cfg.max_inflight > (1 << 16)) return SET_ERR_INVALID;
    if (cfg.mode < SET_MODE_SET || cfg.mode > SET_MODE_MUTEX_QUEUE) return SET_ERR_INVALID;
    if (cfg.io != SET_IO_HOST && cfg.io != SET_IO_DEVICE) return SET_ERR_INVALID;
    if (cfg.queue_capacity < 0 || cfg.queue_capacity > 64 || cfg.num_dispatchers < 0 || cfg.num_dispatchers > 64) return SET_ERR_INVALID;
    if (cfg.queue_capacity == 0) cfg.queue_capacity = 2;
    if (cfg.num_dispatchers == 0) cfg.num_dispatchers = 1;
    if (cfg.spin_us == 0) cfg.spin_us = 50;
    if (cfg.callback_mode < SET_CB_DEFAULT || cfg.callback_mode > SET_CB_HOST_NODE) return SET_ERR_INVALID;
    if (cfg.callback_mode == SET_CB_DEFAULT) cfg.callback_mode = SET_CB_FLAG_POLL;
    if (cfg.completion_fence < SET_FENCE_DEFAULT || cfg.completion_fence > SET_FENCE_NONE) return SET_ERR_INVALID;
    if (cfg.completion_fence == SET_FENCE_DEFAULT) cfg.completion_fence = SET_FENCE_SYSTEM;
    if (cfg.streams_per_lane < 0 || cfg.streams_per_lane > 4096) return SET_ERR_INVALID;
    if (cfg.completion_thread < 0 || cfg.completion_thread > 2) return SET_ERR_INVALID;
    // Measured on B200: once the copy-in kernels keep the link full, config 1 end to end sits at the edge between
    // link-bound and host-bound -- on a box whose cudaGraphLaunch takes 2.2 us instead of 1.95 us a dispatcher that also polls and
    // completes delivers 341-355 K jobs/s, with a completion thread of its own 375-377 K (the link bound).  Binding at launch adds
    // nothing to that (349-351 K without the thread, 376 K with it) and costs config 4 device-resident 10 % (its 3.4 us full
    // rebinds land on the dispatcher): off by default.
    // The hand-off from the completion thread to the dispatcher adds a fraction of a microsecond to every job's turnaround, which
    // a latency-bound configuration feels (config 0, 8 in flight: 316 K -> 297 K jobs/s): the thread is the default from 16 slots up.
    if (cfg.completion_thread == 0) cfg.completion_thread = cfg.max_inflight >= 16 ? 1 : 2;
    if (cfg.bind_at_launch < 0 || cfg.bind_at_launch > 2) return SET_ERR_INVALID;
    if (cfg.bind_at_launch == 0) cfg.bind_at_launch = 2;
    // Default (measured on B200): with host I/O a job's chain is latency-bound (its copy-in waits on the link),
    // so every slot gets a CUDA stream of its own -- the paper's worker W_i = (S_i, G_i, M_i), PAPER.md:110 -- and b chains are
    // in flight instead of S (config 1 end to end 201 K -> 316 K jobs/s, config 0 227 K -> 336 K).  With device-resident I/O
    // the host's launch rate is the limit and more streams only make each launch dearer (404 K -> 360 K): one per lane.
    // The default never goes beyond 32 CUDA streams in all (b = 4096 would otherwise ask for 4096 of them).
    if (cfg.streams_per_lane == 0) cfg.streams_per_lane = cfg.io == SET_IO_HOST ? std::max(1, 32 / cfg.num_streams) : 1;
    if (cfg.mode == SET_MODE_SINGLE_GRAPH) {  // one worker, one stream, one exec by definition
        cfg.num_streams = 1;
        cfg.max_inflight = 1;
        cfg.streams_per_lane = 1;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return SET_ERR_CUDA;
    }
    int dev = cfg.device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return SET_ERR_CUDA;
    if (dev >= ndev) return SET_ERR_INVALID;
    if (cudaSetDevice(dev) != cudaSuccess) return SET_ERR_CUDA;

    set_ctx* c = new (std::nothrow) set_ctx();
    if (!c) return SET_ERR_NOMEM;
    c->cfg = cfg;
    c->device = dev;
    // Nsight Compute's injection library is not safe against concurrent graph update + launch (profiles/r1_ncu.md):
    // serialise them whenever a CUDA injection library is present, unless the environment says otherwise
    for (const char* v : {"CUDA_INJECTION64_PATH", "NV_NSIGHT_INJECTION_PORT_BASE", "NV_NSIGHT_INJECTION_TRANSPORT_TYPE",
                          "NV_COMPUTE_PROFILER_PERFWORKS_DIR", "NV_COMPUTE_PROFILER_LOCAL_CONNECTION_OVERRIDE"})
        if (const char* e = getenv(v)) c->driver_lock = c->driver_lock || e[0] != 0;
    if (const char* dlk = getenv("SET_DRIVER_LOCK")) c->driver_lock = dlk[0] == '1';
    if (const char* cmb = getenv("SET_COPY_MAX_BLOCKS")) c->copy_max_blocks = (uint32_t)atoi(cmb);
    c->S = cfg.num_streams;
    c->b = ((cfg.max_inflight + c->S - 1) / c->S) * c->S;
    c->q = cfg.queue_capacity;
    c->epp = c->q + 1;
    c->own_streams = cfg.streams == nullptr;
    // CUDA streams behind each logical stream (set.h streams_per_lane): never more than the lane has slots
    c->L = c->own_streams ? std::max(1, std::min(cfg.streams_per_lane, c->b / c->S)) : 1;
    c->H = c->S * c->L;
    c->Hw = c->H;
    c->streams.resize(c->H);
    c->notify.resize(c->H);
    c->stream_locks.reset(new SpinLock[c->H]);
    bool ok = true;
    for (int s = 0; s < c->H && ok; ++s) {
        if (c->own_streams)
            ok = cudaStreamCreateWithFlags(&c->streams[s], cudaStreamNonBlocking) == cudaSuccess;
        else
            c->streams[s] = (cudaStream_t)cfg.streams[s];
        ok = ok && cudaStreamCreateWithFlags(&c->notify[s], cudaStreamNonBlocking) == cudaSuccess;
    }
    c->slots.resize(c->b);
    c->cbargs.resize(c->b);
    for (int w = 0; w < c->b && ok; ++w) {
        ok = cudaEventCreateWithFlags(&c->slots[w].done, cudaEventDisableTiming) == cudaSuccess;
        c->cbargs[w] = {c, w};
    }
    if (!ok) {
        cudaGetLastError();
        delete c;
        return SET_ERR_CUDA;
    }
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
        c->encode_tiled = (PFN_encodeTiled)fn;
    else
        cudaGetLastError();
    if (cfg.mode == SET_MODE_SET && cfg.callback_mode == SET_CB_FLAG_POLL) {
        // one 64-byte line per slot in mapped pinned memory; the GPU stores, the dispatcher loads
        size_t bytes = (size_t)c->b * kFlagStride * sizeof(uint32_t);
        if (cudaHostAlloc((void**)&c->flags_host, bytes, cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess ||
            cudaHostGetDevicePointer((void**)&c->flags_dev, c->flags_host, 0) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return SET_ERR_CUDA;
        }
        memset(c->flags_host, 0, bytes);
        c->flag_poll = true;
    }
    if (cfg.timestamps) {
        size_t bytes = (size_t)c->b * 8 * sizeof(unsigned long long);
        if (cudaHostAlloc((void**)&c->ts_host, bytes, cudaHostAllocPortable | cudaHostAllocMapped) != cudaSuccess ||
            cudaHostGetDevicePointer((void**)&c->ts_dev, c->ts_host, 0) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return SET_ERR_CUDA;
        }
        memset(c->ts_host, 0, bytes);
        c->stamps = true;
        c->stamp_recs.reserve(1 << 16);
    }
    if (cfg.mode == SET_MODE_SET)
        c->sched.reset(new Scheduler(c, c->H, c->b, c->q, cfg.num_dispatchers, cfg.steal_policy, cfg.spin_us, cfg.completion_thread == 1));
    *out = c;
    return SET_OK;
}

set_status set_create(int num_streams, int max_inflight, set_ctx** out) {
    set_config cfg{};
    cfg.struct_bytes = sizeof(cfg);
    cfg.num_streams = num_streams;
    cfg.max_inflight = max_inflight;
    cfg.mode = SET_MODE_SET;
    cfg.io = SET_IO_HOST;
    cfg.device = -1;
    return set_create_ex(&cfg, out);
}

set_status set_register_pipeline(set_ctx* c, const set_stage_desc* stages, int num_stages, const set_buffer_desc* bufs,
                                 int num_bufs) {
    if (!c) return SET_ERR_INVALID;
    if (int e = c->err.load()) return e;
    if (c->registered) return SET_ERR_STATE;
    if (!stages || !bufs || num_stages < 1 || num_stages > SET_MAX_STAGES || num_bufs < 1 || num_bufs > SET_MAX_BUFFERS)
        return SET_ERR_INVALID;
    const uint32_t unit[4] = {1, 1, 1, 1};
    for (int s = 0; s < num_stages; ++s) {
        const set_stage_desc& st = stages[s];
        if (!st.func || st.num_args < 0 || st.num_args > SET_MAX_ARGS || st.block[0] == 0) return SET_ERR_INVALID;
        if ((uint64_t)st.block[0] * (st.block[1] ? st.block[1] : 1) * (st.block[2] ? st.block[2] : 1) > 1024) return SET_ERR_INVALID;
        for (int a = 0; a < st.num_args; ++a) {
            const set_arg_desc& d = st.args[a];
            if (d.kind < SET_ARG_BUFFER || d.kind > SET_ARG_COND) return SET_ERR_INVALID;
            if ((d.kind == SET_ARG_BUFFER || d.kind == SET_ARG_TMAP2D) && (d.index < 0 || d.index >= num_bufs)) return SET_ERR_INVALID;
            if (d.kind == SET_ARG_DIM && (d.index < 0 || d.index >= SET_MAX_DIMS)) return SET_ERR_INVALID;
        }
    }
    {  // loop structure (set.h SET_STAGE_LOOP_BEGIN): at most one loop, properly closed; a loop pipeline is bound to its
       // slot, so no kernel of it may depend on the job's dims; SET_ARG_COND only inside the loop
        bool any_loop = false, in_loop = false, closed = false;
        int body_stages = 0;
        for (int s = 0; s < num_stages; ++s) any_loop = any_loop || (stages[s].flags & SET_STAGE_LOOP_BEGIN);
        for (int s = 0; s < num_stages; ++s) {
            const set_stage_desc& st = stages[s];
            if (st.flags & SET_STAGE_LOOP_BEGIN) {
                if (in_loop || closed) return SET_ERR_INVALID;
                in_loop = true;
            }
            auto dim_free = [](const set_size_expr& e) { return e.per_unit == 0 || e.dim_mask == 0; };
            for (int a = 0; a < st.num_args; ++a) {
                const set_arg_desc& d = st.args[a];
                if (d.kind == SET_ARG_COND && !in_loop) return SET_ERR_INVALID;
                if (in_loop && (d.kind == SET_ARG_DIM || !dim_free(d.offset))) return SET_ERR_INVALID;
            }
            if (in_loop)
                for (int k = 0; k < 3; ++k)
                    if (!dim_free(st.grid[k].count)) return SET_ERR_INVALID;
            if (in_loop) ++body_stages;
            if (st.flags & SET_STAGE_LOOP_END) {
                if (!in_loop) return SET_ERR_INVALID;
                in_loop = false;
                closed = true;
            }
        }
        if (in_loop) return SET_ERR_INVALID;
        // Measured on B200 / CUDA 12.9 (profiles/r2_probes.md section 3): a WHILE body of TWO kernel nodes (relaxation ->
        // control) ended in cudaErrorLaunchFailure -- sticky, the context is lost -- about once in 10^5 jobs with 8 such
        // graphs in flight (never with 4); bodies of 3 to 9 nodes ran 6.6 million jobs without one.  Refuse the short body.
        if (any_loop && body_stages < kMinLoopBodyStages)
            return c->fail(SET_ERR_INVALID, "a loop body needs at least %d stages (two-node WHILE bodies are not reliable on this driver)",
                           kMinLoopBodyStages);
        if (any_loop && c->cfg.mode == SET_MODE_SET && c->cfg.steal_policy == SET_STEAL_RETARGET) return SET_ERR_INVALID;
    }
    for (int i = 0; i < num_bufs; ++i) {
        if (bufs[i].bytes == 0) return SET_ERR_INVALID;
        if ((bufs[i].flags & SET_BUF_ZERO) && eval(bufs[i].zero_bytes, unit) == 0) return SET_ERR_INVALID;
    }
    c->bind_thread();
    c->stages.assign(stages, stages + num_stages);
    c->bufs.assign(bufs, bufs + num_bufs);
    if (c->check_sizes(unit)) return SET_ERR_INVALID;

    // ---- memory slots M_w: b pre-allocated, reusable device buffer sets
    auto align_up = [](uint64_t v) { return (v + 1023) & ~1023ull; };
    uint64_t per_slot = 0;
    for (auto& bd : c->bufs) per_slot += align_up(bd.bytes);
    char* arena = (char*)c->cfg.device_arena;
    if (arena) {
        arena = (char*)align_up((uint64_t)(uintptr_t)arena);
        uint64_t lost = (uint64_t)(arena - (char*)c->cfg.device_arena);
        if (c->cfg.device_arena_bytes < lost + per_slot * (uint64_t)c->b)
            return c->fail(SET_ERR_NOMEM, "device arena too small: need %llu bytes", (unsigned long long)(lost + per_slot * c->b));
    }
    for (int w = 0; w < c->b; ++w) {
        char* base;
        if (arena) {
            base = arena + per_slot * (uint64_t)w;
        } else {
            void* p = nullptr;
            cudaError_t e = cudaMalloc(&p, per_slot);
            if (e != cudaSuccess) {
                cudaGetLastError();
                return c->fail(SET_ERR_NOMEM, "cudaMalloc of %llu bytes for slot %d failed: %s", (unsigned long long)per_slot, w,
                               cudaGetErrorString(e));
            }
            c->owned_dev.push_back(p);
            base = (char*)p;
        }
        uint64_t off = 0;
        for (size_t i = 0; i < c->bufs.size(); ++i) {
            c->slots[w].buf[i] = base + off;
            off += align_up(c->bufs[i].bytes);
        }
    }
    // ---- placeholder operands for the template graph
    uint64_t pin = 16, pout = 16;
    for (auto& bd : c->bufs) {
        pin = std::max(pin, eval(bd.h2d_host_off, unit) + eval(bd.h2d_bytes, unit));
        pout = std::max(pout, eval(bd.d2h_host_off, unit) + eval(bd.d2h_bytes, unit));
    }
    c->in_extent_unit = pin;
    c->out_extent_unit = pout;
    if (c->cfg.io == SET_IO_DEVICE) {
        if (cudaMalloc(&c->ph_in, pin) != cudaSuccess || cudaMalloc(&c->ph_out, pout) != cudaSuccess) {
            cudaGetLastError();
            return c->fail(SET_ERR_NOMEM, "placeholder allocation failed");
        }
    } else {
        if (cudaHostAlloc(&c->ph_in, pin, cudaHostAllocPortable) != cudaSuccess ||
            cudaHostAlloc(&c->ph_out, pout, cudaHostAllocPortable) != cudaSuccess) {
            cudaGetLastError();
            return c->fail(SET_ERR_NOMEM, "pinned placeholder allocation failed");
        }
    }
    // ---- which copies become SET_K_COPY kernel nodes: at most sm_copy_max_bytes; a size that depends on the job's dims counts
    // with its buffer's capacity (the node's byte count and grid are part of the per-job update either way)
    {
        // default 256 KiB: below that a copy-engine node costs more in engine hand-off than the copy itself, across the
        // host link and (SET_IO_DEVICE) inside HBM alike (profiles/r1_bench.md, graph_variants)
        int64_t lim = c->cfg.sm_copy_max_bytes != 0 ? c->cfg.sm_copy_max_bytes : 262144;
        for (size_t i = 0; i < c->bufs.size(); ++i) {
            const set_buffer_desc& bd = c->bufs[i];
            auto small = [&](const set_size_expr& e) {
                if (expr_is_zero(e)) return false;
                return (int64_t)(e.per_unit == 0 ? e.fixed : bd.bytes) <= lim;
            };
            c->h2d_sm[i] = small(bd.h2d_bytes);
            c->d2h_sm[i] = small(bd.d2h_bytes);
            c->n_sm_copies += (int)c->h2d_sm[i] + (int)c->d2h_sm[i];
        }
        for (auto& st : c->stages) c->pdl = c->pdl || (st.flags & SET_STAGE_PDL);
        // output-address forwarding: needs an SM copy-in node to carry the address and at least one SM copy-out node to use it
        const char* fo = getenv("SET_FORWARD_OUT");
        if (!(fo && fo[0] == '0')) {
            int first_in = -1;
            bool any_out = false;
            for (size_t i = 0; i < c->bufs.size(); ++i) {
                if (c->h2d_sm[i] && first_in < 0) first_in = (int)i;
                any_out = any_out || c->d2h_sm[i];
            }
            if (first_in >= 0 && any_out) {
                if (cudaMalloc((void**)&c->fwd_dev, 2 * sizeof(void*) * (size_t)c->b) != cudaSuccess ||
                    cudaMemset(c->fwd_dev, 0, 2 * sizeof(void*) * (size_t)c->b) != cudaSuccess) {
                    cudaGetLastError();
                    return c->fail(SET_ERR_NOMEM, "allocation of the forwarding words failed");
                }
                c->fwd_buf = first_in;
                int n_out = 0, only_out = -1;
                for (size_t i = 0; i < c->bufs.size(); ++i) {
                    c->d2h_ind[i] = c->d2h_sm[i];
                    if (!expr_is_zero(c->bufs[i].d2h_bytes)) {
                        n_out += 1;
                        only_out = (int)i;
                    }
                }
                // fold the completion signal into the copy-out node where the job has exactly one and the SMs do it
                const char* fs = getenv("SET_FUSE_SIGNAL");
                if (c->flag_poll && n_out == 1 && c->d2h_sm[only_out] && !(fs && fs[0] == '0')) c->fused_signal_buf = only_out;
            }
        }
    }
    {
        bool in_loop = false;
        for (auto& st : c->stages) {
            c->slot_graphs = c->slot_graphs || (st.flags & SET_STAGE_LOOP_BEGIN);
            in_loop = in_loop || (st.flags & SET_STAGE_LOOP_BEGIN);
            c->stage_in_loop.push_back(in_loop ? 1 : 0);
            if (st.flags & SET_STAGE_LOOP_END) in_loop = false;
        }
    }
    if (c->slot_graphs && c->cfg.mode == SET_MODE_PLAIN_STREAMS)
        return c->fail(SET_ERR_INVALID, "a pipeline with a loop needs a job graph: SET_MODE_PLAIN_STREAMS cannot run it");
    if (c->slot_graphs && c->sched) c->sched->set_slot_bound(true);
    if (c->slot_graphs) {
        // Measured on B200 / CUDA 12.9 (profiles/r2_probes.md section 4): with more than 8 graphs holding a WHILE node in
        // flight at once, a launch now and then ends in cudaErrorLaunchFailure (about once in 10^5 jobs at 32 in flight,
        // never at 8).  Loop pipelines therefore run on at most 8 of the context's CUDA streams: the largest divisor of S
        // that is <= 8, so that slots w and w + H, which the scheduler polls as one in-order list, still share a stream.
        int lim = 1;
        for (int d = 1; d <= kMaxLoopStreams && d <= c->S; ++d)
            if (c->S % d == 0) lim = d;
        c->Hw = lim;
    }
    if (c->sched) c->sched->set_bind_at_launch(c->cfg.bind_at_launch == 1);
    c->nsets.resize(c->slot_graphs ? (size_t)c->b * c->epp : 1);
    if (!c->slot_graphs)
        if (int rc = c->build_graph(0, 0)) return rc;

    // ---- bounded pool of graph executables: q+1 per slot, each re-bound to its slot's M_w
    int nexec = c->b * c->epp;
    c->execs.resize(nexec);
    for (int e = 0; e < nexec; ++e) {
        bool needed = c->cfg.mode == SET_MODE_SET || (e % c->epp == 0);
        if (c->cfg.mode == SET_MODE_PLAIN_STREAMS) needed = false;
        if (!needed) continue;
        int slot = e / c->epp;
        if (c->slot_graphs)
            if (int rc = c->build_graph(slot, e)) return rc;
        cudaError_t er = cudaGraphInstantiate(&c->execs[e].exec, c->nodes_of_exec(e).graph, 0);
        if (er != cudaSuccess) return c->cuda_fail(er, "cudaGraphInstantiate", __LINE__);
        c->execs[e].bound_slot = c->slot_graphs ? slot : 0;  // the template was built on slot 0's buffers (or on this slot's)
        c->execs[e].in = c->ph_in;
        c->execs[e].out = c->ph_out;
        if (slot != 0 && !c->slot_graphs) {
            JobDesc j;
            j.in = c->ph_in;
            j.out = c->ph_out;
            bool dummy;
            // placeholders are pinned (or device) memory, so this never stages
            if (int rc = c->bind(e, slot, j, &dummy)) return rc;
        }
    }
    c->full_rebinds.store(0);
    c->host_rebinds.store(0);
    c->ns_bind.store(0);
    c->registered = true;
    // one job in flight per CUDA stream: a WHILE graph queued on a stream behind a running one slows both down (8 streams:
    // 54 K SSSP jobs/s with 8 slots, 34 K with 16 or 32), so the slots beyond the streams are taken out of service
    if (c->slot_graphs && c->sched) c->sched->retire_slots(c->Hw);
    if (c->cfg.mode == SET_MODE_MUTEX_QUEUE) c->mq_thread = std::thread([c] { c->mq_loop(); });
    return SET_OK;
}

static set_status submit_one(set_ctx* c, const JobDesc& j) {
    if (c->cfg.mode == SET_MODE_SET) return c->sched->submit(j);
    return c->baseline_submit(j);
}

set_status set_submit_dims(set_ctx* c, uint64_t job_id, const void* host_in, void* host_out, const uint32_t dims[SET_MAX_DIMS]) {
    if (!c || !host_in || !host_out) return SET_ERR_INVALID;
    if (int e = c->err.load()) return e;
    if (!c->registered) return SET_ERR_STATE;
    JobDesc j;
    j.id = job_id;
    j.in = host_in;
    j.out = host_out;
    if (dims) memcpy(j.dims, dims, sizeof(j.dims));
    return submit_one(c, j);
}

set_status set_submit(set_ctx* c, uint64_t job_id, const void* host_in, void* host_out) {
    return set_submit_dims(c, job_id, host_in, host_out, nullptr);
}

set_status set_try_submit_dims(set_ctx* c, uint64_t job_id, const void* host_in, void* host_out, const uint32_t dims[SET_MAX_DIMS]) {
    if (!c || !host_in || !host_out) return SET_ERR_INVALID;
    if (int e = c->err.load()) return e;
    if (!c->registered) return SET_ERR_STATE;
    if (c->cfg.mode != SET_MODE_SET) return SET_ERR_STATE;  // the baseline models have no queue to find full
    JobDesc j;
    j.id = job_id;
    j.in = host_in;
    j.out = host_out;
    if (dims) memcpy(j.dims, dims, sizeof(j.dims));
    return c->sched->submit(j, /*blocking=*/false);
}

set_status set_submit_batch(set_ctx* c, int64_t n, uint64_t first_id, const uint64_t* job_ids, const void* const* host_ins,
                            void* const* host_outs, const uint32_t* dims) {
    if (!c || n < 0 || (n > 0 && (!host_ins || !host_outs))) return SET_ERR_INVALID;
    for (int64_t i = 0; i < n; ++i) {
        set_status rc = set_submit_dims(c, job_ids ? job_ids[i] : first_id + (uint64_t)i, host_ins[i], host_outs[i],
                                        dims ? dims + 4 * i : nullptr);
        if (rc != SET_OK) return rc;
    }
    return SET_OK;
}

set_status set_drain(set_ctx* c) {
    if (!c) return SET_ERR_INVALID;
    if (!c->registered) return c->err.load();
    int rc = c->cfg.mode == SET_MODE_SET ? c->sched->drain() : c->baseline_drain();
    if (int e = c->err.load()) return e;
    return rc;
}

set_status set_destroy(set_ctx* c) {
    if (!c) return SET_OK;
    cudaSetDevice(c->device);
    if (c->registered && c->err.load() == 0) set_drain(c);
    if (c->sched) c->sched->stop();
    if (c->mq_thread.joinable()) {
        c->mq_stop.store(true);
        c->mq_cv.notify_all();
        c->mq_thread.join();
    }
    for (auto s : c->streams) cudaStreamSynchronize(s);
    for (auto s : c->notify) cudaStreamSynchronize(s);  // host functions have returned after this
    for (auto& es : c->execs) {
        if (es.exec) cudaGraphExecDestroy(es.exec);
        if (es.stage_in) cudaFreeHost(es.stage_in);
        if (es.stage_out) cudaFreeHost(es.stage_out);
    }
    for (auto& ns : c->nsets)
        if (ns.graph) cudaGraphDestroy(ns.graph);
    for (auto& sm : c->slots) {
        if (sm.done) cudaEventDestroy(sm.done);
        if (sm.t0) cudaEventDestroy(sm.t0);
    }
    for (auto p : c->owned_dev) cudaFree(p);
    if (c->ph_in) (c->cfg.io == SET_IO_DEVICE ? cudaFree(c->ph_in) : cudaFreeHost(c->ph_in));
    if (c->ph_out) (c->cfg.io == SET_IO_DEVICE ? cudaFree(c->ph_out) : cudaFreeHost(c->ph_out));
    for (auto& ha : c->host_allocs) cudaFreeHost(ha.first);
    if (c->fwd_dev) cudaFree(c->fwd_dev);
    if (c->flags_host) cudaFreeHost(c->flags_host);
    if (c->ts_host) cudaFreeHost(c->ts_host);
    for (int s = 0; s < c->H; ++s) {
        if (c->own_streams && c->streams[s]) cudaStreamDestroy(c->streams[s]);
        if (c->notify[s]) cudaStreamDestroy(c->notify[s]);
    }
    cudaGetLastError();
    c->sched.reset();
    delete c;
    return SET_OK;
}

void* set_host_alloc(set_ctx* c, size_t bytes) {
    if (!c || bytes == 0) return nullptr;
    c->bind_thread();
    void* p = nullptr;
    if (cudaHostAlloc(&p, bytes, cudaHostAllocPortable) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    {
        std::lock_guard<std::mutex> g(c->hostmu);
        c->host_allocs.push_back({p, bytes});
    }
    c->add_pinned_range(p, bytes);
    return p;
}

void set_host_free(set_ctx* c, void* p) {
    if (!c || !p) return;
    std::lock_guard<std::mutex> g(c->hostmu);
    for (size_t i = 0; i < c->host_allocs.size(); ++i)
        if (c->host_allocs[i].first == p) {
            c->range_lock.lock();
            for (size_t k = 0; k < c->pinned_ranges.size(); ++k)
                if (c->pinned_ranges[k].lo == (uintptr_t)p) {
                    c->pinned_ranges.erase(c->pinned_ranges.begin() + (long)k);
                    break;
                }
            c->range_lock.unlock();
            cudaFreeHost(p);
            c->host_allocs.erase(c->host_allocs.begin() + (long)i);
            return;
        }
}

set_status set_host_register(set_ctx* c, const void* p, size_t bytes) {
    if (!c || !p || bytes == 0) return SET_ERR_INVALID;
    c->bind_thread();
    // both ends must be pinned host memory that the device addresses at the host's own address (SM copies dereference it)
    for (const char* q : {(const char*)p, (const char*)p + bytes - 1}) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, q) != cudaSuccess) {
            cudaGetLastError();
            return SET_ERR_INVALID;
        }
        if (at.type != cudaMemoryTypeHost || at.devicePointer != (const void*)q) return SET_ERR_INVALID;
    }
    c->add_pinned_range(p, bytes);
    return SET_OK;
}

set_status set_host_unregister(set_ctx* c, const void* p) {
    if (!c || !p) return SET_ERR_INVALID;
    set_status rc = SET_ERR_INVALID;
    c->range_lock.lock();
    for (size_t k = 0; k < c->pinned_ranges.size(); ++k)
        if (c->pinned_ranges[k].lo == (uintptr_t)p) {
            c->pinned_ranges.erase(c->pinned_ranges.begin() + (long)k);
            rc = SET_OK;
            break;
        }
    c->range_lock.unlock();
    return rc;
}

set_status set_get_stats(set_ctx* c, set_stats* out) {
    if (!c || !out) return SET_ERR_INVALID;
    memset(out, 0, sizeof(*out));
    if (c->sched && c->cfg.mode == SET_MODE_SET) {
        CoreStats& st = c->sched->stats();
        out->submitted = st.submitted.load();
        out->completed = st.completed.load();
        out->launched = st.launched.load();
        out->steals = st.steals.load();
        out->submit_stalls = st.submit_stalls.load();
        out->dispatcher_sleeps = st.dispatcher_sleeps.load();
        out->ns_submit = st.ns_submit.load();
        out->ns_launch = st.ns_launch.load();
        out->ns_callback = st.ns_callback.load();
        out->max_inflight_seen = st.max_inflight.load();
    } else {
        out->submitted = c->base_submitted.load();
        out->completed = c->base_completed.load();
        out->launched = c->base_launched.load();
        out->ns_submit = c->base_ns_submit.load();
        out->ns_launch = c->base_ns_launch.load();
        out->max_inflight_seen = (uint64_t)c->b;
    }
    out->full_rebinds = c->full_rebinds.load();
    out->host_rebinds = c->host_rebinds.load();
    out->staged_jobs = c->staged_jobs.load();
    out->kernel_nodes = c->kernel_nodes.load();
    out->signal_nodes = c->signal_nodes.load();
    out->copy_nodes = c->copy_nodes.load();
    out->early_completions = c->early_completions.load();
    out->cuda_streams = (uint64_t)c->Hw;
    out->ns_bind = c->ns_bind.load();
    out->ns_sync = c->ns_sync.load();
    return SET_OK;
}

set_status set_reset_stats(set_ctx* c) {
    if (!c) return SET_ERR_INVALID;
    if (c->sched) {
        CoreStats& st = c->sched->stats();
        st.submitted = 0; st.completed = 0; st.launched = 0; st.steals = 0; st.submit_stalls = 0; st.dispatcher_sleeps = 0;
        st.ns_submit = 0; st.ns_launch = 0; st.ns_callback = 0; st.max_inflight = 0;
    }
    c->base_submitted = 0; c->base_completed = 0; c->base_launched = 0; c->base_ns_submit = 0; c->base_ns_launch = 0;
    c->full_rebinds = 0; c->host_rebinds = 0; c->staged_jobs = 0; c->kernel_nodes = 0; c->signal_nodes = 0; c->copy_nodes = 0; c->early_completions = 0;
    c->stamp_lock.lock();
    c->stamp_recs.clear();
    c->stamp_lock.unlock(); c->ns_bind = 0; c->ns_sync = 0;
    return SET_OK;
}

set_status set_get_gap_stats(set_ctx* c, set_gap_stats* out) {
    if (!c || !out) return SET_ERR_INVALID;
    memset(out, 0, sizeof(*out));
    c->stamp_lock.lock();
    std::vector<set_ctx::StampRec> v = c->stamp_recs;
    c->stamp_lock.unlock();
    if (v.empty()) return SET_OK;
    // jobs of one stream ran one after the other: order them by start time, whatever order their completions were seen in
    std::sort(v.begin(), v.end(), [](const set_ctx::StampRec& a, const set_ctx::StampRec& b) {
        return a.stream != b.stream ? a.stream < b.stream : a.start < b.start;
    });
    std::vector<double> gaps;
    gaps.reserve(v.size());
    double job_sum = 0;
    uint64_t t0 = UINT64_MAX, t1 = 0;
    for (size_t i = 0; i < v.size(); ++i) {
        job_sum += (double)(v[i].end - v[i].start) * 1e-3;
        t0 = std::min(t0, v[i].start);
        t1 = std::max(t1, v[i].end);
        if (i > 0 && v[i - 1].stream == v[i].stream)
            gaps.push_back(v[i].start > v[i - 1].end ? (double)(v[i].start - v[i - 1].end) * 1e-3 : 0.0);
    }
    {  // |union of the jobs' intervals| over all streams: sweep in start order
        std::vector<std::pair<uint64_t, uint64_t>> iv;
        iv.reserve(v.size());
        for (auto& r : v) iv.push_back({r.start, r.end});
        std::sort(iv.begin(), iv.end());
        uint64_t busy = 0, lo = iv[0].first, hi = iv[0].second, idle = 0, nidle = 0;
        for (size_t i = 1; i < iv.size(); ++i) {
            if (iv[i].first > hi) {
                idle += iv[i].first - hi;
                nidle += 1;
                busy += hi - lo;
                lo = iv[i].first;
                hi = iv[i].second;
            } else if (iv[i].second > hi) {
                hi = iv[i].second;
            }
        }
        busy += hi - lo;
        out->busy_union_us = (double)busy * 1e-3;
        out->idle_gaps = (double)nidle;
        out->idle_gap_mean_us = nidle ? (double)idle * 1e-3 / (double)nidle : 0.0;
    }
    out->jobs = v.size();
    out->gaps = gaps.size();
    out->job_mean_us = job_sum / (double)v.size();
    out->span_us = (double)(t1 - t0) * 1e-3;
    out->stream_busy_frac = out->span_us > 0 ? job_sum / (out->span_us * (double)c->H) : 0.0;
    out->idle_frac = out->span_us > 0 ? 1.0 - out->busy_union_us / out->span_us : 0.0;
    if (!gaps.empty()) {
        std::sort(gaps.begin(), gaps.end());
        double sum = 0;
        for (double g : gaps) sum += g;
        auto q = [&](double p) { return gaps[std::min(gaps.size() - 1, (size_t)(p * (double)(gaps.size() - 1) + 0.5))]; };
        out->gap_mean_us = sum / (double)gaps.size();
        out->gap_p50_us = q(0.50);
        out->gap_p99_us = q(0.99);
        out->gap_max_us = gaps.back();
    }
    return SET_OK;
}

const char* set_last_error(set_ctx* c) {
    if (!c) return "";
    std::lock_guard<std::mutex> g(c->errmu);
    return c->errmsg;
}

set_status set_get_geometry(set_ctx* c, int* out_slots, int* out_streams, int* out_execs_per_slot) {
    if (!c) return SET_ERR_INVALID;
    if (out_slots) *out_slots = c->b;
    if (out_streams) *out_streams = c->S;
    if (out_execs_per_slot) *out_execs_per_slot = c->epp;
    return SET_OK;
}

set_status set_time_stage(set_ctx* c, int stage, const uint32_t* dims, int warmup, int iters, float* out_avg_us) {
    if (!c || !out_avg_us || iters < 1 || warmup < 0) return SET_ERR_INVALID;
    if (!c->registered) return SET_ERR_STATE;
    if (stage < 0 || stage >= (int)c->stages.size()) return SET_ERR_INVALID;
    if (int e = c->err.load()) return e;
    c->bind_thread();
    const uint32_t unit[4] = {1, 1, 1, 1};
    if (!dims) dims = unit;
    if (c->check_sizes(dims)) return SET_ERR_SIZE;
    const set_stage_desc& sd = c->stages[stage];
    for (int a = 0; a < sd.num_args; ++a)
        if (sd.args[a].kind == SET_ARG_COND) return SET_ERR_INVALID;  // a loop's control kernel means nothing outside its WHILE node
    ArgPack ap;
    dim3 grid;
    if (int rc = c->build_args(sd, 0, dims, ap, grid)) return rc;
    dim3 block(sd.block[0], sd.block[1] ? sd.block[1] : 1, sd.block[2] ? sd.block[2] : 1);
    cudaStream_t st = c->streams[0];
    if (sd.smem_bytes > 48 * 1024) cudaFuncSetAttribute(sd.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sd.smem_bytes);
    // A chain of `iters` kernel nodes in one graph: no host launch cost between the kernels, so the average is the
    // kernel's device time plus the graph's node-to-node hand-off -- what the kernel costs inside a job graph.
    cudaGraph_t g = nullptr;
    cudaGraphExec_t ge = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t er = cudaGraphCreate(&g, 0);
    cudaGraphNode_t prev = nullptr;
    for (int i = 0; i < iters && er == cudaSuccess; ++i) {
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void*>(sd.func);
        kp.gridDim = grid;
        kp.blockDim = block;
        kp.sharedMemBytes = sd.smem_bytes;
        kp.kernelParams = ap.ptrs;
        cudaGraphNode_t node;
        if (prev && (sd.flags & SET_STAGE_PDL)) {
            // the stage was registered with a programmatic edge in front of it: chain it the same way, so that the figure is
            // what the kernel costs behind another kernel of a job graph (the next launch is resident while this one drains)
            er = cudaGraphAddKernelNode(&node, g, nullptr, 0, &kp);
            cudaGraphEdgeData ed{};
            ed.from_port = cudaGraphKernelNodePortProgrammatic;
            ed.to_port = 0;
            ed.type = cudaGraphDependencyTypeProgrammatic;
            if (er == cudaSuccess) er = cudaGraphAddDependencies_v2(g, &prev, &node, &ed, 1);
        } else {
            er = cudaGraphAddKernelNode(&node, g, prev ? &prev : nullptr, prev ? 1 : 0, &kp);
        }
        prev = node;
    }
    if (er == cudaSuccess) er = cudaGraphInstantiate(&ge, g, 0);
    if (er == cudaSuccess) er = cudaEventCreate(&e0);
    if (er == cudaSuccess) er = cudaEventCreate(&e1);
    for (int i = 0; i < (warmup > 0 ? 1 + warmup / iters : 0) && er == cudaSuccess; ++i) er = cudaGraphLaunch(ge, st);
    if (er == cudaSuccess) er = cudaEventRecord(e0, st);
    if (er == cudaSuccess) er = cudaGraphLaunch(ge, st);
    if (er == cudaSuccess) er = cudaEventRecord(e1, st);
    if (er == cudaSuccess) er = cudaEventSynchronize(e1);
    float ms = 0;
    if (er == cudaSuccess) er = cudaEventElapsedTime(&ms, e0, e1);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (ge) cudaGraphExecDestroy(ge);
    if (g) cudaGraphDestroy(g);
    if (er != cudaSuccess) return c->cuda_fail(er, "set_time_stage", __LINE__);
    *out_avg_us = ms * 1000.0f / (float)iters;
    return SET_OK;
}

}  // extern "C"
