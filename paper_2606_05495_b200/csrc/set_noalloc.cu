// set_noalloc.cu -- set_sssp_noalloc(): one SSSP job (config 5's computation, readings S5-1..S5-4 of DESIGN.md)
// through an entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid allocation).  The contract is in include/set.h next to the declaration.
//
// The kernel is a variant of K22 (set_k_sssp_relax, kernels/paper_kernels.cu): the same 8-lanes-per-vertex in-place
// relaxation with atomicMin and the same double-buffered frontier flags, but ONE block of 1024 threads runs the whole job --
// initialisation, every round, the round count -- with __syncthreads() between rounds, so it needs neither the WHILE node
// nor a set_ctx with its device buffers.  Its scratch (the frontier flags) lives in g_noalloc_scratch below.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "kernels/kernels.h"
#include "set.h"

namespace {

// The scratch of every set_sssp_noalloc call on a device: frontier flags [2][SET_NOALLOC_MAX_VERTICES] uint32 = 128 KiB.
// Every GPU that loads libset.so holds it until the process exits.  In HOST code this name is a host-side stand-in, not a
// device address: the launch below passes what cudaGetSymbolAddress returned for the current device.
static __device__ __align__(256) uint32_t g_noalloc_scratch[2 * SET_NOALLOC_MAX_VERTICES];

constexpr int kSoloThreads = 1024;
constexpr int32_t kInf = 0x7fffffff;

// img = int32 [V, E, src, 0][row_ptr V+1][col E][w E]; out = int32 [dist V][rounds, 0, 0, 0] (the layouts of config 5).
// Everything the job reads from the scratch it writes first (flags 0 .. V-1 of both halves): the last call's contents
// never matter.
__global__ void __launch_bounds__(kSoloThreads) set_k_sssp_solo(const int32_t* __restrict__ img, int32_t* __restrict__ out,
                                                                uint32_t* __restrict__ scratch, uint32_t max_v) {
    __shared__ uint32_t s_changed;
    const uint32_t V = min((uint32_t)img[0], max_v), src = (uint32_t)img[2];
    const int32_t* row_ptr = img + 4;
    const int32_t* col = row_ptr + V + 1;
    const int32_t* wgt = col + img[1];
    uint32_t* flags[2] = {scratch, scratch + SET_NOALLOC_MAX_VERTICES};
    for (uint32_t v = threadIdx.x; v < V; v += kSoloThreads) {
        out[v] = v == src ? 0 : kInf;
        flags[0][v] = v == src ? 1u : 0u;
        flags[1][v] = 0u;
    }
    constexpr uint32_t kPerWarp = 32 / kSsspLanes, kPerSweep = kSoloThreads / kSsspLanes;
    const uint32_t g = threadIdx.x % kSsspLanes, in_warp = (threadIdx.x % 32) / kSsspLanes, warp = threadIdx.x / 32;
    uint32_t rounds = 0;
    // a round with a frontier: the first always has one ({src}); the next has one iff this one lowered a distance
    for (bool go = V > 0 && src < V; go;) {
        if (threadIdx.x == 0) s_changed = 0u;
        __syncthreads();  // the flags and distances of the previous round (or the initialisation) are visible to the block
        uint32_t* fin = flags[rounds & 1u];
        uint32_t* fout = flags[(rounds + 1u) & 1u];
        bool any = false;
        for (uint32_t base = warp * kPerWarp; base < V; base += kPerSweep) {  // uniform over the warp
            const uint32_t u = base + in_warp;
            const uint32_t f = u < V ? fin[u] : 0u;
            __syncwarp();
            if (!f) continue;
            if (g == 0) fin[u] = 0u;
            const int32_t du = *reinterpret_cast<volatile int32_t*>(out + u);  // finite: u entered the frontier by getting a distance
            const int32_t e1 = __ldg(row_ptr + u + 1);
            for (int32_t e = __ldg(row_ptr + u) + (int32_t)g; e < e1; e += (int32_t)kSsspLanes) {
                const int32_t v = __ldg(col + e), nd = du + __ldg(wgt + e);
                if (nd < atomicMin(out + v, nd)) {
                    fout[v] = 1u;
                    any = true;
                }
            }
        }
        if (any) s_changed = 1u;
        rounds += 1u;
        __syncthreads();
        go = s_changed != 0u && rounds <= V;  // at most V rounds: Bellman-Ford's bound with non-negative weights
        __syncthreads();                      // everyone has read s_changed before thread 0 clears it
    }
    if (threadIdx.x < 4) out[V + threadIdx.x] = threadIdx.x == 0 ? (int32_t)rounds : 0;
}

// ---- host side --------------------------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
std::mutex g_mu;
uint32_t* g_scratch_dev[kMaxDevices];  // per device: the address of g_noalloc_scratch ON that device (set-up, once)
thread_local char t_err[256];

set_status fail(set_status st, const char* what, cudaError_t e) {
    if (e != cudaSuccess)
        snprintf(t_err, sizeof t_err, "set_sssp_noalloc: %s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    else
        snprintf(t_err, sizeof t_err, "set_sssp_noalloc: %s", what);
    return st;
}

// Set-up, once per device, with that device current: the device address of the scratch array.
set_status scratch_for_current_device(uint32_t** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(SET_ERR_CUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= kMaxDevices) return fail(SET_ERR_INVALID, "device ordinal out of range", cudaSuccess);
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_dev[dev]) {
        uint32_t* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return fail(SET_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch)", e);
        g_scratch_dev[dev] = p;
    }
    *out = g_scratch_dev[dev];
    return SET_OK;
}

}  // namespace

extern "C" set_status set_sssp_noalloc(const void* dev_image, void* dev_out, uint32_t num_vertices, void* stream) {
    t_err[0] = 0;
    if (num_vertices > SET_NOALLOC_MAX_VERTICES) {
        snprintf(t_err, sizeof t_err, "set_sssp_noalloc: %u vertices exceed the static scratch's maximum of %u (SET_NOALLOC_MAX_VERTICES)",
                 num_vertices, (unsigned)SET_NOALLOC_MAX_VERTICES);
        return SET_ERR_SIZE;
    }
    uint32_t* scratch = nullptr;
    if (set_status st = scratch_for_current_device(&scratch)) return st;
    if (num_vertices == 0) return SET_OK;  // set-up only
    if (!dev_image || !dev_out) return fail(SET_ERR_INVALID, "dev_image and dev_out must be device pointers", cudaSuccess);
    set_k_sssp_solo<<<1, kSoloThreads, 0, (cudaStream_t)stream>>>((const int32_t*)dev_image, (int32_t*)dev_out, scratch, num_vertices);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SET_ERR_CUDA, "kernel launch", e);
    return SET_OK;
}

extern "C" const char* set_noalloc_last_error(void) { return t_err; }
