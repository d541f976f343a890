// set_noalloc.cu -- set_sssp_noalloc(): one SSSP job (config 5's computation, readings S5-1..S5-4 of DESIGN.md)
// through an entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid allocation).  The contract is in include/set.h next to the declaration.
//
// The kernel is K25 (set_k_sssp_solo, kernels/paper_kernels.cu), a variant of K22: the same 8-lanes-per-vertex in-place
// relaxation with atomicMin, but ONE block of 1024 threads runs the whole job -- initialisation, every round, the round
// count -- with __syncthreads() between rounds, so it needs neither the WHILE node nor a set_ctx with its device buffers.
// Distances and frontier flags sit in shared memory; its scratch in global memory (the work list of frontier vertices) is
// g_noalloc_scratch below.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "kernels/kernels.h"
#include "set.h"

namespace {

// The scratch of every set_sssp_noalloc call on a device: the work list, uint32[SET_NOALLOC_MAX_VERTICES] = 64 KiB.
// Every GPU that loads libset.so holds it until the process exits.  In HOST code this name is a host-side stand-in, not a
// device address: the launch below passes what cudaGetSymbolAddress returned for the current device.
static __device__ __align__(256) uint32_t g_noalloc_scratch[SET_NOALLOC_MAX_VERTICES];

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
        // the kernel keeps 5 bytes per vertex in dynamic shared memory: allow the maximum once (an attribute, not an allocation)
        e = cudaFuncSetAttribute((const void*)set_k_sssp_solo, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)set_sssp_solo_smem_bytes(SET_NOALLOC_MAX_VERTICES));
        if (e != cudaSuccess) return fail(SET_ERR_CUDA, "cudaFuncSetAttribute(set_k_sssp_solo)", e);
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
    // work list: scratch[0 .. V), V <= SET_NOALLOC_MAX_VERTICES
    void* args[4] = {(void*)&dev_image, (void*)&dev_out, (void*)&scratch, (void*)&num_vertices};
    cudaError_t e = cudaLaunchKernel((const void*)set_k_sssp_solo, dim3(1), dim3(kSsspSoloThreads), args, set_sssp_solo_smem_bytes(num_vertices),
                                     (cudaStream_t)stream);
    if (e != cudaSuccess) return fail(SET_ERR_CUDA, "kernel launch", e);
    return SET_OK;
}

extern "C" const char* set_noalloc_last_error(void) { return t_err; }
