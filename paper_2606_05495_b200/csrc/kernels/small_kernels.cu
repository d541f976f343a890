// small_kernels.cu -- stage kernels K1-K7 and K13 (configs 0 and 1; BASELINE.json:configs[0..1]).
// Hand-written CUDA for sm_100a.  These are latency-class kernels: one job's data (16-128 KB) sits in L2
// right after its H2D copy, so the design goal is the shortest possible critical path -- one block for the
// scan / histogram / reduction (no inter-block synchronisation), 128-bit accesses, warp-shuffle scans and
// reductions, and no FMA contraction anywhere (reading C1-1).
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.h"

namespace {

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

// 128-bit accesses need 16-byte aligned operands; the device image mirrors the host image, so an operand that
// starts at byte 4n of a buffer (the bias vector of config 1) is only aligned when n is a multiple of 4.
__device__ __forceinline__ bool aligned16(const void* a, const void* b = nullptr) {
    return (((uintptr_t)a | (uintptr_t)b) & 15u) == 0;
}

}  // namespace

// K1: inclusive prefix sum of n int32, one block of 1024 threads.
// Per 4096-element chunk: 128-bit load -> 4-element serial scan in registers -> warp shuffle scan of the
// thread totals -> 32 warp totals scanned by warp 0 in shared memory -> carry from the previous chunk.
extern "C" __global__ void __launch_bounds__(1024) set_k_scan_i32(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                                  uint32_t n) {
    set_pdl_sync(in);
    __shared__ int warp_tot[32];
    __shared__ int chunk_tot;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int carry = 0;
    for (uint32_t base = 0; base < n; base += 4096) {
        uint32_t i = base + 4u * tid;
        int4 v = make_int4(0, 0, 0, 0);
        if (i + 3 < n) {
            v = *reinterpret_cast<const int4*>(in + i);
        } else {
            if (i < n) v.x = in[i];
            if (i + 1 < n) v.y = in[i + 1];
            if (i + 2 < n) v.z = in[i + 2];
        }
        v.y += v.x;
        v.z += v.y;
        v.w += v.z;
        int incl = warp_incl_scan(v.w, lane);
        if (lane == 31) warp_tot[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int t = warp_tot[lane];
            int s = warp_incl_scan(t, lane);
            warp_tot[lane] = s - t;  // exclusive prefix of the warp totals
            if (lane == 31) chunk_tot = s;
        }
        __syncthreads();
        int off = carry + warp_tot[wid] + (incl - v.w);
        v.x += off;
        v.y += off;
        v.z += off;
        v.w += off;
        if (i + 3 < n) {
            *reinterpret_cast<int4*>(out + i) = v;
        } else {
            if (i < n) out[i] = v.x;
            if (i + 1 < n) out[i + 1] = v.y;
            if (i + 2 < n) out[i + 2] = v.z;
        }
        carry += chunk_tot;
        __syncthreads();  // warp_tot / chunk_tot are rewritten by the next chunk
    }
}

// K2: hist[b] = #{i : v[i] mod 64 == b}, v >= 0 (reading C0-3), one block of 256 threads.
// Every thread's first four 128-bit loads are issued before the shared histograms are cleared.  One private 64-bin
// histogram per warp in shared memory (8 x 64 counters) keeps atomic contention inside a warp; the 8 copies are then
// summed, one bin per thread.
extern "C" __global__ void __launch_bounds__(256) set_k_hist_mod64(const int32_t* __restrict__ in, uint32_t* __restrict__ hist,
                                                                   uint32_t n) {
    set_pdl_sync(in);
    __shared__ uint32_t h[8][64 + 1];
    const int tid = threadIdx.x, wid = tid >> 5;
    const uint32_t n4 = n / 4;
    int4 first[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t i = tid + 256u * k;
        first[k] = i < n4 ? reinterpret_cast<const int4*>(in)[i] : make_int4(0, 0, 0, 0);
    }
    for (int k = tid; k < 8 * 65; k += 256) (&h[0][0])[k] = 0;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (tid + 256u * k < n4) {
            atomicAdd(&h[wid][first[k].x & 63], 1u);
            atomicAdd(&h[wid][first[k].y & 63], 1u);
            atomicAdd(&h[wid][first[k].z & 63], 1u);
            atomicAdd(&h[wid][first[k].w & 63], 1u);
        }
    }
    for (uint32_t i = tid + 1024u; i < n4; i += 256) {
        int4 v = reinterpret_cast<const int4*>(in)[i];
        atomicAdd(&h[wid][v.x & 63], 1u);
        atomicAdd(&h[wid][v.y & 63], 1u);
        atomicAdd(&h[wid][v.z & 63], 1u);
        atomicAdd(&h[wid][v.w & 63], 1u);
    }
    for (uint32_t i = n4 * 4 + tid; i < n; i += 256) atomicAdd(&h[wid][in[i] & 63], 1u);
    __syncthreads();
    if (tid < 64) {
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += h[w][tid];
        hist[tid] = s;
    }
}

// K3..K6: one fp32 operation per element per kernel (reading C1-5: the chain stays unfused).  256 threads x 4
// elements per block; __fmul_rn/__fadd_rn are never contracted into an FMA (reading C1-1).
extern "C" __global__ void __launch_bounds__(256) set_k_affine_f32(const float* __restrict__ x, float* __restrict__ y, uint32_t n) {
    set_pdl_sync(x);
    uint32_t i = 4u * (blockIdx.x * 256u + threadIdx.x);
    if (i + 3 < n && aligned16(x, y)) {
        float4 v = *reinterpret_cast<const float4*>(x + i);
        v.x = __fadd_rn(__fmul_rn(2.5f, v.x), 0.1f);
        v.y = __fadd_rn(__fmul_rn(2.5f, v.y), 0.1f);
        v.z = __fadd_rn(__fmul_rn(2.5f, v.z), 0.1f);
        v.w = __fadd_rn(__fmul_rn(2.5f, v.w), 0.1f);
        *reinterpret_cast<float4*>(y + i) = v;
    } else {
        for (uint32_t e = i + 4; i < n && i < e; ++i) y[i] = __fadd_rn(__fmul_rn(2.5f, x[i]), 0.1f);
    }
}

extern "C" __global__ void __launch_bounds__(256) set_k_add_bias_f32(float* __restrict__ y, const float* __restrict__ bias, uint32_t n) {
    set_pdl_sync(bias);
    uint32_t i = 4u * (blockIdx.x * 256u + threadIdx.x);
    if (i + 3 < n && aligned16(y, bias)) {
        float4 v = *reinterpret_cast<float4*>(y + i);
        float4 b = *reinterpret_cast<const float4*>(bias + i);
        v.x = __fadd_rn(v.x, b.x);
        v.y = __fadd_rn(v.y, b.y);
        v.z = __fadd_rn(v.z, b.z);
        v.w = __fadd_rn(v.w, b.w);
        *reinterpret_cast<float4*>(y + i) = v;
    } else {
        for (uint32_t e = i + 4; i < n && i < e; ++i) y[i] = __fadd_rn(y[i], bias[i]);
    }
}

extern "C" __global__ void __launch_bounds__(256) set_k_relu_f32(float* __restrict__ y, uint32_t n) {
    set_pdl_sync();
    uint32_t i = 4u * (blockIdx.x * 256u + threadIdx.x);
    if (i + 3 < n && aligned16(y)) {
        float4 v = *reinterpret_cast<float4*>(y + i);
        v.x = v.x > 0.0f ? v.x : 0.0f;
        v.y = v.y > 0.0f ? v.y : 0.0f;
        v.z = v.z > 0.0f ? v.z : 0.0f;
        v.w = v.w > 0.0f ? v.w : 0.0f;
        *reinterpret_cast<float4*>(y + i) = v;
    } else {
        for (uint32_t e = i + 4; i < n && i < e; ++i) y[i] = y[i] > 0.0f ? y[i] : 0.0f;
    }
}

extern "C" __global__ void __launch_bounds__(256) set_k_square_f32(float* __restrict__ y, uint32_t n) {
    set_pdl_sync();
    uint32_t i = 4u * (blockIdx.x * 256u + threadIdx.x);
    if (i + 3 < n && aligned16(y)) {
        float4 v = *reinterpret_cast<float4*>(y + i);
        v.x = __fmul_rn(v.x, v.x);
        v.y = __fmul_rn(v.y, v.y);
        v.z = __fmul_rn(v.z, v.z);
        v.w = __fmul_rn(v.w, v.w);
        *reinterpret_cast<float4*>(y + i) = v;
    } else {
        for (uint32_t e = i + 4; i < n && i < e; ++i) y[i] = __fmul_rn(y[i], y[i]);
    }
}

// K7: out[0] = sum_i y[i], one block of 1024 threads, fixed-shape tree (deterministic run to run):
// per thread: pairwise sum inside each float4, sequential over the thread's strided float4s;
// then xor-shuffle tree inside the warp, then the 32 warp sums by warp 0 (reading C1-2: any fixed tree within
// the 1e-6 tolerance of the double-accumulated oracle; measured ~1e-8).
extern "C" __global__ void __launch_bounds__(1024) set_k_block_sum_f32(const float* __restrict__ y, float* __restrict__ out,
                                                                       uint32_t n) {
    set_pdl_sync(y);
    __shared__ float wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    float acc = 0.0f;
    const uint32_t n4 = n / 4;
    // four strided float4 loads in flight per thread; the adds keep the order i = tid, tid + 1024, ... so the tree (and
    // the result, bit for bit) is the one a plain loop gives
    for (uint32_t i = tid; i < n4; i += 4096) {
        float4 v[4];
#pragma unroll
        for (uint32_t k = 0; k < 4; ++k)
            v[k] = (i + k * 1024u < n4) ? reinterpret_cast<const float4*>(y)[i + k * 1024u] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (uint32_t k = 0; k < 4; ++k)
            if (i + k * 1024u < n4) acc = __fadd_rn(acc, __fadd_rn(__fadd_rn(v[k].x, v[k].y), __fadd_rn(v[k].z, v[k].w)));
    }
    for (uint32_t i = n4 * 4 + tid; i < n; i += 1024) acc = __fadd_rn(acc, y[i]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc = __fadd_rn(acc, __shfl_xor_sync(0xffffffffu, acc, d));
    if (lane == 0) wsum[wid] = acc;
    __syncthreads();
    if (wid == 0) {
        float s = wsum[lane];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s = __fadd_rn(s, __shfl_xor_sync(0xffffffffu, s, d));
        if (lane == 0) out[0] = s;
    }
}

// K13: debug delay stage (SURVEY.md §5 fault injection): one thread busy-waits `ns` nanoseconds so that job
// completions reorder and slots stay occupied; scratch[0] receives the waited time.
extern "C" __global__ void set_k_spin(uint32_t* scratch, uint32_t ns) {
    set_pdl_sync();
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    } while (t - t0 < (unsigned long long)ns);
    if (scratch) scratch[0] = (uint32_t)(t - t0);
}

// K14: completion signal of SET_CB_FLAG_POLL.  Last node of the job graph: it depends on every D2H copy node (memcpy
// node or SET_K_COPY kernel node).  One thread stores 1 to the slot's word in mapped pinned host memory, which the
// dispatcher thread is watching.
//   fence != 0 (SET_FENCE_SYSTEM, the default): fence.acq_rel.sys, then the store.  The job's output was written by an
//     EARLIER grid; its completion (or griddepcontrol.wait) makes those writes visible to this thread, and the system-
//     scope fence is cumulative, so they are ordered before the word for an observer on the host: a release pattern
//     the PTX memory model guarantees.  Costs about 2.5 us of the signal node's time on B200, which
//     set_config.streams_per_lane takes off the job-to-job critical path (the next job of the lane runs on another
//     CUDA stream and does not wait for this node).
//   fence == 0 (SET_FENCE_NONE): plain volatile store, relying on grid completion alone to have pushed the output out.
//     Two unfenced stores of ONE thread were seen to reach host memory out of order on this machine (the stamp and the
//     word below), and with several CUDA streams per lane the library's own hook caught the word overtaking a job's
//     output about once in 30,000 jobs (profiles/r2_signal_soak.md): unsafe, kept as a measurement arm only.
extern "C" __global__ void set_k_signal(uint32_t* flag, unsigned long long* stamp, uint32_t fence) {
    set_pdl_sync();
    if (stamp) {  // set_config.timestamps: when the job ended on the device
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        *reinterpret_cast<volatile unsigned long long*>(stamp) = t;
    }
    if (fence) asm volatile("fence.acq_rel.sys;" ::: "memory");
    *reinterpret_cast<volatile uint32_t*>(flag) = 1u;
}

// K16: timestamp node of set_config.timestamps.  As a root of the job graph it runs when the graph starts (beside the
// first copy); as the last node (modes without a signal node) when it ends.  One thread, one 8-byte store to mapped
// pinned host memory.
extern "C" __global__ void set_k_stamp(unsigned long long* stamp) {
    set_pdl_sync();
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    *reinterpret_cast<volatile unsigned long long*>(stamp) = t;
}

// K15: copy node executed by the SMs.  A job of configs 0-1 moves 16-128 KB per direction;
// a copy-engine memcpy node costs ~10 us of engine hand-off on each side of it, far more than the wire time, so
// copies up to set_config.sm_copy_max_bytes are kernel nodes instead: the SMs read pinned host memory directly
// over the link (H2D) or store into it (D2H).  Each thread moves two 128-bit words, both loads issued before the
// first store so that 8 KB per block are in flight; unaligned operands or sizes fall back to a byte loop.
namespace {
__device__ __forceinline__ void copy_bytes(const void* __restrict__ src, void* __restrict__ dst, uint32_t bytes) {
    const uint32_t tid = threadIdx.x;
    const bool vec = aligned16(src, dst);
    for (uint32_t base = blockIdx.x * (uint32_t)kCopyBytesPerBlock; base < bytes; base += gridDim.x * (uint32_t)kCopyBytesPerBlock) {
        if (vec) {
            const uint32_t o0 = base + tid * 16u, o1 = o0 + 256u * 16u;
            uint4 a = make_uint4(0, 0, 0, 0), b = a;
            const bool f0 = o0 + 16u <= bytes, f1 = o1 + 16u <= bytes;
            if (f0) a = *reinterpret_cast<const uint4*>(static_cast<const char*>(src) + o0);
            if (f1) b = *reinterpret_cast<const uint4*>(static_cast<const char*>(src) + o1);
            if (f0) *reinterpret_cast<uint4*>(static_cast<char*>(dst) + o0) = a;
            if (f1) *reinterpret_cast<uint4*>(static_cast<char*>(dst) + o1) = b;
            // ragged tail (< 16 bytes), by the thread whose word would have covered it
            if (!f0 && o0 < bytes)
                for (uint32_t k = o0; k < bytes; ++k) static_cast<char*>(dst)[k] = static_cast<const char*>(src)[k];
            if (!f1 && o1 < bytes)
                for (uint32_t k = o1; k < bytes; ++k) static_cast<char*>(dst)[k] = static_cast<const char*>(src)[k];
        } else {
            const uint32_t end = min(base + (uint32_t)kCopyBytesPerBlock, bytes);
            for (uint32_t k = base + tid; k < end; k += 256u) static_cast<char*>(dst)[k] = static_cast<const char*>(src)[k];
        }
    }
}
}  // namespace

// fwd_slot != NULL: the copy-in node also carries the job's OUTPUT address into the slot's device word, from which the
// copy-out node (K24) takes its destination -- so that a job costs ONE graph-node update instead of two (the update and the
// launch go through the same driver lock, about 0.5 us per node: DESIGN.md 5d).
extern "C" __global__ void __launch_bounds__(256) set_k_copy(const void* __restrict__ src, void* __restrict__ dst, uint32_t bytes, void** fwd_slot,
                                                             void* fwd_value) {
    set_pdl_sync(src);
    if (fwd_slot && blockIdx.x == 0 && threadIdx.x == 0) *fwd_slot = fwd_value;
    copy_bytes(src, dst, bytes);
}

// K24: copy-out whose destination is *dst_slot + dst_off: the address the job's copy-in node left in the slot's device word.
// Every kernel between the two is ordered behind its predecessor (plain edge or griddepcontrol.wait), so the word is visible.
// flag != NULL: this node is also the job's completion signal (K14 folded in: one node less per job -- the GPU's front end
// works through about three million graph nodes a second, which is what bounds the short-job configs).  Every
// block, after its part of the copy, takes a ticket with a gpu-scope release; the block that draws the last ticket has thereby
// acquired every other block's stores, fences them out at system scope (unless fence == 0) and stores the slot's word.
extern "C" __global__ void __launch_bounds__(256) set_k_copy_out(const void* __restrict__ src, void* const* __restrict__ dst_slot, unsigned long long dst_off,
                                                                 uint32_t bytes, uint32_t* flag, unsigned long long* stamp, uint32_t fence) {
    set_pdl_sync(src, dst_slot);
    char* dst = static_cast<char*>(*reinterpret_cast<void* const volatile*>(dst_slot)) + dst_off;
    copy_bytes(src, dst, bytes);
    if (flag) {
        __syncthreads();  // the block's stores are ordered before thread 0's release below (cta-scope barrier, then cumulativity)
        if (threadIdx.x == 0) {
            uint32_t* ticket = reinterpret_cast<uint32_t*>(const_cast<void**>(dst_slot) + 1);  // the word behind the forwarded address
            uint32_t drawn;
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(drawn) : "l"(ticket) : "memory");
            if (drawn == gridDim.x - 1u) {
                *ticket = 0u;  // for the slot's next job (ordered before its launch by the completion itself)
                if (stamp) {
                    unsigned long long t;
                    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
                    *reinterpret_cast<volatile unsigned long long*>(stamp) = t;
                }
                if (fence) asm volatile("fence.acq_rel.sys;" ::: "memory");
                *reinterpret_cast<volatile uint32_t*>(flag) = 1u;
            }
        }
    }
}
