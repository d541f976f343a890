// kernels.h -- declarations of the built-in stage kernels (definitions in this folder).
// Argument lists are documented in include/set.h next to the SET_K_* ids.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

extern "C" {
__global__ void set_k_scan_i32(const int32_t* in, int32_t* out, uint32_t n);
__global__ void set_k_hist_mod64(const int32_t* in, uint32_t* hist, uint32_t n);
__global__ void set_k_affine_f32(const float* x, float* y, uint32_t n);
__global__ void set_k_add_bias_f32(float* y, const float* bias, uint32_t n);
__global__ void set_k_relu_f32(float* y, uint32_t n);
__global__ void set_k_square_f32(float* y, uint32_t n);
__global__ void set_k_block_sum_f32(const float* y, float* out, uint32_t n);
__global__ void set_k_jacobi5_f32(const float* u, float* v, uint32_t h, uint32_t w, uint32_t flip);
__global__ void set_k_rgb2gray_u8(const uint8_t* rgb, uint8_t* gray, uint32_t w, uint32_t h);
__global__ void set_k_blur3x3_u8(const uint8_t* g, uint8_t* out, uint32_t w, uint32_t h);
__global__ void set_k_hist256_u8(const uint8_t* p, uint32_t* hist, uint32_t w, uint32_t h);
__global__ void set_k_spin(uint32_t* scratch, uint32_t ns);
__global__ void set_k_signal(uint32_t* flag, unsigned long long* stamp, uint32_t fence);
__global__ void set_k_stamp(unsigned long long* stamp);
__global__ void set_k_copy(const void* src, void* dst, uint32_t bytes, void** fwd_slot, void* fwd_value);
__global__ void set_k_copy_out(const void* src, void* const* dst_slot, unsigned long long dst_off, uint32_t bytes, uint32_t* flag,
                               unsigned long long* stamp, uint32_t fence);
__global__ void set_k_sobel3x3_u8(const uint8_t* n, uint8_t* e, uint32_t w, uint32_t h);
__global__ void set_k_mean3x3_u8(const uint8_t* e, uint8_t* m, uint32_t w, uint32_t h);
__global__ void set_k_threshold_u8(const uint8_t* m, uint8_t* t, uint32_t w, uint32_t h, uint32_t thresh);
__global__ void set_k_blend_u8(const uint8_t* t, const uint8_t* n, uint8_t* out, uint32_t w, uint32_t h);
__global__ void set_k_sssp_init(const int32_t* img, int32_t* out, uint32_t* scratch, uint32_t max_v);
__global__ void set_k_sssp_relax(const int32_t* img, int32_t* out, uint32_t* scratch, uint32_t max_v, uint32_t sub);
__global__ void set_k_sssp_solo(const int32_t* img, int32_t* out, uint32_t* scratch, uint32_t max_v);
__global__ void set_k_sssp_control(const int32_t* img, int32_t* out, uint32_t* scratch, uint32_t max_v, uint32_t unroll, cudaGraphConditionalHandle loop);
}

// Programmatic dependent launch (SET_STAGE_PDL edges of the job graph): let the next kernel node be scheduled now,
// then wait until every kernel this one depends on has finished and its writes are visible.  Both instructions do
// nothing in a kernel that was launched over an ordinary edge, so every built-in kernel starts with this.
#ifdef __CUDACC__
// The pointers a kernel READS what earlier nodes wrote through are passed in and come back "laundered" through an empty asm
// placed after the wait.  Without that the compiler may issue a load through a `const T* __restrict__` parameter BEFORE the
// wait: it treats such loads as invariant (ld.global.nc), and invariant loads are not held back by a "memory" clobber.
// Seen in SASS: K21's load of V sat in front of ACQBULK and read what the slot's previous job had left (round 2).
template <typename T>  // T: a pointer type, __restrict__ and all
__device__ __forceinline__ void set_pdl_launder(T& p) {
    static_assert(sizeof(T) == 8, "pointers only");
    asm volatile("" : "+l"(p));
}
template <typename... P>
__device__ __forceinline__ void set_pdl_sync(P&... inputs) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    (set_pdl_launder(inputs), ...);
}
// The same without the early trigger, for kernels whose grid covers a frame (K10-K12, K17-K20): with launch_dependents at the
// top, the NEXT kernel's blocks become resident at once and sit on SM slots and registers, spinning in their wait, while
// blocks of THIS kernel have yet to start -- config 6 device-resident ran at 119 K jobs/s with the trigger and 145 K without
// (profiles/r2_probes.md section 8).  Without a trigger the dependent launches when this grid completes, as over a plain edge.
template <typename... P>
__device__ __forceinline__ void set_pdl_wait(P&... inputs) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    (set_pdl_launder(inputs), ...);
}
#endif

// Tile shapes the host-side grid rules in set_builtin.cu must agree with.
constexpr int kJacobiRows = 16;        // rows per block
constexpr int kJacobiCols = 1024;      // columns per block (256 threads x float4)
constexpr unsigned kJacobiUnroll = 4;  // rows whose loads are in flight together
constexpr int kGrayPixPerBlock = 256 * 16;
constexpr int kBlurTileW = 512, kBlurTileH = 16;  // 32 lanes x 16 pixels, 4 warps x 4 rows (a 1280 x 720 frame: 135 blocks)
constexpr int kHistPixPerBlock = 256 * 16;  // one 128-bit load per thread; a 1280 x 720 frame: 225 blocks
constexpr int kCopyBytesPerBlock = 256 * 16 * 2;  // set_k_copy: 256 threads x two 128-bit words
constexpr int kBytePixPerBlock = 256 * 16;                // K19/K20: one 128-bit word per thread
constexpr int kSsspSoloThreads = 1024;                    // K25: one block runs the job
constexpr unsigned kSsspSoloMaxV = 40000;                 // K25: 5 bytes of shared memory per vertex (200 KB of the SM's 227)
extern "C" uint32_t set_sssp_solo_smem_bytes(uint32_t max_v);
constexpr unsigned kSsspLanes = 8;                        // K22: threads per vertex (blocks of 256 threads: 32 vertices each)
