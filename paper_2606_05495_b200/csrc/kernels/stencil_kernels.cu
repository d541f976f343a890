// stencil_kernels.cu -- K8 (config 2: 5-point Jacobi) and K10-K12 (config 4: gray -> blur -> hist256).
// Hand-written CUDA for sm_100a.  These are the bandwidth-class stages: 128-bit (or 32-bit for the byte images)
// coalesced global accesses, vertical register rolling so that every input row is read once per block, and
// warp shuffles for the horizontal neighbours.  No tensor cores: none of this is a dense contraction.
#include "kernels.h"

// ------------------------------------------------------------------------------------------------------------
// K8: one Jacobi sweep  v[i][j] = 0.2f * ((((c + w) + e) + n) + s), zero halo (readings C2-1..C2-3).
// Block = 256 threads = 1024 columns x kJacobiRows rows.  Each thread owns one float4 column group and walks
// down the rows keeping (up, mid, down) in registers: each element is loaded once per block plus the two halo
// rows; left/right neighbours come from the adjacent lane by shuffle, from global memory only at warp edges.
// The add order is exactly the oracle's, and there is no multiply-add pair, so results are bit-identical.
// ------------------------------------------------------------------------------------------------------------
namespace {
__device__ __forceinline__ float jac(float c, float w, float e, float n, float s) {
    return __fmul_rn(0.2f, __fadd_rn(__fadd_rn(__fadd_rn(__fadd_rn(c, w), e), n), s));
}
__device__ __forceinline__ float at0(const float* __restrict__ u, uint32_t h, uint32_t w, int64_t i, int64_t j) {
    return (i < 0 || j < 0 || i >= (int64_t)h || j >= (int64_t)w) ? 0.0f : __ldg(u + i * (int64_t)w + j);
}
}  // namespace

extern "C" __global__ void __launch_bounds__(256) set_k_jacobi5_f32(const float* __restrict__ u, float* __restrict__ v, uint32_t h,
                                                                    uint32_t w, uint32_t flip) {
    set_pdl_sync(u);
    // flip = 1: walk the row blocks bottom-up.  Consecutive sweeps alternate direction, so a sweep starts on the rows
    // the previous sweep wrote last -- the part of the ping-pong pair (2 x 64 MiB) that is still in the 126 MB L2.
    const uint32_t by = flip ? gridDim.y - 1u - blockIdx.y : blockIdx.y;
    const uint32_t r0 = by * kJacobiRows;
    const uint32_t r1 = min(r0 + (uint32_t)kJacobiRows, h);
    const uint32_t c4 = (blockIdx.x * 256u + threadIdx.x) * 4u;
    if ((w & 3u) == 0) {
        const int lane = threadIdx.x & 31;
        const bool active = c4 < w;
        const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
        auto row = [&](uint32_t r) -> float4 {
            return active ? __ldg(reinterpret_cast<const float4*>(u + (size_t)r * w + c4)) : zero;
        };
        // the warp's edge lanes need one scalar from the neighbouring column group (0 outside the grid = the halo)
        auto edge = [&](uint32_t r) -> float {
            if (lane == 0) return (active && c4 > 0) ? __ldg(u + (size_t)r * w + c4 - 1) : 0.0f;
            if (lane == 31) return (active && c4 + 4 < w) ? __ldg(u + (size_t)r * w + c4 + 4) : 0.0f;
            return 0.0f;
        };
        float4 up = (r0 > 0) ? row(r0 - 1) : zero;
        float4 mid = row(r0);
        float e_mid = edge(r0);
        // kJacobiUnroll rows per round: all of the round's loads are issued before the first add, so every thread keeps
        // kJacobiUnroll 128-bit loads in flight (one load per thread does not cover the HBM latency at 7 blocks per SM)
        for (uint32_t r = r0; r < r1; r += kJacobiUnroll) {
            float4 dn[kJacobiUnroll];
            float e_dn[kJacobiUnroll];
#pragma unroll
            for (uint32_t k = 0; k < kJacobiUnroll; ++k) {
                const uint32_t rr = r + 1 + k;  // row below output row r + k; row r1 is the block's lower halo
                const bool need = rr < h && rr <= r1;
                dn[k] = need ? row(rr) : zero;
                e_dn[k] = (need && rr < r1) ? edge(rr) : 0.0f;
            }
#pragma unroll
            for (uint32_t k = 0; k < kJacobiUnroll; ++k) {
                if (r + k < r1) {
                    float left = __shfl_up_sync(0xffffffffu, mid.w, 1);
                    float right = __shfl_down_sync(0xffffffffu, mid.x, 1);  // an inactive neighbour holds 0 = the halo
                    if (lane == 0) left = e_mid;
                    if (lane == 31) right = e_mid;
                    if (active) {
                        float4 o;
                        o.x = jac(mid.x, left, mid.y, up.x, dn[k].x);
                        o.y = jac(mid.y, mid.x, mid.z, up.y, dn[k].y);
                        o.z = jac(mid.z, mid.y, mid.w, up.z, dn[k].z);
                        o.w = jac(mid.w, mid.z, right, up.w, dn[k].w);
                        *reinterpret_cast<float4*>(v + (size_t)(r + k) * w + c4) = o;
                    }
                    up = mid;
                    mid = dn[k];
                    e_mid = e_dn[k];
                }
            }
        }
    } else {  // ragged width: rows are not 16-byte aligned, one element at a time
        for (uint32_t r = r0; r < r1; ++r)
            for (uint32_t k = 0; k < 4; ++k) {
                uint32_t c = c4 + k;
                if (c < w)
                    v[(size_t)r * w + c] = jac(at0(u, h, w, r, c), at0(u, h, w, r, (int64_t)c - 1), at0(u, h, w, r, c + 1),
                                               at0(u, h, w, (int64_t)r - 1, c), at0(u, h, w, r + 1, c));
            }
    }
}

// ------------------------------------------------------------------------------------------------------------
// K10: gray = (77R + 150G + 29B) >> 8 on interleaved RGB (readings C4-1, C4-2).  16 pixels per thread:
// three 128-bit loads (48 contiguous bytes), one 128-bit store.
// ------------------------------------------------------------------------------------------------------------
extern "C" __global__ void __launch_bounds__(256) set_k_rgb2gray_u8(const uint8_t* __restrict__ rgb, uint8_t* __restrict__ gray,
                                                                    uint32_t w, uint32_t h) {
    set_pdl_wait(rgb);
    const uint32_t npix = w * h;
    const uint32_t p0 = (blockIdx.x * 256u + threadIdx.x) * 16u;
    if (p0 + 15 < npix) {
        union {
            uint4 v[3];
            uint8_t b[48];
        } in;
        const uint4* src = reinterpret_cast<const uint4*>(rgb + (size_t)p0 * 3);
        in.v[0] = __ldg(src);
        in.v[1] = __ldg(src + 1);
        in.v[2] = __ldg(src + 2);
        union {
            uint4 v;
            uint8_t b[16];
        } o;
#pragma unroll
        for (int k = 0; k < 16; ++k)
            o.b[k] = (uint8_t)((77u * in.b[3 * k] + 150u * in.b[3 * k + 1] + 29u * in.b[3 * k + 2]) >> 8);
        *reinterpret_cast<uint4*>(gray + p0) = o.v;
    } else {
        for (uint32_t p = p0; p < npix && p < p0 + 16; ++p)
            gray[p] = (uint8_t)((77u * rgb[3 * (size_t)p] + 150u * rgb[3 * (size_t)p + 1] + 29u * rgb[3 * (size_t)p + 2]) >> 8);
    }
}

// ------------------------------------------------------------------------------------------------------------
// K11: 3x3 blur [1 2 1; 2 4 2; 1 2 1] >> 4, clamp-to-edge.  Evaluated separably -- horizontal [1 2 1] sums per
// row (<= 1020), then vertical [1 2 1] (<= 4080) and ONE final >> 4 -- which is exactly the 2-D form in integers.
// blockDim = (32, 4), tile = 512 pixels x 16 rows: a lane owns 16 pixels (one 128-bit word) of 4 consecutive rows.
// All six input rows of a lane (4 + the row above and below) are loaded before the first add, so 96 bytes per
// thread are in flight; horizontal neighbours come from the adjacent lanes by shuffle.  Sums are kept as two 16-bit
// halves per register (even pixels / odd pixels of a 32-bit word): every partial sum fits 16 bits, so packed adds
// never carry between the halves.
// ------------------------------------------------------------------------------------------------------------
namespace {
struct HRow {
    uint32_t ev[4], od[4];  // horizontal sums of the even (b0, b2) and odd (b1, b3) pixels of each 32-bit word
};
// wd: the lane's 16 pixels; lb / rb: the pixel left of b0 and right of b15 (already clamped at the image edge)
__device__ __forceinline__ HRow hsum16(const uint4& wd, uint32_t lb, uint32_t rb) {
    const uint32_t x[4] = {wd.x, wd.y, wd.z, wd.w};
    HRow h;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t ev = x[k] & 0x00ff00ffu, od = (x[k] >> 8) & 0x00ff00ffu;
        const uint32_t prev_b3 = k == 0 ? lb : x[k - 1] >> 24;
        const uint32_t next_b0 = k == 3 ? rb : x[k + 1] & 0xffu;
        h.ev[k] = ((od << 16) | prev_b3) + 2u * ev + od;            // (b-1 + 2 b0 + b1, b1 + 2 b2 + b3)
        h.od[k] = ev + 2u * od + ((ev >> 16) | (next_b0 << 16));    // (b0 + 2 b1 + b2, b2 + 2 b3 + b4)
    }
    return h;
}
}  // namespace

extern "C" __global__ void __launch_bounds__(256) set_k_blur3x3_u8(const uint8_t* __restrict__ g, uint8_t* __restrict__ out, uint32_t w,
                                                                   uint32_t h) {
    set_pdl_wait(g);
    const uint32_t r0 = blockIdx.y * kBlurTileH + threadIdx.y * 4u;
    if ((w & 15u) == 0) {
        const uint32_t lane = threadIdx.x;
        const uint32_t x16 = (blockIdx.x * 32u + lane) * 16u;
        const bool active = x16 < w;
        if (r0 >= h) return;  // warp-uniform
        uint4 wd[6];
        uint32_t le[6], re[6];  // edge pixels fetched from memory by the warp's first / last lane
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const uint32_t rr = min(max((int)r0 - 1 + k, 0), (int)h - 1);  // clamp-to-edge rows
            const uint8_t* row = g + (size_t)rr * w;
            wd[k] = active ? __ldg(reinterpret_cast<const uint4*>(row + x16)) : make_uint4(0, 0, 0, 0);
            le[k] = (active && lane == 0 && x16 > 0) ? __ldg(row + x16 - 1) : 0u;
            re[k] = (active && lane == 31 && x16 + 16 < w) ? __ldg(row + x16 + 16) : 0u;
        }
        HRow hr[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            uint32_t lb = __shfl_up_sync(0xffffffffu, wd[k].w >> 24, 1);
            uint32_t rb = __shfl_down_sync(0xffffffffu, wd[k].x & 0xffu, 1);
            if (lane == 0) lb = x16 > 0 ? le[k] : (wd[k].x & 0xffu);             // clamp at the left edge
            if (x16 + 16 >= w) rb = wd[k].w >> 24;                                // clamp at the right edge
            else if (lane == 31) rb = re[k];
            hr[k] = hsum16(wd[k], lb, rb);
        }
        if (!active) return;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (r0 + k < h) {
                uint32_t o[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t ve = hr[k].ev[q] + 2u * hr[k + 1].ev[q] + hr[k + 2].ev[q];
                    const uint32_t vo = hr[k].od[q] + 2u * hr[k + 1].od[q] + hr[k + 2].od[q];
                    o[q] = ((ve >> 4) & 0x00ff00ffu) | (((vo >> 4) & 0x00ff00ffu) << 8);
                }
                *reinterpret_cast<uint4*>(out + (size_t)(r0 + k) * w + x16) = make_uint4(o[0], o[1], o[2], o[3]);
            }
        }
    } else {  // ragged width (rows are not 16-byte aligned): per-pixel 9-tap with explicit clamping over the same tile
        const uint32_t x0 = (blockIdx.x * 32u + threadIdx.x) * 16u;
        for (uint32_t r = r0; r < min(r0 + 4u, h); ++r)
            for (uint32_t x = x0; x < min(x0 + 16u, w); ++x) {
                int acc = 0;
#pragma unroll
                for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) {
                        int yy = min(max((int)r + dy, 0), (int)h - 1), xx = min(max((int)x + dx, 0), (int)w - 1);
                        acc += (2 - (dy < 0 ? -dy : dy)) * (2 - (dx < 0 ? -dx : dx)) * (int)g[(size_t)yy * w + xx];
                    }
                out[(size_t)r * w + x] = (uint8_t)(acc >> 4);
            }
    }
}

// ------------------------------------------------------------------------------------------------------------
// K12: 256-bin histogram.  Blurred pixels concentrate (sigma ~ 19 levels), so every warp keeps a private
// histogram in shared memory; the 8 copies are summed and added to the (pre-zeroed) global bins with one
// atomic per non-empty bin per block.
// ------------------------------------------------------------------------------------------------------------
extern "C" __global__ void __launch_bounds__(256) set_k_hist256_u8(const uint8_t* __restrict__ p, uint32_t* __restrict__ hist,
                                                                   uint32_t w, uint32_t h) {
    set_pdl_wait(p);
    static_assert(kHistPixPerBlock == 256 * 16, "one 128-bit load per thread");
    const uint32_t n = w * h;
    __shared__ uint32_t sh[8][256];
    const int tid = threadIdx.x, wid = tid >> 5;
    const uint32_t end = min((blockIdx.x + 1u) * (uint32_t)kHistPixPerBlock, n);
    const uint32_t i = blockIdx.x * (uint32_t)kHistPixPerBlock + tid * 16u;
    const bool full = i + 15 < end;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (full) v = __ldg(reinterpret_cast<const uint4*>(p + i));  // in flight while the histograms are cleared
    for (int k = tid; k < 8 * 256; k += 256) (&sh[0][0])[k] = 0;
    __syncthreads();
    uint32_t* my = sh[wid];
    if (full) {
        const uint32_t wds[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            atomicAdd(&my[wds[k] & 0xff], 1u);
            atomicAdd(&my[(wds[k] >> 8) & 0xff], 1u);
            atomicAdd(&my[(wds[k] >> 16) & 0xff], 1u);
            atomicAdd(&my[wds[k] >> 24], 1u);
        }
    } else {
        for (uint32_t j = i; j < end; ++j) atomicAdd(&my[p[j]], 1u);  // ragged tail of the image
    }
    __syncthreads();
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += sh[k][tid];
    if (s) atomicAdd(&hist[tid], s);
}
