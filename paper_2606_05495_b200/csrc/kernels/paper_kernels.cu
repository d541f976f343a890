// paper_kernels.cu -- stage kernels of the two paper workloads added in round 2:
//   config 6, the five-stage Sobel chain:  K10 gray (stencil_kernels.cu) -> K17 sobel -> K18 mean3x3 ->
//             K19 threshold -> K20 blend, all integer, bit-exact (readings S6-1..S6-6)
//   config 5, frontier Bellman-Ford SSSP:  K21 init -> WHILE { K22 relax x U -> K23 control } (readings S5-1..S5-4);
//             the loop is a conditional WHILE node of the job graph and K23 sets its condition on the device;
//             variant 1: K25, the whole job in one kernel of one block.
// Hand-written CUDA for sm_100a.  The frames (0.3 - 2 MB) and graphs (~0.6 MB) sit in L2 right after the H2D copy, so
// these are latency-class kernels like those of configs 0, 1 and 4: coalesced 128-bit accesses; only K25 uses shared memory.
#include "kernels.h"

namespace {

// ---- 3 x 3 neighbourhoods on a byte image, clamp-to-edge, in K11's arrangement (stencil_kernels.cu) ---------------------
// blockDim = (32, 4), tile = 512 pixels x 16 rows: a lane owns 16 pixels (one 128-bit word) of 4 consecutive rows.  The six
// input rows of a lane (4 + the row above and below) are loaded before the first add; horizontal neighbours come from the
// adjacent lanes by shuffle.  Per row, sums are kept as two 16-bit halves per register (the even pixels b0, b2 and the odd
// pixels b1, b3 of each 32-bit word): every partial sum below fits 16 bits, so packed adds never carry between the halves.
struct Packed16 {
    uint32_t ev[4], od[4];
};
// left / right neighbours of the even and of the odd pixels of word k, as packed halves
__device__ __forceinline__ void neighbours(const uint32_t (&x)[4], int k, uint32_t lb, uint32_t rb, uint32_t& ev, uint32_t& od, uint32_t& le,
                                           uint32_t& re, uint32_t& lo, uint32_t& ro) {
    ev = x[k] & 0x00ff00ffu;          // (b0, b2)
    od = (x[k] >> 8) & 0x00ff00ffu;   // (b1, b3)
    const uint32_t prev_b3 = k == 0 ? lb : x[k - 1] >> 24;
    const uint32_t next_b0 = k == 3 ? rb : x[k + 1] & 0xffu;
    le = (od << 16) | prev_b3;        // left of (b0, b2) = (b-1, b1)
    re = od;                          // right of (b0, b2) = (b1, b3)
    lo = ev;                          // left of (b1, b3) = (b0, b2)
    ro = (ev >> 16) | (next_b0 << 16);  // right of (b1, b3) = (b2, b4)
}
// per row: horizontal [1 c 1] sums (c = 1: <= 765, c = 2: <= 1020) and biased horizontal differences right - left + 255 (0 .. 510)
template <uint32_t kCentre>
__device__ __forceinline__ Packed16 hsum16(const uint4& wd, uint32_t lb, uint32_t rb) {
    const uint32_t x[4] = {wd.x, wd.y, wd.z, wd.w};
    Packed16 r;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint32_t ev, od, le, re, lo, ro;
        neighbours(x, k, lb, rb, ev, od, le, re, lo, ro);
        r.ev[k] = le + kCentre * ev + re;
        r.od[k] = lo + kCentre * od + ro;
    }
    return r;
}
__device__ __forceinline__ Packed16 hdiff16(const uint4& wd, uint32_t lb, uint32_t rb) {
    const uint32_t x[4] = {wd.x, wd.y, wd.z, wd.w};
    Packed16 r;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint32_t ev, od, le, re, lo, ro;
        neighbours(x, k, lb, rb, ev, od, le, re, lo, ro);
        r.ev[k] = (re + 0x00ff00ffu) - le;  // each half: 255 - left >= 0, so no borrow crosses into the other half
        r.od[k] = (ro + 0x00ff00ffu) - lo;
    }
    return r;
}
// The lane's 16 pixels of rows r0 - 1 .. r0 + 4 (clamped) and the pixel on either side of them (clamped at the image's edge).
struct Lane16 {
    uint4 wd[6];
    uint32_t lb[6], rb[6];
};
__device__ __forceinline__ void load_lane16(const uint8_t* __restrict__ in, uint32_t w, uint32_t h, uint32_t r0, uint32_t x16, bool active, Lane16& L) {
    const uint32_t lane = threadIdx.x;
    uint32_t le[6], re[6];  // edge pixels fetched from memory by the warp's first / last lane
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const uint32_t rr = min(max((int)r0 - 1 + k, 0), (int)h - 1);
        const uint8_t* row = in + (size_t)rr * w;
        L.wd[k] = active ? __ldg(reinterpret_cast<const uint4*>(row + x16)) : make_uint4(0, 0, 0, 0);
        le[k] = (active && lane == 0 && x16 > 0) ? __ldg(row + x16 - 1) : 0u;
        re[k] = (active && lane == 31 && x16 + 16 < w) ? __ldg(row + x16 + 16) : 0u;
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        uint32_t lb = __shfl_up_sync(0xffffffffu, L.wd[k].w >> 24, 1);
        uint32_t rb = __shfl_down_sync(0xffffffffu, L.wd[k].x & 0xffu, 1);
        if (lane == 0) lb = x16 > 0 ? le[k] : (L.wd[k].x & 0xffu);  // clamp at the left edge
        if (x16 + 16 >= w) rb = L.wd[k].w >> 24;                    // clamp at the right edge
        else if (lane == 31) rb = re[k];
        L.lb[k] = lb;
        L.rb[k] = rb;
    }
}
// ragged width (rows are not 16-byte aligned): the thread's 16 x 4 pixels one by one, nine clamped taps each
template <typename F>
__device__ __forceinline__ void stencil_ragged(const uint8_t* __restrict__ in, uint8_t* __restrict__ out, uint32_t w, uint32_t h, uint32_t r0, F f) {
    const uint32_t x0 = (blockIdx.x * 32u + threadIdx.x) * 16u;
    for (uint32_t r = r0; r < min(r0 + 4u, h); ++r)
        for (uint32_t x = x0; x < min(x0 + 16u, w); ++x) {
            int t[9];
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) {
                    const int yy = min(max((int)r + dy, 0), (int)h - 1), xx = min(max((int)x + dx, 0), (int)w - 1);
                    t[(dy + 1) * 3 + dx + 1] = in[(size_t)yy * w + xx];
                }
            out[(size_t)r * w + x] = (uint8_t)f(t[0], t[1], t[2], t[3], t[4], t[5], t[6], t[7], t[8]);
        }
}
__device__ __forceinline__ uint32_t interleave(uint32_t ev, uint32_t od) { return (ev & 0x00ff00ffu) | ((od & 0x00ff00ffu) << 8); }

}  // namespace

// K17: e = min(255, |gx| + |gy|), gx = [-1 0 1; -2 0 2; -1 0 1] * n, gy = its transpose (reading S6-2).
// gx = vertical [1 2 1] of the rows' horizontal differences (right - left), gy = the bottom row's horizontal [1 2 1] sum
// minus the top row's.  Both are carried with a bias of 1020 so that the packed halves stay non-negative (0 .. 2040).
extern "C" __global__ void __launch_bounds__(128) set_k_sobel3x3_u8(const uint8_t* __restrict__ n, uint8_t* __restrict__ e, uint32_t w, uint32_t h) {
    set_pdl_wait(n);
    const uint32_t r0 = blockIdx.y * kBlurTileH + threadIdx.y * 4u;
    if ((w & 15u) != 0) {
        stencil_ragged(n, e, w, h, r0, [](int a, int b, int c, int d, int, int f, int g, int hh, int i) -> uint32_t {
            const int gx = (c - a) + 2 * (f - d) + (i - g);
            const int gy = (g - a) + 2 * (hh - b) + (i - c);
            const int m = abs(gx) + abs(gy);
            return (uint32_t)(m > 255 ? 255 : m);
        });
        return;
    }
    const uint32_t x16 = (blockIdx.x * 32u + threadIdx.x) * 16u;
    const bool active = x16 < w;
    if (r0 >= h) return;  // warp-uniform
    Lane16 L;
    load_lane16(n, w, h, r0, x16, active, L);
    Packed16 hd[6], hs[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        hd[k] = hdiff16(L.wd[k], L.lb[k], L.rb[k]);
        hs[k] = hsum16<2>(L.wd[k], L.lb[k], L.rb[k]);
    }
    if (!active) return;
    constexpr uint32_t kBias = 0x03fc03fcu;  // 1020 in both halves
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (r0 + k >= h) break;
        uint32_t o[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t m[2];
#pragma unroll
            for (int par = 0; par < 2; ++par) {  // even pixels, odd pixels
                const uint32_t* d0 = par ? hd[k].od : hd[k].ev;
                const uint32_t* d1 = par ? hd[k + 1].od : hd[k + 1].ev;
                const uint32_t* d2 = par ? hd[k + 2].od : hd[k + 2].ev;
                const uint32_t* s0 = par ? hs[k].od : hs[k].ev;
                const uint32_t* s2 = par ? hs[k + 2].od : hs[k + 2].ev;
                const uint32_t gxb = d0[q] + 2u * d1[q] + d2[q];   // gx + 1020 per half
                const uint32_t gyb = s2[q] + (kBias - s0[q]);      // gy + 1020 per half (s0 <= 1020: no borrow)
                const uint32_t ax = __vabsdiffu2(gxb, kBias), ay = __vabsdiffu2(gyb, kBias);
                m[par] = __vminu2(ax + ay, 0x00ff00ffu);           // |gx| + |gy| <= 2040: no carry between the halves
            }
            o[q] = interleave(m[0], m[1]);
        }
        *reinterpret_cast<uint4*>(e + (size_t)(r0 + k) * w + x16) = make_uint4(o[0], o[1], o[2], o[3]);
    }
}

// K18: m = (sum of the 3 x 3 neighbourhood) / 9, integer division (reading S6-3).  Sum <= 2295; floor(v / 9) =
// (v * 7282) >> 16 for every v in that range (checked exhaustively in tests/test_host_logic.py).
extern "C" __global__ void __launch_bounds__(128) set_k_mean3x3_u8(const uint8_t* __restrict__ e, uint8_t* __restrict__ m, uint32_t w, uint32_t h) {
    set_pdl_wait(e);
    const uint32_t r0 = blockIdx.y * kBlurTileH + threadIdx.y * 4u;
    if ((w & 15u) != 0) {
        stencil_ragged(e, m, w, h, r0, [](int a, int b, int c, int d, int ee, int f, int g, int hh, int i) -> uint32_t {
            return (uint32_t)(a + b + c + d + ee + f + g + hh + i) / 9u;
        });
        return;
    }
    const uint32_t x16 = (blockIdx.x * 32u + threadIdx.x) * 16u;
    const bool active = x16 < w;
    if (r0 >= h) return;  // warp-uniform
    Lane16 L;
    load_lane16(e, w, h, r0, x16, active, L);
    Packed16 hs[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) hs[k] = hsum16<1>(L.wd[k], L.lb[k], L.rb[k]);
    if (!active) return;
    auto div9 = [](uint32_t v) { return (((v & 0xffffu) * 7282u) >> 16) | ((((v >> 16) * 7282u) >> 16) << 16); };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (r0 + k >= h) break;
        uint32_t o[4];
#pragma unroll
        for (int q = 0; q < 4; ++q)
            o[q] = interleave(div9(hs[k].ev[q] + hs[k + 1].ev[q] + hs[k + 2].ev[q]), div9(hs[k].od[q] + hs[k + 1].od[q] + hs[k + 2].od[q]));
        *reinterpret_cast<uint4*>(m + (size_t)(r0 + k) * w + x16) = make_uint4(o[0], o[1], o[2], o[3]);
    }
}

// K19: t = m >= thresh ? 255 : 0 (reading S6-4).  16 pixels per thread: one 128-bit load, one 128-bit store.
extern "C" __global__ void __launch_bounds__(256) set_k_threshold_u8(const uint8_t* __restrict__ m, uint8_t* __restrict__ t, uint32_t w, uint32_t h,
                                                                      uint32_t thresh) {
    set_pdl_wait(m);
    const uint32_t npix = w * h;
    const uint32_t p0 = (blockIdx.x * 256u + threadIdx.x) * 16u;
    const uint32_t th4 = thresh * 0x01010101u;
    if (p0 + 15 < npix && ((reinterpret_cast<uintptr_t>(m) | reinterpret_cast<uintptr_t>(t)) & 15u) == 0) {
        uint4 v = __ldg(reinterpret_cast<const uint4*>(m + p0));
        // per-byte unsigned compare: 0xff where m >= thresh
        v.x = __vcmpgeu4(v.x, th4);
        v.y = __vcmpgeu4(v.y, th4);
        v.z = __vcmpgeu4(v.z, th4);
        v.w = __vcmpgeu4(v.w, th4);
        *reinterpret_cast<uint4*>(t + p0) = v;
    } else {
        for (uint32_t p = p0; p < npix && p < p0 + 16; ++p) t[p] = m[p] >= thresh ? 255 : 0;
    }
}

// K20: out = (128 t + 128 n) >> 8 = (t + n) >> 1 per byte (reading S6-5): the halving add without rounding.
extern "C" __global__ void __launch_bounds__(256) set_k_blend_u8(const uint8_t* __restrict__ t, const uint8_t* __restrict__ n, uint8_t* __restrict__ out,
                                                                  uint32_t w, uint32_t h) {
    set_pdl_wait(t, n);
    const uint32_t npix = w * h;
    const uint32_t p0 = (blockIdx.x * 256u + threadIdx.x) * 16u;
    if (p0 + 15 < npix && ((reinterpret_cast<uintptr_t>(t) | reinterpret_cast<uintptr_t>(n) | reinterpret_cast<uintptr_t>(out)) & 15u) == 0) {
        const uint4 a = __ldg(reinterpret_cast<const uint4*>(t + p0)), b = __ldg(reinterpret_cast<const uint4*>(n + p0));
        uint4 o;
        o.x = __vhaddu4(a.x, b.x);
        o.y = __vhaddu4(a.y, b.y);
        o.z = __vhaddu4(a.z, b.z);
        o.w = __vhaddu4(a.w, b.w);
        *reinterpret_cast<uint4*>(out + p0) = o;
    } else {
        for (uint32_t p = p0; p < npix && p < p0 + 16; ++p) out[p] = (uint8_t)(((uint32_t)t[p] + (uint32_t)n[p]) >> 1);
    }
}

// ------------------------------------------------------------------------------------------------------------
// SSSP.  Device image of a job (mirrors host_in): int32 [V, E, src, 0][row_ptr V+1][col E][w E].
// out: int32 [dist V][rounds, 0, 0, 0] (mirrors host_out).
// scratch: uint32 flags[2][maxV], then ctrl[16] = {-, rounds, relaxations done, -, changed[0..U-1], ...}.
// The frontier is a flag per vertex, double-buffered by the parity of the relaxation's running number, so that a
// relaxation never clears a flag another thread of the same relaxation is setting.  Distances are relaxed IN PLACE with
// atomicMin: a vertex may pick up a distance lowered earlier in the same round, so the GPU needs at most as many rounds
// as the oracle's synchronous rounds and ends on the same, unique, distances (reading S5-4).
// One pass of the WHILE body is U relaxation kernels (sub = 0 .. U-1) and the control kernel: every pass of a WHILE node
// costs a device-side relaunch that the chip serialises over all graphs in flight (about 4-5 us), while
// a relaxation over an empty frontier is a 2 us kernel, so U = 4 trades up to U-1 of those for 3/4 of the relaunches.
// ------------------------------------------------------------------------------------------------------------
constexpr int kSsspInf = 0x7fffffff;
constexpr uint32_t kSsspCtrlWords = 16, kSsspRounds = 1, kSsspDone = 2, kSsspChanged = 4;

extern "C" __global__ void __launch_bounds__(256) set_k_sssp_init(const int32_t* __restrict__ img, int32_t* __restrict__ out, uint32_t* __restrict__ scratch,
                                                                  uint32_t max_v) {
    set_pdl_sync(img);
    const uint32_t V = min((uint32_t)img[0], max_v), src = (uint32_t)img[2];
    uint32_t* f0 = scratch;
    uint32_t* f1 = scratch + max_v;
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < V; v += gridDim.x * blockDim.x) {
        out[v] = v == src ? 0 : kSsspInf;
        f0[v] = v == src ? 1u : 0u;
        f1[v] = 0u;
    }
    if (blockIdx.x == 0 && threadIdx.x < kSsspCtrlWords) {
        scratch[2 * (size_t)max_v + threadIdx.x] = 0u;
        if (threadIdx.x < 4) out[V + threadIdx.x] = 0;
    }
}

// K22: kSsspLanes threads per vertex (a group never straddles a warp): lane g of the group relaxes edges g, g + 8, ... of
// its vertex, so a round is one dependent chain flag -> row_ptr -> (col, w) -> atomicMin whatever the out-degree, instead
// of out-degree atomics one behind the other.  The flag is read by the whole group before lane 0 clears it.
extern "C" __global__ void __launch_bounds__(256) set_k_sssp_relax(const int32_t* __restrict__ img, int32_t* __restrict__ out, uint32_t* __restrict__ scratch,
                                                                   uint32_t max_v, uint32_t sub) {
    set_pdl_sync(img);
    const uint32_t V = min((uint32_t)img[0], max_v);
    const int32_t* row_ptr = img + 4;
    const int32_t* col = row_ptr + V + 1;
    const int32_t* wgt = col + img[1];
    uint32_t* ctrl = scratch + 2 * (size_t)max_v;
    const uint32_t number = ctrl[kSsspDone] + sub;  // this relaxation's running number within the job
    uint32_t* fin = scratch + (number & 1u) * (size_t)max_v;
    uint32_t* fout = scratch + ((number + 1u) & 1u) * (size_t)max_v;
    constexpr uint32_t kPerWarp = 32 / kSsspLanes;
    const uint32_t g = threadIdx.x % kSsspLanes, in_warp = (threadIdx.x % 32) / kSsspLanes;
    const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) / 32, warps = gridDim.x * blockDim.x / 32;
    bool any = false;
    for (uint32_t base = warp * kPerWarp; base < V; base += warps * kPerWarp) {  // uniform over the warp
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
    if (any) ctrl[kSsspChanged + sub] = 1u;  // the next relaxation's frontier is not empty
}

// K23: the loop's condition.  One thread: count the rounds that had a frontier (relaxation 0 of a pass always has one;
// relaxation s + 1 has one iff relaxation s lowered a distance), report the count, and keep the WHILE node going while the
// last relaxation of the pass lowered some distance (at most V rounds: Bellman-Ford's bound with non-negative weights).
extern "C" __global__ void set_k_sssp_control(const int32_t* __restrict__ img, int32_t* __restrict__ out, uint32_t* __restrict__ scratch, uint32_t max_v,
                                              uint32_t unroll, cudaGraphConditionalHandle loop) {
    set_pdl_sync(img);
    const uint32_t V = min((uint32_t)img[0], max_v);
    uint32_t* ctrl = scratch + 2 * (size_t)max_v;
    uint32_t rounds = ctrl[kSsspRounds] + 1u;
    for (uint32_t s = 0; s + 1 < unroll; ++s) rounds += ctrl[kSsspChanged + s] ? 1u : 0u;
    const uint32_t last = ctrl[kSsspChanged + unroll - 1];
    for (uint32_t s = 0; s < unroll; ++s) ctrl[kSsspChanged + s] = 0u;
    ctrl[kSsspRounds] = rounds;
    ctrl[kSsspDone] += unroll;
    out[V] = (int32_t)rounds;
    cudaGraphSetConditional(loop, (last != 0u && rounds <= V) ? 1u : 0u);
}

// K25: the whole SSSP job in ONE kernel of ONE block (config 5 variant 1, and set_sssp_noalloc): initialisation, every
// round, the round count -- with __syncthreads() between rounds instead of a pass of a WHILE node (a device-side relaunch
// of 4 - 5 us that the chip serialises over all graphs in flight).  Same image, same out, same result as
// K21-K23.  The distances and the frontier flags live in SHARED memory for the whole job (one SM's atomic and scattered
// store traffic to L2 bounded the first version: 150 us per job at V = 4096 with everything in global memory); global
// memory sees the read-only graph, the work list and, at the end, one coalesced store of the distances.
// A round is two phases of the block:
//   A  every thread looks at the frontier flags of its own vertices (one 32-bit load = 4 byte flags), clears them and
//      appends the flagged vertices to the work list (position from a shared-memory counter);
//   B  groups of kSsspLanes threads take the list's vertices and relax their out-edges in place with atomicMin (K22's
//      relaxation), flagging every vertex whose distance got smaller for the next round.
// Phases never overlap, so ONE flag array is enough, and only frontier vertices cost a dependent chain of loads.
// Dynamic shared memory: set_sssp_solo_smem_bytes(max_v) = int32 dist[max_v] + byte flags[max_v]; scratch (global): the
// work list, uint32[max_v].  Everything the job reads from either it writes first: an earlier job's leftovers never matter.
// A block is the limit of this variant (max_v <= kSsspSoloMaxV so that the distances fit one SM's shared memory; a round
// of a full frontier is V / 128 steps of the block): it is meant for graphs of a few thousand vertices -- the paper's
// "many small jobs" -- and the WHILE-node pipeline stays the general one.
extern "C" uint32_t set_sssp_solo_smem_bytes(uint32_t max_v) { return 4u * max_v + ((max_v + 3u) & ~3u); }

extern "C" __global__ void __launch_bounds__(kSsspSoloThreads) set_k_sssp_solo(const int32_t* __restrict__ img, int32_t* __restrict__ out,
                                                                               uint32_t* __restrict__ scratch, uint32_t max_v) {
    set_pdl_sync(img);
    extern __shared__ __align__(16) uint8_t solo_smem[];
    __shared__ uint32_t s_n[2];  // length of the work list, by the parity of the round
    int32_t* dist = reinterpret_cast<int32_t*>(solo_smem);
    uint32_t* flag_words = reinterpret_cast<uint32_t*>(solo_smem + 4u * (size_t)max_v);
    uint8_t* flags = reinterpret_cast<uint8_t*>(flag_words);
    uint32_t* list = scratch;
    const uint32_t V = min((uint32_t)img[0], max_v), src = (uint32_t)img[2];
    const int32_t* row_ptr = img + 4;
    const int32_t* col = row_ptr + V + 1;
    const int32_t* wgt = col + img[1];
    const uint32_t words = (V + 3u) / 4u;
    for (uint32_t v = threadIdx.x; v < V; v += kSsspSoloThreads) dist[v] = v == src ? 0 : kSsspInf;
    for (uint32_t w = threadIdx.x; w < words; w += kSsspSoloThreads) flag_words[w] = (src < V && src / 4u == w) ? 1u << (8u * (src % 4u)) : 0u;
    if (threadIdx.x < 2) s_n[threadIdx.x] = 0u;
    const uint32_t g = threadIdx.x % kSsspLanes, group = threadIdx.x / kSsspLanes;
    constexpr uint32_t kGroups = kSsspSoloThreads / kSsspLanes;
    uint32_t rounds = 0;
    for (;;) {
        __syncthreads();  // the flags and distances of the previous round (or the initialisation) are visible to the block
        uint32_t* n_now = &s_n[rounds & 1u];
        for (uint32_t w = threadIdx.x; w < words; w += kSsspSoloThreads) {  // phase A
            const uint32_t f = flag_words[w];
            if (f == 0u) continue;
            flag_words[w] = 0u;
            const uint32_t cnt = (f & 1u) + ((f >> 8) & 1u) + ((f >> 16) & 1u) + ((f >> 24) & 1u);
            uint32_t pos = atomicAdd(n_now, cnt);
#pragma unroll
            for (uint32_t b = 0; b < 4; ++b)
                if ((f >> (8u * b)) & 1u) list[pos++] = 4u * w + b;
        }
        __syncthreads();
        const uint32_t n = *n_now;
        if (n == 0u) break;                          // the frontier is empty: done
        rounds += 1u;                                // a round that had a frontier
        if (threadIdx.x == 0) s_n[rounds & 1u] = 0u;  // the next round's counter: last read before the barrier above
        for (uint32_t i = group; i < n; i += kGroups) {  // phase B
            const uint32_t u = list[i];
            const int32_t du = *reinterpret_cast<volatile int32_t*>(dist + u);  // finite: u entered the frontier by getting a distance
            const int32_t e1 = __ldg(row_ptr + u + 1);
            for (int32_t e = __ldg(row_ptr + u) + (int32_t)g; e < e1; e += (int32_t)kSsspLanes) {
                const int32_t v = __ldg(col + e), nd = du + __ldg(wgt + e);
                if (nd < atomicMin(dist + v, nd)) flags[v] = 1u;
            }
        }
        if (rounds > V) break;  // at most V rounds: Bellman-Ford's bound with non-negative weights (uniform over the block)
    }
    __syncthreads();
    for (uint32_t v = threadIdx.x; v < V; v += kSsspSoloThreads) out[v] = dist[v];
    if (threadIdx.x < 4) out[V + threadIdx.x] = threadIdx.x == 0 ? (int32_t)rounds : 0;
}
