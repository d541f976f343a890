// gemm_sm100.cu -- K9: C = bf16( GELU( A.B + bias ) ), bf16 operands, fp32 accumulation on the 5th-generation tensor
// cores (BASELINE.json:configs[3]; readings C3-1..C3-4).  Hand-written for sm_100a: a CTA PAIR (cluster of two
// CTAs on the two SMs of a TPC) computes one 256 x 256 tile with tcgen05.mma.cta_group::2; TMA (cp.async.bulk.tensor)
// stages 128-byte-swizzled operand tiles in shared memory, the pair's leader issues the MMAs with the accumulator in
// tensor memory (TMEM) of both SMs, and eight epilogue warps per CTA read it back with tcgen05.ld, apply bias + erf-GELU +
// round-to-nearest-even bf16 and store the tile through TMA.
//
//   A : bf16 [M][K] row-major  -> K-major operand.  CTA r of the pair loads rows m0 + 128 r .. + 127: box 64 (K) x 128 (M) = 16 KiB
//   B : bf16 [K][N] row-major  -> MN-major operand (no host transpose).  CTA r loads columns n0 + 128 r .. + 127 as two
//       boxes 64 (N) x 64 (K) = 16 KiB: each SM stages HALF of B and the tensor cores read the other half from the peer's
//       shared memory, so a 256 x 256 tile costs 64 KiB of L2 -> SM traffic per 64-deep k-block instead of the 96 KiB of
//       two independent 128 x 256 tiles.  The one-CTA version of this kernel (round 1) moved 192 MB from L2 for 2048^3,
//       30,000 cycles at the ~6,300 B/cycle the L2 delivers chip-wide against 16,400 cycles of MMA: it was L2-bound.
//   D : fp32, rows 128 r .. 128 r + 127 of the pair's tile x 256 columns = 256 TMEM columns x 128 lanes in CTA r
//
// Grid = (2 * ceil(M / 256), ceil(N / 256)), cluster (2, 1, 1): blockIdx.x >> 1 is the pair's row block, %cluster_ctarank
// the CTA's rank r.  Warp roles (576 threads): warp 0 = TMA producer (both CTAs, each for its own halves, all signalling the
// LEADER's "full" barrier), warp 1 = TMEM allocator (both CTAs) + MMA issuer (leader only; tcgen05.commit multicasts the
// "stage empty" / "accumulator full" arrivals to both CTAs), warps 2..17 = epilogue (warp w may only touch TMEM lanes
// 32*(w%4) .. 32*(w%4)+31; four warps share each lane quarter and take 64 of the 256 columns each).  The epilogue stages the
// tile's bias values in shared memory while the main loop runs, then per 32-column round: tcgen05.ld (the next round's load
// already in flight), packed-f32x2 bias + GELU, bf16 rows into 64-byte-swizzled shared memory, and the 32 x 32 box goes to the
// TMA unit at once (cp.async.bulk.tensor store) so that it drains under the next round's arithmetic.
// What was measured on B200 at 2048^3 (one wave of 64 pairs on 74 TPCs; profiles/r2_k9.md): kernel entry -> first MMA 0.6 us,
// main loop 10.0 us (L2-bound: 128 MB at ~12.8 TB/s; the MMAs alone need 8.3 us), epilogue 3.2 us, kernel-to-kernel 1.9 us.
// Ragged shapes: TMA zero-fills out-of-bounds rows/columns of a load box, so partial tiles in M, N and K contribute
// zeros, and clips a store box to the matrix (N and K must be multiples of 8: 16-byte TMA pitches); a box that starts
// outside the matrix is never requested (its accumulator rows / columns are never stored).
#include <cuda_bf16.h>

#include "kernels.h"

namespace {

constexpr uint32_t kBlockM = 128, kBlockN = 256, kBlockK = 64, kUmmaK = 16;  // per CTA: 128 rows of the pair's 256 x 256 tile
constexpr uint32_t kPairM = 2 * kBlockM, kHalfN = kBlockN / 2;
constexpr uint32_t kStages = 6;
constexpr uint32_t kABytes = kBlockM * kBlockK * 2;          // 16 KiB
constexpr uint32_t kBBoxN = 64;                              // one 128-byte swizzle atom of N per box
constexpr uint32_t kBBoxBytes = kBBoxN * kBlockK * 2;        // 8 KiB
constexpr uint32_t kBBoxes = kHalfN / kBBoxN;                // 2 boxes: this CTA's half of B
constexpr uint32_t kBBytes = kBBoxBytes * kBBoxes;           // 16 KiB
constexpr uint32_t kStageBytes = kABytes + kBBytes;          // 32 KiB
constexpr uint32_t kCBoxBytes = 32 * 32 * 2;                 // epilogue staging: one TMA store box, 32 columns x 32 rows of bf16, 64-byte swizzle
static_assert(32 * kCBoxBytes <= kStages * kStageBytes, "the epilogue stages its 32 boxes in the idle operand ring");
constexpr uint32_t kTmemCols = 256;
constexpr uint32_t kEpiWarps = 16;                      // four per TMEM lane quarter, 64 columns (one TMA store box) each
constexpr uint32_t kThreads = (2 + kEpiWarps) * 32;     // + TMA producer warp + MMA issuer warp = 576
constexpr uint32_t kBarrierBytes = 256;
constexpr uint32_t kBiasBytes = kBlockN * 4;  // the tile's 256 bias values, staged by the epilogue warps while the main loop runs
constexpr uint32_t kSmemBytes = kStages * kStageBytes + kBarrierBytes + kBiasBytes + 1024;  // + slack for 1024-byte alignment

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity)
        : "memory");
}
// TMA load into THIS CTA's shared memory whose completion bytes are counted on `bar`, a shared::cluster address that may
// belong to the other CTA of the pair (the leader's "full" barrier)
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int32_t c_inner, int32_t c_outer) {
    asm volatile("cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
                 "l"(tm), "r"(bar), "r"(c_inner), "r"(c_outer)
                 : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    // no .release.cluster: a cluster-scope release drains the thread's outstanding TMA loads first (measured: the non-leader's
    // ring then runs one stage at a time, 0.65 us per k-block whatever its depth).  The data itself is published by the TMA
    // unit's complete_tx on the same barrier; this arrival only balances the barrier's count.
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Cluster barrier without memory ordering: for "nobody leaves before everybody is done".  (A releasing arrive waits for the
// thread's outstanding writes, TMA stores included, to be performed -- a microsecond at the end of the epilogue.)
__device__ __forceinline__ void cluster_sync_relaxed() {
    asm volatile("barrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}

// Shared-memory matrix descriptor (tcgen05): start address, leading / stride byte offsets (all >> 4), descriptor
// version 1, 128-byte swizzle.  K-major A tile [128 rows][64 k]: 8-row groups are 1024 B apart (SBO), LBO unused.
// MN-major B tile: 64 (N) x 8 (K) swizzle atoms; the next 8 K rows are 1024 B on (SBO), the next 64 columns of N
// are one TMA box = 8 KiB on (LBO).
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((addr >> 4) & 0x3fffu);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32;
    d |= 1ull << 46;  // descriptor version (Blackwell)
    d |= 2ull << 61;  // SWIZZLE_128B
    return d;
}

// Instruction descriptor, kind::f16: D fp32, A and B bf16, A K-major, B MN-major, N >> 3, M >> 4 -- the shape is the
// PAIR's: M = 256 (128 rows per CTA), N = 256 (128 columns of B staged per CTA).
constexpr uint32_t kInstrDesc = (1u << 4) | (1u << 7) | (1u << 10) | (0u << 15) | (1u << 16) | ((kBlockN >> 3) << 17) | ((kPairM >> 4) << 24);

__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(kInstrDesc), "r"(accumulate)
        : "memory");
}
// Arrives on the mbarrier at this shared-memory offset in BOTH CTAs of the pair once every tcgen05.mma issued so far by
// this thread has completed.
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
    const uint16_t both = 3;
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar), "h"(both)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
          "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
          "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}

// GELU, erf form (reading C3-3): 0.5 z (1 + erf(z / sqrt 2)), evaluated in fp32, TWO elements per call.  The epilogue is
// issue- and MUFU-bound (32,768 elements per CTA through four schedulers and four 4-lane MUFU units; the scalar erff()
// version compiled to ~30 instructions per element and took 6 us of the kernel's 17), so (1) erf is one branch-free
// expression with ONE special-function instruction per element:
//     erfc(|x|) = 1 / (1 + a1 |x| + ... + a6 |x|^6)^16        (Abramowitz & Stegun 7.1.28, |error| <= 3e-7 absolute;
// the 1 / sqrt 2 of x = z / sqrt 2 is folded into the coefficients; round 2's first version used 7.1.26, which needs a
// reciprocal AND an exponential: 2 MUFU per element, 2.1 us of MUFU time per CTA), and 0.5 z (1 + erf x) =
// hz + |hz| (1 - erfc|x|) with hz = z / 2: for z < 0 the sum cancels to hz erfc|x| with an absolute error of an ulp of hz,
// far below the bf16 rounding of anything that is not itself negligible (tests: <= 1 bf16 ulp where |GELU| >= 1e-3, 4e-6
// absolute below); and (2) every multiply and add is a packed f32x2 instruction (sm_100 FFMA2 / FMUL2 / FADD2: two fp32
// lanes per issue slot).  A power that overflows gives rcp(inf) = 0: erf = 1.  Per pair: 13 packed FP, 2 MUFU, 4 LOP.
__device__ __forceinline__ float2 gelu_erf2(float2 z) {
    constexpr float kA1 = 0.0705230784f * 0.70710678118654752440f, kA2 = 0.0422820123f * 0.5f,
                    kA3 = 0.0092705272f * 0.35355339059327376220f, kA4 = 0.0001520143f * 0.25f,
                    kA5 = 0.0002765672f * 0.17677669529663688110f, kA6 = 0.0000430638f * 0.125f;
    const float2 az = make_float2(fabsf(z.x), fabsf(z.y));
    float2 d = __ffma2_rn(make_float2(kA6, kA6), az, make_float2(kA5, kA5));
    d = __ffma2_rn(d, az, make_float2(kA4, kA4));
    d = __ffma2_rn(d, az, make_float2(kA3, kA3));
    d = __ffma2_rn(d, az, make_float2(kA2, kA2));
    d = __ffma2_rn(d, az, make_float2(kA1, kA1));
    d = __ffma2_rn(d, az, make_float2(1.0f, 1.0f));
    d = __fmul2_rn(d, d);
    d = __fmul2_rn(d, d);
    d = __fmul2_rn(d, d);
    d = __fmul2_rn(d, d);  // (1 + ...)^16
    float2 r;              // erfc(|x|)
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r.x) : "f"(d.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r.y) : "f"(d.y));
    const float2 hz = __fmul2_rn(z, make_float2(0.5f, 0.5f));
    const float2 m = __fadd2_rn(make_float2(1.0f, 1.0f), make_float2(-r.x, -r.y));  // erf(|x|)
    return __ffma2_rn(make_float2(fabsf(hz.x), fabsf(hz.y)), m, hz);
}

}  // namespace

extern "C" uint32_t set_gemm_smem_bytes(void) { return kSmemBytes; }
extern "C" uint32_t set_gemm_threads(void) { return kThreads; }

extern "C" __global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
set_k_gemm_bias_gelu_bf16(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                          const __grid_constant__ CUtensorMap tmC, const float* __restrict__ bias, uint32_t M, uint32_t N, uint32_t K) {
    extern __shared__ uint8_t smem_raw[];
    // Both CTAs of the pair must carve shared memory identically: the MMA reads the peer's operand tiles at the leader's
    // offsets and tcgen05.commit signals the peer's barriers at the leader's offsets.  The dynamic shared memory base is
    // the same in every CTA of a launch, so the same rounding gives the same offsets.
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;  // 128-byte swizzle atoms repeat every 1024 B
    const uint32_t bars = base + kStages * kStageBytes;
    // barrier block: full[kStages] (used in the leader only), empty[kStages], accum_full, then the TMEM base address
    auto full_bar = [&](uint32_t s) { return bars + 8u * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8u * (kStages + s); };
    const uint32_t accum_bar = bars + 8u * (2 * kStages);
    const uint32_t tmem_ready = bars + 8u * (2 * kStages + 1);  // in the leader: TMEM allocated in both CTAs
    const uint32_t tmem_slot = bars + 8u * (2 * kStages + 2);
    const uint32_t bias_tile = bars + kBarrierBytes;  // float[256]
    auto a_tile = [&](uint32_t s) { return base + s * kStageBytes; };
    auto b_tile = [&](uint32_t s) { return base + s * kStageBytes + kABytes; };

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();             // 0 = leader of the pair
    const uint32_t mp0 = (blockIdx.x >> 1) * kPairM;     // first row of the pair's tile
    const uint32_t m0 = mp0 + rank * kBlockM;            // first row of THIS CTA's half
    const uint32_t n0 = blockIdx.y * kBlockN;            // first column of the pair's tile
    const uint32_t num_kb = (K + kBlockK - 1) / kBlockK;
    // What CTA r stages per k-block: its A box if its rows start inside the matrix, and the B boxes of its column half that
    // start inside the matrix.  The leader expects the bytes of both CTAs on its "full" barrier.
    auto a_valid = [&](uint32_t r) { return mp0 + r * kBlockM < M; };
    auto b_boxes = [&](uint32_t r) {
        const uint32_t nb = n0 + r * kHalfN;
        return nb >= N ? 0u : min((N - nb + kBBoxN - 1) / kBBoxN, kBBoxes);
    };
    const bool my_a = a_valid(rank);
    const uint32_t my_boxes = b_boxes(rank);
    const uint32_t pair_tx = (a_valid(0) ? kABytes : 0u) + (a_valid(1) ? kABytes : 0u) + (b_boxes(0) + b_boxes(1)) * kBBoxBytes;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmC) : "memory");
        for (uint32_t s = 0; s < kStages; ++s) {
            mbar_init(full_bar(s), 2);  // the leader's arrive.expect_tx and the peer's remote arrive
            mbar_init(empty_bar(s), 1);
        }
        mbar_init(accum_bar, 1);
        mbar_init(tmem_ready, 2);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster_sync_all();  // barriers initialised in BOTH CTAs before anyone signals
    // Programmatic dependent launch (set.h SET_STAGE_PDL): the prologue above (tensor-map prefetch, barrier init) and the
    // TMEM allocation below may overlap the node before this one; nothing may read A, B or bias, or write C, before that
    // node's writes are visible.  Both instructions do nothing over an ordinary edge.
    set_pdl_sync(bias);
    // The producer warp goes straight to its first loads; the TMEM allocation (0.2 - 0.4 us) runs beside their latency.
    uint32_t tmem_base = 0;
    if (warp != 0) {
        if (warp == 1) {  // TMEM: 256 columns in each CTA for its 128 x 256 fp32 half of the accumulator
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(kTmemCols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
            if (lane == 0) mbar_arrive_cluster(map_to_cta(tmem_ready, 0));  // the leader's issuer waits for both allocations
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        asm volatile("bar.sync 2, %0;" ::"n"((1 + kEpiWarps) * 32) : "memory");  // issuer warp + epilogue warps: the address is in shared memory
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot) : "memory");
    }

    if (warp == 0) {
        // ===== TMA producer: every CTA stages its own halves; all bytes are counted on the leader's barrier =====
        if (elect_one()) {
            for (uint32_t kb = 0; kb < num_kb; ++kb) {
                const uint32_t s = kb % kStages, round = kb / kStages;
                mbar_wait(empty_bar(s), (round & 1u) ^ 1u);  // first pass over the ring falls through
                const uint32_t lead_full = map_to_cta(full_bar(s), 0);
                if (rank == 0)
                    mbar_expect_tx(full_bar(s), pair_tx);
                else
                    mbar_arrive_cluster(lead_full);
                if (my_a) tma_load_2d(a_tile(s), &tmA, lead_full, (int32_t)(kb * kBlockK), (int32_t)m0);
                for (uint32_t j = 0; j < my_boxes; ++j)
                    tma_load_2d(b_tile(s) + j * kBBoxBytes, &tmB, lead_full, (int32_t)(n0 + rank * kHalfN + j * kBBoxN), (int32_t)(kb * kBlockK));
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: one thread of the LEADER drives the tensor cores of both SMs =====
        if (rank == 0 && elect_one()) {
            mbar_wait(tmem_ready, 0);
            for (uint32_t kb = 0; kb < num_kb; ++kb) {
                const uint32_t s = kb % kStages, round = kb / kStages;
                mbar_wait(full_bar(s), round & 1u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (uint32_t k = 0; k < kBlockK / kUmmaK; ++k) {
                    // A: 16 K-elements = 32 bytes further along the swizzled 128-byte row
                    const uint64_t adesc = smem_desc(a_tile(s) + k * kUmmaK * 2u, 16u, 1024u);
                    // B: 16 K-rows = two 8-row groups = 2048 bytes further; the next 64 columns are one box on
                    const uint64_t bdesc = smem_desc(b_tile(s) + k * kUmmaK * 128u, kBBoxBytes, 1024u);
                    umma_bf16(tmem_base, adesc, bdesc, (kb | k) != 0u);
                }
                umma_commit_pair(empty_bar(s));  // both CTAs may refill the stage once these MMAs have read it
            }
            umma_commit_pair(accum_bar);  // accumulator complete in both CTAs
        }
    } else {
        // ===== epilogue: TMEM -> registers -> bias + GELU -> bf16 -> swizzled smem -> TMA store =====
        // Eight warps: warp w reads TMEM lane quarter q = w % 4 (the only lanes it may touch) and column half
        // h = (w - 2) / 4, i.e. a 32-row x 128-column piece of the tile = two 64-column TMA boxes of 4 KiB.  The
        // operand ring is idle once accum_bar has fired (every MMA has read it, in both CTAs), so the boxes are staged there.
        // While the main loop runs these warps have nothing to do: they stage the tile's 256 bias values in shared memory
        // (zero beyond N), so that the epilogue proper never waits for a global load -- in the first version every
        // 8-column chunk issued its own two bias loads behind the previous chunk's shared-memory store (the asm memory
        // clobbers keep them in order), about 600 cycles each, sixteen times per warp: most of the epilogue's 6 us.
        {
            const uint32_t t = threadIdx.x - 64u;  // 0 .. 511: the first 256 epilogue threads load one bias value each
            if (t < kBlockN) {
                const float bv = n0 + t < N ? __ldg(bias + n0 + t) : 0.0f;
                asm volatile("st.shared.f32 [%0], %1;" ::"r"(bias_tile + 4u * t), "f"(bv) : "memory");
            }
            asm volatile("bar.sync 1, %0;" ::"n"(kEpiWarps * 32) : "memory");  // named barrier: the epilogue warps only
        }
        mbar_wait(accum_bar, 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // Sixteen warps: warp w reads TMEM lane quarter q = w % 4 (the only lanes it may touch) and column group cg = (w - 2) / 4,
        // i.e. a 32-row x 64-column piece of the tile = one TMA store box of 4 KiB.  The operand ring is idle once accum_bar
        // has fired (every MMA has read it, in both CTAs), so the boxes are staged there.  The arithmetic is a dependent chain of
        // ~20 instructions per pair of elements: with eight warps the schedulers issued 15 % of the time (ncu), hence sixteen.
        const uint32_t q = warp & 3u, cg = (warp - 2u) >> 2;
        const uint32_t box0 = base + (cg * 4u + q) * 2u * kCBoxBytes;  // this warp's two store boxes
        // Two rounds of 32 columns; the TMEM load of the second is issued before the first is computed.
        if (m0 + q * 32u < M && n0 + cg * 64u < N) {  // warp-uniform: something of this box lies inside the matrix
            const uint32_t trow = tmem_base + ((q * 32u) << 16) + cg * 64u;
            uint32_t va[32], vb[32];
            tmem_ld32(trow, va);
#pragma unroll
            for (uint32_t r = 0; r < 2; ++r) {
                const uint32_t c0 = cg * 64u + r * 32u;  // first column of the round inside the tile
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (r == 0) tmem_ld32(trow + 32u, vb);
                const uint32_t (&v)[32] = r ? vb : va;
                const uint32_t box = box0 + r * kCBoxBytes;
                const uint32_t srow = box + lane * 64u;  // this lane's 64-byte row of the box
                if (n0 + c0 < N) {  // warp-uniform; N is a multiple of 8, so an 8-column chunk is inside or outside as a whole
#pragma unroll
                    for (uint32_t g = 0; g < 4; ++g) {  // 8 columns -> one 16-byte chunk
                        float4 b0, b1;  // bias of columns c0 + 8g .. + 7 (a broadcast read: every lane reads the same address)
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(b0.x), "=f"(b0.y), "=f"(b0.z), "=f"(b0.w) : "r"(bias_tile + 4u * (c0 + 8u * g)));
                        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(b1.x), "=f"(b1.y), "=f"(b1.z), "=f"(b1.w) : "r"(bias_tile + 4u * (c0 + 8u * g + 4u)));
                        const float2 bb[4] = {make_float2(b0.x, b0.y), make_float2(b0.z, b0.w), make_float2(b1.x, b1.y), make_float2(b1.z, b1.w)};
                        uint32_t o[4];
#pragma unroll
                        for (int t = 0; t < 4; ++t) {
                            const float2 acc = make_float2(__uint_as_float(v[8 * g + 2 * t]), __uint_as_float(v[8 * g + 2 * t + 1]));
                            const float2 res = gelu_erf2(__fadd2_rn(acc, bb[t]));
                            __nv_bfloat162 hh = __floats2bfloat162_rn(res.x, res.y);
                            o[t] = *reinterpret_cast<uint32_t*>(&hh);
                        }
                        // 64-byte swizzle (byte-address bits 4-5 ^= bits 7-8): chunk g of row r lives at chunk position g ^ ((r >> 1) & 3)
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(srow + ((g ^ ((lane >> 1) & 3u)) << 4)), "r"(o[0]), "r"(o[1]),
                                     "r"(o[2]), "r"(o[3]));
                    }
                    // The round's 32 x 32 box goes to the TMA unit at once, so that the first store of every warp (half of the
                    // tile's 64 KiB) drains while the second round is computed.
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the TMA engine
                    __syncwarp();
                    if (lane == 0) {  // rows >= M and columns >= N of the box are clipped by the TMA unit
                        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(&tmC), "r"(box),
                                     "r"((int32_t)(n0 + c0)), "r"((int32_t)(m0 + q * 32u))
                                     : "memory");
                        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                    }
                }
            }
        }
        // the staging memory may go away once the TMA unit has READ it; the writes themselves complete before the grid does
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    // Neither CTA may leave (or free its TMEM) while the other still uses the pair's resources.  The producer and issuer
    // warps ran their loops in one elected lane: reconverge before the warp-aligned cluster barrier.
    __syncwarp();
    cluster_sync_relaxed();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
    }
}
