// set_builtin.cu -- table of the built-in stage kernels and the descriptor constructors for the five pipelines
// of BASELINE.json:configs[0..4] (include/set.h "Built-in stage kernels").  Host code only; the kernels live in
// csrc/kernels/.
#include <cstring>

#include "../../include/set.h"
#include "kernels/kernels.h"

extern "C" __global__ void set_k_gemm_bias_gelu_bf16(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                                                     const __grid_constant__ CUtensorMap tmC, const float* bias, uint32_t M, uint32_t N,
                                                     uint32_t K);
extern "C" uint32_t set_gemm_smem_bytes(void);
extern "C" uint32_t set_gemm_threads(void);

namespace {

set_size_expr fixed(uint64_t v) { return set_size_expr{v, 0, 0, 0}; }
set_size_expr scaled(uint64_t per_unit, uint32_t mask) { return set_size_expr{0, per_unit, mask, 0}; }

set_arg_desc arg_buf(int idx, set_size_expr off = set_size_expr{0, 0, 0, 0}) {
    set_arg_desc a{};
    a.kind = SET_ARG_BUFFER;
    a.index = idx;
    a.offset = off;
    return a;
}
set_arg_desc arg_u32(uint32_t v) {
    set_arg_desc a{};
    a.kind = SET_ARG_IMM32;
    a.imm = v;
    return a;
}
set_arg_desc arg_cond() {
    set_arg_desc a{};
    a.kind = SET_ARG_COND;
    return a;
}
set_arg_desc arg_dim(int i) {
    set_arg_desc a{};
    a.kind = SET_ARG_DIM;
    a.index = i;
    return a;
}
set_arg_desc arg_tmap(int idx, uint64_t off, uint32_t elem, uint64_t inner, uint64_t outer, uint32_t box_in, uint32_t box_out,
                      uint32_t swizzle = SET_SWIZZLE_128B) {
    set_arg_desc a{};
    a.kind = SET_ARG_TMAP2D;
    a.index = idx;
    a.offset = fixed(off);
    a.tmap.elem_bytes = elem;
    a.tmap.swizzle = swizzle;
    a.tmap.inner = inner;
    a.tmap.outer = outer;
    a.tmap.pitch_bytes = inner * elem;
    a.tmap.box_inner = box_in;
    a.tmap.box_outer = box_out;
    return a;
}

set_stage_desc stage(int kernel_id, set_grid_rule gx, set_grid_rule gy, uint32_t bx, uint32_t by, uint32_t smem,
                     std::initializer_list<set_arg_desc> args) {
    set_stage_desc s{};
    s.func = set_builtin_kernel(kernel_id);
    s.grid[0] = gx;
    s.grid[1] = gy;
    s.grid[2] = set_grid_rule{fixed(1), 1, 0};
    s.block[0] = bx;
    s.block[1] = by;
    s.block[2] = 1;
    s.smem_bytes = smem;
    s.num_args = 0;
    for (auto& a : args) s.args[s.num_args++] = a;
    return s;
}
set_grid_rule grid_fixed(uint32_t v) { return set_grid_rule{fixed(v), 1, 0}; }
set_grid_rule grid_div(set_size_expr e, uint32_t d) { return set_grid_rule{e, d, 0}; }

set_buffer_desc buffer(uint64_t bytes) {
    set_buffer_desc b{};
    b.bytes = bytes;
    return b;
}

}  // namespace

extern "C" const void* set_builtin_kernel(int id) {
    switch (id) {
        case SET_K_SCAN_I32: return (const void*)set_k_scan_i32;
        case SET_K_HIST_MOD64: return (const void*)set_k_hist_mod64;
        case SET_K_AFFINE_F32: return (const void*)set_k_affine_f32;
        case SET_K_ADD_BIAS_F32: return (const void*)set_k_add_bias_f32;
        case SET_K_RELU_F32: return (const void*)set_k_relu_f32;
        case SET_K_SQUARE_F32: return (const void*)set_k_square_f32;
        case SET_K_BLOCK_SUM_F32: return (const void*)set_k_block_sum_f32;
        case SET_K_JACOBI5_F32: return (const void*)set_k_jacobi5_f32;
        case SET_K_GEMM_BIAS_GELU: return (const void*)set_k_gemm_bias_gelu_bf16;
        case SET_K_RGB2GRAY_U8: return (const void*)set_k_rgb2gray_u8;
        case SET_K_BLUR3X3_U8: return (const void*)set_k_blur3x3_u8;
        case SET_K_HIST256_U8: return (const void*)set_k_hist256_u8;
        case SET_K_SPIN: return (const void*)set_k_spin;
        case SET_K_SIGNAL: return (const void*)set_k_signal;
        case SET_K_COPY: return (const void*)set_k_copy;
        case SET_K_COPY_OUT: return (const void*)set_k_copy_out;
        case SET_K_STAMP: return (const void*)set_k_stamp;
        case SET_K_SOBEL3X3_U8: return (const void*)set_k_sobel3x3_u8;
        case SET_K_MEAN3X3_U8: return (const void*)set_k_mean3x3_u8;
        case SET_K_THRESHOLD_U8: return (const void*)set_k_threshold_u8;
        case SET_K_BLEND_U8: return (const void*)set_k_blend_u8;
        case SET_K_SSSP_INIT: return (const void*)set_k_sssp_init;
        case SET_K_SSSP_RELAX: return (const void*)set_k_sssp_relax;
        case SET_K_SSSP_CONTROL: return (const void*)set_k_sssp_control;
        case SET_K_SSSP_SOLO: return (const void*)set_k_sssp_solo;
        default: return nullptr;
    }
}

extern "C" set_status set_builtin_pipeline(int config, int variant, const uint32_t* params, int num_params, set_stage_desc* st,
                                           int* num_stages, set_buffer_desc* bf, int* num_bufs, uint64_t* host_in_bytes,
                                           uint64_t* host_out_bytes) {
    if (!st || !bf || !num_stages || !num_bufs || num_params < 0 || (num_params > 0 && !params)) return SET_ERR_INVALID;
    auto P = [&](int i, uint32_t dflt) { return i < num_params ? params[i] : dflt; };
    const bool with_spin = (variant & 0x100) != 0;
    variant &= 0xff;
    int ns = 0, nb = 0;
    uint64_t in_bytes = 0, out_bytes = 0;
    switch (config) {
        case 0: {  // scan -> hist64 -> D2H [scan][hist]   (BASELINE.json:configs[0]; readings C0-1, C0-2)
            uint32_t n = P(0, 4096);
            if (n == 0) return SET_ERR_INVALID;
            in_bytes = 4ull * n;
            out_bytes = 4ull * n + 256;
            bf[0] = buffer(in_bytes);
            bf[0].h2d_bytes = fixed(in_bytes);
            bf[1] = buffer(out_bytes);
            bf[1].d2h_bytes = fixed(out_bytes);
            nb = 2;
            st[ns++] = stage(SET_K_SCAN_I32, grid_fixed(1), grid_fixed(1), 1024, 1, 0, {arg_buf(0), arg_buf(1), arg_u32(n)});
            st[ns++] = stage(SET_K_HIST_MOD64, grid_fixed(1), grid_fixed(1), 256, 1, 0,
                             {variant == 1 ? arg_buf(0) : arg_buf(1), arg_buf(1, fixed(4ull * n)), arg_u32(n)});
            break;
        }
        case 1: {  // affine -> add bias -> relu -> square -> block sum   (configs[1]; readings C1-1..C1-5)
            uint32_t n = P(0, 16384);
            if (n == 0) return SET_ERR_INVALID;
            in_bytes = 8ull * n;  // [x][bias]
            out_bytes = 4;
            bf[0] = buffer(in_bytes);
            bf[0].h2d_bytes = fixed(in_bytes);
            bf[1] = buffer(4ull * n);
            bf[2] = buffer(256);
            bf[2].d2h_bytes = fixed(4);
            nb = 3;
            set_grid_rule g = grid_fixed((n + 1023) / 1024);
            st[ns++] = stage(SET_K_AFFINE_F32, g, grid_fixed(1), 256, 1, 0, {arg_buf(0), arg_buf(1), arg_u32(n)});
            st[ns++] = stage(SET_K_ADD_BIAS_F32, g, grid_fixed(1), 256, 1, 0, {arg_buf(1), arg_buf(0, fixed(4ull * n)), arg_u32(n)});
            st[ns++] = stage(SET_K_RELU_F32, g, grid_fixed(1), 256, 1, 0, {arg_buf(1), arg_u32(n)});
            st[ns++] = stage(SET_K_SQUARE_F32, g, grid_fixed(1), 256, 1, 0, {arg_buf(1), arg_u32(n)});
            st[ns++] = stage(SET_K_BLOCK_SUM_F32, grid_fixed(1), grid_fixed(1), 1024, 1, 0, {arg_buf(1), arg_buf(2), arg_u32(n)});
            break;
        }
        case 2: {  // `sweeps` Jacobi sweeps, ping-pong between buffers 0 and 1   (configs[2]; readings C2-1..C2-3)
            uint32_t h = P(0, 4096), w = P(1, 4096), sweeps = P(2, 10), alternate = P(3, 1);
            if (h == 0 || w == 0 || sweeps == 0) return SET_ERR_INVALID;
            in_bytes = out_bytes = 4ull * h * w;
            bf[0] = buffer(in_bytes);
            bf[0].h2d_bytes = fixed(in_bytes);
            bf[1] = buffer(in_bytes);
            nb = 2;
            int cur = 0;
            uint32_t left = sweeps;
            while (left > 0) {
                if (ns >= SET_MAX_STAGES) return SET_ERR_INVALID;
                {
                    st[ns++] = stage(SET_K_JACOBI5_F32, grid_fixed((w + kJacobiCols - 1) / kJacobiCols),
                                     grid_fixed((h + kJacobiRows - 1) / kJacobiRows), 256, 1, 0,
                                     {arg_buf(cur), arg_buf(cur ^ 1), arg_u32(h), arg_u32(w), arg_u32(alternate ? (sweeps - left) & 1u : 0u)});
                    left -= 1;
                }
                cur ^= 1;
            }
            bf[cur].d2h_bytes = fixed(out_bytes);
            break;
        }
        case 3: {  // C = bf16(GELU(A.B + bias)), tcgen05   (configs[3]; readings C3-1..C3-4)
            uint32_t M = P(0, 2048), N = P(1, 2048), K = P(2, 2048);
            if (M == 0 || N == 0 || K == 0 || (N % 8) || (K % 8)) return SET_ERR_INVALID;  // TMA needs 16-byte row pitches
            uint64_t a_bytes = 2ull * M * K, b_bytes = 2ull * K * N;
            in_bytes = a_bytes + b_bytes + 4ull * N;  // [A][B][bias]
            out_bytes = 2ull * M * N;
            bf[0] = buffer(in_bytes);
            bf[0].h2d_bytes = fixed(in_bytes);
            bf[1] = buffer(out_bytes);
            bf[1].d2h_bytes = fixed(out_bytes);
            nb = 2;
            // A: row-major MxK, box = 64 K-elements (128 B) x 128 rows.  B: row-major KxN, box = 64 N-elements x 64 K-rows.
            // C: row-major MxN, store box = 32 N-elements x 32 rows (half of one epilogue warp's piece), 64-byte swizzle.
            // grid: CTA pairs (cluster 2 x 1 x 1) along x, one pair per 256 x 256 tile -- gemm_sm100.cu
            st[ns++] = stage(SET_K_GEMM_BIAS_GELU, grid_fixed(2 * ((M + 255) / 256)), grid_fixed((N + 255) / 256), set_gemm_threads(), 1, set_gemm_smem_bytes(),
                             {arg_tmap(0, 0, 2, K, M, 64, 128), arg_tmap(0, a_bytes, 2, N, K, 64, 64), arg_tmap(1, 0, 2, N, M, 32, 32, SET_SWIZZLE_64B),
                              arg_buf(0, fixed(a_bytes + b_bytes)), arg_u32(M), arg_u32(N), arg_u32(K)});
            break;
        }
        case 4: {  // gray -> blur -> hist256; dims = {w, h}   (configs[4]; readings C4-1..C4-4)
            uint32_t mw = P(0, 1920), mh = P(1, 1080);
            if (mw == 0 || mh == 0) return SET_ERR_INVALID;
            uint64_t maxpix = (uint64_t)mw * mh;
            in_bytes = 3 * maxpix;
            out_bytes = maxpix + 1024;
            const uint32_t WH = 0x3;  // dims[0]*dims[1]
            bf[0] = buffer(3 * maxpix);
            bf[0].h2d_bytes = scaled(3, WH);
            bf[1] = buffer(maxpix);  // gray
            bf[2] = buffer(maxpix);  // blurred
            bf[2].d2h_bytes = scaled(1, WH);
            bf[3] = buffer(1024);  // histogram, zeroed at the start of every job
            bf[3].flags = SET_BUF_ZERO;
            bf[3].zero_bytes = fixed(1024);
            bf[3].d2h_bytes = fixed(1024);
            bf[3].d2h_host_off = scaled(1, WH);  // host image = [blur w*h][hist 1024]  (reading C4-3)
            nb = 4;
            st[ns++] = stage(SET_K_RGB2GRAY_U8, grid_div(scaled(1, WH), kGrayPixPerBlock), grid_fixed(1), 256, 1, 0,
                             {arg_buf(0), arg_buf(1), arg_dim(0), arg_dim(1)});
            st[ns++] = stage(SET_K_BLUR3X3_U8, grid_div(scaled(1, 0x1), kBlurTileW), grid_div(scaled(1, 0x2), kBlurTileH), 32, 4, 0,
                             {arg_buf(1), arg_buf(2), arg_dim(0), arg_dim(1)});
            st[ns++] = stage(SET_K_HIST256_U8, grid_div(scaled(1, WH), kHistPixPerBlock), grid_fixed(1), 256, 1, 0,
                             {arg_buf(2), arg_buf(3), arg_dim(0), arg_dim(1)});
            break;
        }
        case 5: {  // SSSP by frontier Bellman-Ford: init -> WHILE { relax x U -> control }   (readings S5-1..S5-4)
            uint32_t maxv = P(0, 4096), maxe = P(1, 15 * 4096), unroll = P(2, 4);  // U relaxations per pass of the loop (paper_kernels.cu)
            if (maxv == 0 || maxe == 0 || unroll < 2 || unroll > 8) return SET_ERR_INVALID;  // U = 1 is a two-node body: set_register_pipeline refuses it
            const uint64_t head = 16ull + 4ull * (maxv + 1);  // [V, E, src, 0][row_ptr]; then col and w, 8 bytes per edge
            in_bytes = head + 8ull * maxe;
            out_bytes = 4ull * maxv + 16;                      // [dist][rounds, 0, 0, 0]
            bf[0] = buffer(in_bytes);
            bf[0].h2d_bytes = set_size_expr{head, 8, 0x1, 0};  // dims[0] = E of the job
            bf[1] = buffer(out_bytes);
            bf[1].d2h_bytes = fixed(out_bytes);
            bf[2] = buffer(8ull * maxv + 64);                  // frontier flags [2][maxV], ctrl[16]
            nb = 3;
            if (variant == 1) {  // the whole job in one kernel of one block: no WHILE node (K25)
                if (maxv > kSsspSoloMaxV) return SET_ERR_INVALID;  // the distances must fit one SM's shared memory
                st[ns++] = stage(SET_K_SSSP_SOLO, grid_fixed(1), grid_fixed(1), kSsspSoloThreads, 1, set_sssp_solo_smem_bytes(maxv),
                                 {arg_buf(0), arg_buf(1), arg_buf(2), arg_u32(maxv)});
                break;
            }
            const set_grid_rule g = grid_fixed((maxv + 255) / 256);
            st[ns++] = stage(SET_K_SSSP_INIT, g, grid_fixed(1), 256, 1, 0, {arg_buf(0), arg_buf(1), arg_buf(2), arg_u32(maxv)});
            for (uint32_t sub = 0; sub < unroll; ++sub) {
                st[ns] = stage(SET_K_SSSP_RELAX, grid_fixed((uint32_t)(((uint64_t)maxv * kSsspLanes + 255) / 256)), grid_fixed(1), 256, 1, 0,
                               {arg_buf(0), arg_buf(1), arg_buf(2), arg_u32(maxv), arg_u32(sub)});
                st[ns++].flags = sub == 0 ? SET_STAGE_LOOP_BEGIN : 0u;
            }
            st[ns] = stage(SET_K_SSSP_CONTROL, grid_fixed(1), grid_fixed(1), 1, 1, 0,
                           {arg_buf(0), arg_buf(1), arg_buf(2), arg_u32(maxv), arg_u32(unroll), arg_cond()});
            st[ns++].flags = SET_STAGE_LOOP_END;
            break;
        }
        case 6: {  // Sobel chain: gray -> sobel -> mean3x3 -> threshold -> blend; dims = {w, h}   (readings S6-1..S6-6)
            uint32_t mw = P(0, 1920), mh = P(1, 1080), thresh = P(2, 64);
            if (mw == 0 || mh == 0) return SET_ERR_INVALID;
            uint64_t maxpix = (uint64_t)mw * mh;
            in_bytes = 3 * maxpix;
            out_bytes = maxpix;
            const uint32_t WH = 0x3;  // dims[0]*dims[1]
            bf[0] = buffer(3 * maxpix);
            bf[0].h2d_bytes = scaled(3, WH);
            bf[1] = buffer(maxpix);  // n: normalised intensity, kept for the blend
            bf[2] = buffer(maxpix);  // ping
            bf[3] = buffer(maxpix);  // pong; the blended output ends here
            bf[3].d2h_bytes = scaled(1, WH);
            nb = 4;
            const set_grid_rule gx = grid_div(scaled(1, 0x1), kBlurTileW), gy = grid_div(scaled(1, 0x2), kBlurTileH);  // K11's tile
            const set_grid_rule gp = grid_div(scaled(1, WH), kBytePixPerBlock);
            st[ns++] = stage(SET_K_RGB2GRAY_U8, grid_div(scaled(1, WH), kGrayPixPerBlock), grid_fixed(1), 256, 1, 0,
                             {arg_buf(0), arg_buf(1), arg_dim(0), arg_dim(1)});
            st[ns++] = stage(SET_K_SOBEL3X3_U8, gx, gy, 32, 4, 0, {arg_buf(1), arg_buf(2), arg_dim(0), arg_dim(1)});
            st[ns++] = stage(SET_K_MEAN3X3_U8, gx, gy, 32, 4, 0, {arg_buf(2), arg_buf(3), arg_dim(0), arg_dim(1)});
            st[ns++] = stage(SET_K_THRESHOLD_U8, gp, grid_fixed(1), 256, 1, 0, {arg_buf(3), arg_buf(2), arg_dim(0), arg_dim(1), arg_u32(thresh)});
            st[ns++] = stage(SET_K_BLEND_U8, gp, grid_fixed(1), 256, 1, 0, {arg_buf(2), arg_buf(1), arg_buf(3), arg_dim(0), arg_dim(1)});
            break;
        }
        default:
            return SET_ERR_INVALID;
    }
    if (with_spin) {  // debug delay stage: busy-waits dims[3] nanoseconds (reorders completions)
        if (ns >= SET_MAX_STAGES || nb >= SET_MAX_BUFFERS) return SET_ERR_INVALID;
        bf[nb] = buffer(256);
        st[ns++] = stage(SET_K_SPIN, grid_fixed(1), grid_fixed(1), 1, 1, 0, {arg_buf(nb), arg_dim(3)});
        nb++;
    }
    for (int i = 0; i < ns; ++i)
        if (!st[i].func) return SET_ERR_INVALID;
    *num_stages = ns;
    *num_bufs = nb;
    if (host_in_bytes) *host_in_bytes = in_bytes;
    if (host_out_bytes) *host_out_bytes = out_bytes;
    return SET_OK;
}
