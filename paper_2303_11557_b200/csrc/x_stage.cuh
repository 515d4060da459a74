// x_stage.cuh — X stage: per output channel, the Hermitian contraction V = Y Y^H over (time x contributing fine
// channels), lower triangle only, on tcgen05 tensor cores, with the time integration, the fine-channel
// averaging and the lower-triangle store fused into the epilogue.
//
// PAPER.md §2.1, §2.5.2 L278-282 (cross-multiply every pair incl. autos, accumulate over the integration),
// §2.6 L286-298 (average fine channels); DESIGN.md §5.2.
//
// Complex Gram through ONE real MMA.  A row of Z holds the 2n interleaved reals [re_0, im_0, re_1, im_1, ...]
// of one (channel, time) sample.  G = Z^T Z (2n x 2n real, contraction over rows) contains every product:
//     Re V_ij = G[2i][2j] + G[2i+1][2j+1]        Im V_ij = G[2i+1][2j] - G[2i][2j+1]     (V_ij = sum x_i conj(x_j))
// so the executed real MACs equal the complex-MAC count: no operand duplication, no negated copy.
// Z's layout [row][2n] makes both operands MN-major (the contraction index is the slow axis): TMA (SWIZZLE_128B)
// drops 128-byte x BK-row boxes into shared memory in exactly the canonical MN-major UMMA layout.
//
// Kernel shape: persistent CTAs, 6 warps: warp 0 = TMA producer, warp 1 = MMA issuer (+ TMEM owner),
// warps 2..5 = epilogue (TMEM lanes 32*(warp%4)..+31).  A work item is (output channel c, G-tile (mi, nj)):
// a 128 x BN fp32/int32 accumulator in TMEM, double buffered so the epilogue of one item overlaps the MMAs of
// the next.  Work items are ordered channel-major so concurrently running CTAs share a channel's rows in L2.
#pragma once
#include <cuda_fp16.h>
#include "ptx.cuh"

namespace mwax {

struct XParams {
    int n_inputs;       // n
    int T;              // rows (time samples) per fine channel
    int K;              // fine channels in Z (taps are taken cyclically mod K)
    int n_out;          // C output channels
    int n_tiles;        // lower-triangle G tiles per channel
    const uint8_t *tiles;     // [n_tiles][2] = (mi, nj), device
    const int *tap_start;     // [C] first fine-channel position of output channel c
    int n_taps;               // taps per output channel (fine channels summed into one output)
    const float *scale;       // [C] epilogue scale (float path only)
    void *out;                // float2 / int2 [C][n(n+1)/2]
    long long out_chan_stride;  // n(n+1)/2
};

template <bool kInt8, int BN>
struct XConfig {
    static constexpr int BM = 128;
    static constexpr int ESIZE = kInt8 ? 1 : 2;
    static constexpr int BK = kInt8 ? 128 : 64;          // rows (contraction) per pipeline stage
    static constexpr int KINST = kInt8 ? 32 : 16;        // rows per tcgen05.mma
    static constexpr int CHUNK_ELEMS = 128 / ESIZE;      // MN elements per 128-byte TMA box row
    static constexpr int A_CHUNKS = BM / CHUNK_ELEMS;
    static constexpr int B_CHUNKS = BN / CHUNK_ELEMS;
    static constexpr int CHUNK_BYTES = 128 * BK;         // one TMA box
    static constexpr int A_BYTES = A_CHUNKS * CHUNK_BYTES;
    static constexpr int B_BYTES = B_CHUNKS * CHUNK_BYTES;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int STAGES = (BN == 256) ? 4 : 6;
    static constexpr int ACC_STAGES = 2;
    static constexpr int TMEM_COLS = 512;                // ACC_STAGES * BN <= 512, power of two
    static constexpr int EPI_STAGE_WORDS = 16 * 34;      // per epilogue warp: 16 inputs x (16 complex + pad)
    static constexpr int SMEM_BYTES = 1024 /*align slack*/ + STAGES * STAGE_BYTES + 4 * EPI_STAGE_WORDS * 4 + 256;
    static constexpr uint32_t IDESC = ptx::make_idesc(kInt8 ? 2u : 1u, kInt8 ? 1u : 0u, BM, BN);
    static constexpr int THREADS = 192;
};

template <bool kInt8, int BN>
__global__ void __launch_bounds__(192, 1) x_stage_kernel(const __grid_constant__ CUtensorMap tmap, const XParams P)
{
    using C = XConfig<kInt8, BN>;
    extern __shared__ uint8_t smem_raw[];
    // SWIZZLE_128B atoms need 1024-byte alignment
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *smem_gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t stage_base = smem_base;
    float *epi_stage = reinterpret_cast<float *>(smem_gen + C::STAGES * C::STAGE_BYTES);
    const uint32_t bar_base = smem_base + C::STAGES * C::STAGE_BYTES + 4 * C::EPI_STAGE_WORDS * 4;
    // barriers: full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2]; then the TMEM base address word
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (C::STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * C::STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * C::STAGES + 2 + s); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * C::STAGES + 4);
    volatile uint32_t *tmem_slot_gen =
        reinterpret_cast<volatile uint32_t *>(smem_gen + C::STAGES * C::STAGE_BYTES + 4 * C::EPI_STAGE_WORDS * 4 +
                                              8 * (2 * C::STAGES + 4));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < C::STAGES; ++s) {
            ptx::mbar_init(full_bar(s), 1);
            ptx::mbar_init(empty_bar(s), 1);
        }
        for (int s = 0; s < C::ACC_STAGES; ++s) {
            ptx::mbar_init(tfull_bar(s), 1);
            ptx::mbar_init(tempty_bar(s), 4);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    const int n_items = P.n_out * P.n_tiles;
    const int kb_per_tap = (P.T + C::BK - 1) / C::BK;

    if (warp == 0) {
        // ------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const int c = item / P.n_tiles;
                const int tile = item - c * P.n_tiles;
                const int mi = P.tiles[2 * tile], nj = P.tiles[2 * tile + 1];
                const int p0 = P.tap_start[c];
                for (int tap = 0; tap < P.n_taps; ++tap) {
                    int p = p0 + tap;
                    if (p >= P.K) p -= P.K;
                    for (int kb = 0; kb < kb_per_tap; ++kb) {
                        ptx::mbar_wait(empty_bar(s), ph ^ 1u);
                        ptx::mbar_arrive_expect_tx(full_bar(s), C::STAGE_BYTES);
                        const uint32_t a_dst = stage_base + s * C::STAGE_BYTES;
                        const uint32_t b_dst = a_dst + C::A_BYTES;
#pragma unroll
                        for (int ch = 0; ch < C::A_CHUNKS; ++ch)
                            ptx::tma_load_3d(a_dst + ch * C::CHUNK_BYTES, &tmap, mi * C::BM + ch * C::CHUNK_ELEMS,
                                             kb * C::BK, p, full_bar(s));
#pragma unroll
                        for (int ch = 0; ch < C::B_CHUNKS; ++ch)
                            ptx::tma_load_3d(b_dst + ch * C::CHUNK_BYTES, &tmap, nj * BN + ch * C::CHUNK_ELEMS,
                                             kb * C::BK, p, full_bar(s));
                        if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (one thread)
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            int as = 0;
            uint32_t aph = 0;
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                ptx::mbar_wait(tempty_bar(as), aph ^ 1u);
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
                uint32_t accumulate = 0;
                for (int tap = 0; tap < P.n_taps; ++tap) {
                    for (int kb = 0; kb < kb_per_tap; ++kb) {
                        int rows = P.T - kb * C::BK;
                        if (rows > C::BK) rows = C::BK;
                        const int ksteps = (rows + C::KINST - 1) / C::KINST;   // rows past T are TMA zero fill
                        ptx::mbar_wait(full_bar(s), ph);
                        ptx::tc_fence_after();
                        const uint32_t a_src = stage_base + s * C::STAGE_BYTES;
                        const uint32_t b_src = a_src + C::A_BYTES;
                        for (int ks = 0; ks < ksteps; ++ks) {
                            // KINST rows = KINST/8 swizzle atoms of 1024 B further along the contraction
                            const uint32_t koff = (uint32_t)ks * (C::KINST / 8) * 1024u;
                            const uint64_t a_desc = ptx::make_smem_desc_mn_sw128(a_src + koff, C::CHUNK_BYTES, 1024);
                            const uint64_t b_desc = ptx::make_smem_desc_mn_sw128(b_src + koff, C::CHUNK_BYTES, 1024);
                            if (kInt8) ptx::mma_i8_ss(d_tmem, a_desc, b_desc, C::IDESC, accumulate);
                            else ptx::mma_f16_ss(d_tmem, a_desc, b_desc, C::IDESC, accumulate);
                            accumulate = 1;
                        }
                        ptx::tc_commit(empty_bar(s));   // frees the smem slot when these MMAs have read it
                        if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                    }
                }
                ptx::tc_commit(tfull_bar(as));          // accumulator complete -> epilogue
                if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue (4 warps)
        const int q = warp & 3;                       // TMEM lane quadrant this warp may read
        float *stg = epi_stage + (warp - 2) * C::EPI_STAGE_WORDS;
        int as = 0;
        uint32_t aph = 0;
        const int n = P.n_inputs;
        for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
            const int c = item / P.n_tiles;
            const int tile = item - c * P.n_tiles;
            const int mi = P.tiles[2 * tile], nj = P.tiles[2 * tile + 1];
            const int i_base = mi * (C::BM / 2) + q * 16;       // first input of this warp's 16
            const float sc = kInt8 ? 1.0f : P.scale[c];
            ptx::mbar_wait(tfull_bar(as), aph);
            ptx::tc_fence_after();
            const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * BN);
#pragma unroll 1
            for (int cc = 0; cc < BN / 32; ++cc) {
                const int j0 = nj * (BN / 2) + cc * 16;         // first of this chunk's 16 inputs j
                if (j0 > i_base + 15 || j0 >= n || i_base >= n) continue;   // warp-uniform: nothing below the diagonal
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(t_row + (uint32_t)(cc * 32), r);
                ptx::tmem_ld_wait();
                // even lane (G row 2i): Re = G[2i][2j] + G[2i+1][2j+1]; odd lane (row 2i+1): Im = G[2i+1][2j] - G[2i][2j+1]
#pragma unroll
                for (int jj = 0; jj < 16; ++jj) {
                    const uint32_t other = __shfl_xor_sync(0xffffffffu, r[2 * jj + 1], 1);
                    float v;
                    if (kInt8) {
                        const int a = (int)r[2 * jj], b = (int)other;
                        const int w = (lane & 1) ? (a - b) : (a + b);
                        v = __int_as_float(w);
                    } else {
                        const float a = __uint_as_float(r[2 * jj]), b = __uint_as_float(other);
                        v = ((lane & 1) ? (a - b) : (a + b)) * sc;
                    }
                    stg[(lane >> 1) * 34 + 2 * jj + (lane & 1)] = v;
                }
                __syncwarp();
                // coalesced store: two rows (inputs i) x 16 complex per instruction
                const int jl = lane & 15;
                const int j = j0 + jl;
#pragma unroll
                for (int it = 0; it < 8; ++it) {
                    const int row = 2 * it + (lane >> 4);
                    const int i = i_base + row;
                    float2 v = *reinterpret_cast<const float2 *>(&stg[row * 34 + 2 * jl]);
                    if (i < n && j <= i) {
                        if (i == j) v.y = 0.0f;       // autos: Im := 0 exactly (int path: bit pattern 0 as well)
                        const long long o = (long long)c * P.out_chan_stride + ((long long)i * (i + 1) / 2 + j);
                        reinterpret_cast<float2 *>(P.out)[o] = v;
                    }
                }
                __syncwarp();
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty_bar(as));
            if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, C::TMEM_COLS);
    }
}

}  // namespace mwax
