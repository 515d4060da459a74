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
// This file: the SINGLE-CTA kernel (tcgen05 cta_group::1; selected with MWAX_X_PAIR=0, the cross-check of the CTA-pair
// kernel in x_stage2.cuh, which is the default) and the epilogue both kernels share.
// Kernel shape: persistent CTAs, 6 warps: warp 0 = TMA producer (one lane), warp 1 = MMA issuer (+ TMEM owner; all
// lanes run the loops, one elected lane issues), warps 2..5 = epilogue (TMEM lanes 32*(warp%4)..+31).  A work item is
// (output channel c, G-tile): a 128 x 256 (128 x 128 on the diagonal) fp32/int32 accumulator in TMEM, double buffered
// so the epilogue of one item overlaps the MMAs of the next.  Work items are ordered channel-major so concurrently
// running CTAs share a channel's rows in L2.
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
    const uint8_t *tiles;     // [n_tiles][4] = (mi, nj, w, 0): G rows 128 mi.., G columns 128 nj.. of width 128 w; device
    const int *tap_start;     // [C] first fine-channel position of output channel c
    int n_taps;               // taps per output channel (fine channels summed into one output)
    const float *scale;       // [C] epilogue scale (float path only)
    void *out;                // float2 / int2 [C][n(n+1)/2]
    long long out_chan_stride;  // n(n+1)/2
    int accumulate;             // float path: add to what `out` already holds (integration across calls) instead of overwriting
    int edge_runs;              // pair kernel, even F, centre-symmetric averaging: > 0 = shared-edge schedule with this many
                                // runs of adjacent output channels per tile (x_stage2.cuh); 0 = every channel on its own
};

// Shared-edge schedule: with even F the outermost fine channel of an output channel is shared, at half
// weight, with its neighbour.  Instead of contracting it twice, a CTA pair walks a RUN of adjacent
// output channels of one tile and keeps a running sum S per accumulator element in shared memory (thread private):
//   INIT  edge tap below the run's first channel:        S  = e
//   ADD   the F - 1 interior taps of channel c:          S += m
//   OUT   the edge tap above channel c:                  V[c] = scale_c (S + e),  S = e   (it is also c + 1's lower edge)
enum { X_EDGE_NONE = 0, X_EDGE_INIT = 1, X_EDGE_ADD = 2, X_EDGE_OUT = 3 };

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

// Epilogue of one accumulator tile, run by one warp on its 32 TMEM lanes (G rows 2 i, 2 i + 1 of 16 inputs i from
// i_base) and `ncc` chunks of 32 G columns (16 inputs j from j_base + 16 cc): tcgen05.ld, the 2 x 2 real -> complex
// fold, scale, Im(auto) := 0, triangle mask, and stores staged through padded shared memory so that
// each instruction writes 16 consecutive baselines of two rows.  `stg` = this warp's EPI_STAGE_WORDS floats.
template <bool kInt8, bool kEdge = false>
__device__ __forceinline__ void x_epilogue_tile(const XParams &P, float *stg, uint32_t t_row, int c, int i_base, int j_base,
                                                int ncc, float sc, int lane, int mode = X_EDGE_NONE, float *S = nullptr)
{
    const int n = P.n_inputs;
#pragma unroll 1
    for (int cc = 0; cc < ncc; ++cc) {
        const int j0 = j_base + cc * 16;         // first of this chunk's 16 inputs j
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
                float w = (lane & 1) ? (a - b) : (a + b);
                if (kEdge) {                      // running sum over the run's taps: S[chunk][jj][lane], this warp's slice
                    float *sp = S + (cc * 16 + jj) * 32 + lane;
                    if (mode == X_EDGE_INIT) {
                        *sp = w;
                    } else if (mode == X_EDGE_ADD) {
                        *sp += w;
                    } else {
                        const float sum = *sp + w;
                        *sp = w;
                        w = sum;
                    }
                }
                v = w * sc;
            }
            if (!kEdge || mode == X_EDGE_OUT) stg[(lane >> 1) * 34 + 2 * jj + (lane & 1)] = v;
        }
        if (kEdge && mode != X_EDGE_OUT) continue;   // warp-uniform: nothing to store yet
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
                if (!kInt8 && P.accumulate) {
                    const float2 old = reinterpret_cast<const float2 *>(P.out)[o];
                    v.x += old.x;
                    v.y += old.y;
                }
                reinterpret_cast<float2 *>(P.out)[o] = v;
            }
        }
        __syncwarp();
    }
}

template <bool kInt8, int BN>
__global__ void __launch_bounds__(192, 1) x_stage_kernel(const __grid_constant__ CUtensorMap tmap,
                                                         const __grid_constant__ CUtensorMap tmap_flat, const XParams P)
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
        ptx::prefetch_tensormap(&tmap_flat);
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

    // K-loop schedule of one work item (identical in the producer and the MMA issuer).  The taps of an output
    // channel are adjacent channel positions, i.e. ADJACENT ROWS of Y[p][t]: when T >= BK the contraction runs over
    // the flattened rows (p T + t) in whole BK-row blocks through `tmap_flat`, so only the END of a run is a partial
    // block (C4: 51 taps x 200 rows = 159 blocks + 24 rows instead of 51 x (3 blocks + 8 rows)).  The partial block is
    // fetched through the per-channel map, whose rows past T read as zero.  A tap window that wraps past K (cyclic
    // taps, Q8) is two runs.
    const bool flat = (P.n_taps > 1) && (P.T >= C::BK);

    if (warp == 0) {
        // ------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            auto load_block = [&](const CUtensorMap *m, int mi, int nj, int bch, int row, int chan) {
                ptx::mbar_wait(empty_bar(s), ph ^ 1u);
                ptx::mbar_arrive_expect_tx(full_bar(s), (uint32_t)(C::A_BYTES + bch * C::CHUNK_BYTES));
                const uint32_t a_dst = stage_base + s * C::STAGE_BYTES;
                const uint32_t b_dst = a_dst + C::A_BYTES;
#pragma unroll
                for (int ch = 0; ch < C::A_CHUNKS; ++ch)
                    ptx::tma_load_3d(a_dst + ch * C::CHUNK_BYTES, m, mi * C::BM + ch * C::CHUNK_ELEMS, row, chan, full_bar(s));
                for (int ch = 0; ch < bch; ++ch)
                    ptx::tma_load_3d(b_dst + ch * C::CHUNK_BYTES, m, nj * 128 + ch * C::CHUNK_ELEMS, row, chan, full_bar(s));
                if (++s == C::STAGES) { s = 0; ph ^= 1u; }
            };
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const int c = item / P.n_tiles;
                const int tile = item - c * P.n_tiles;
                const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1];
                const int bch = P.tiles[4 * tile + 2] * (128 / C::CHUNK_ELEMS);   // 128-byte B chunks of this tile
                const int p0 = P.tap_start[c];
                if (flat) {
                    const int n1 = min(P.n_taps, P.K - p0);
                    for (int run = 0; run < 2; ++run) {
                        const int pf = run ? 0 : p0, nt = run ? P.n_taps - n1 : n1;
                        if (nt <= 0) continue;
                        const int rows = nt * P.T, nfull = rows / C::BK, tail = rows - nfull * C::BK;
                        for (int q = 0; q < nfull; ++q) load_block(&tmap_flat, mi, nj, bch, pf * P.T + q * C::BK, 0);
                        if (tail) load_block(&tmap, mi, nj, bch, P.T - tail, pf + nt - 1);
                    }
                } else {
                    for (int tap = 0; tap < P.n_taps; ++tap) {
                        int p = p0 + tap;
                        if (p >= P.K) p -= P.K;
                        for (int kb = 0; kb < kb_per_tap; ++kb) load_block(&tmap, mi, nj, bch, kb * C::BK, p);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (the whole warp runs the loops so
        // that every operand is warp-uniform, one elected lane issues: see ptx::elect_one)
        {
            int s = 0;
            uint32_t ph = 0;
            int as = 0;
            uint32_t aph = 0;
            uint32_t d_tmem = 0, idesc = 0, accumulate = 0;
            auto mma_block = [&](int rows) {
                ptx::mbar_wait(full_bar(s), ph);
                ptx::tc_fence_after();
                const uint32_t a_src = stage_base + s * C::STAGE_BYTES;
                if (ptx::elect_one()) {
                    ptx::mma_block_issue<kInt8, false, C::BK, C::KINST>(a_src, a_src + C::A_BYTES, C::CHUNK_BYTES, d_tmem, idesc, rows,
                                                                         accumulate);
                    ptx::tc_commit(empty_bar(s));       // frees the smem slot when these MMAs have read it
                }
                __syncwarp();
                accumulate = 1;
                if (++s == C::STAGES) { s = 0; ph ^= 1u; }
            };
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const int c = item / P.n_tiles;
                const int tile = item - c * P.n_tiles;
                ptx::mbar_wait(tempty_bar(as), aph ^ 1u);
                ptx::tc_fence_after();
                d_tmem = tmem_base + (uint32_t)(as * BN);
                idesc = ptx::make_idesc(kInt8 ? 2u : 1u, kInt8 ? 1u : 0u, C::BM, 128u * P.tiles[4 * tile + 2]);
                accumulate = 0;
                if (flat) {
                    const int p0 = P.tap_start[c];
                    const int n1 = min(P.n_taps, P.K - p0);
                    for (int run = 0; run < 2; ++run) {
                        const int nt = run ? P.n_taps - n1 : n1;
                        if (nt <= 0) continue;
                        const int rows = nt * P.T, nfull = rows / C::BK, tail = rows - nfull * C::BK;
                        for (int q = 0; q < nfull; ++q) mma_block(C::BK);
                        if (tail) mma_block(tail);
                    }
                } else {
                    for (int tap = 0; tap < P.n_taps; ++tap)
                        for (int kb = 0; kb < kb_per_tap; ++kb) mma_block(min(C::BK, P.T - kb * C::BK));
                }
                if (ptx::elect_one()) ptx::tc_commit(tfull_bar(as));          // accumulator complete -> epilogue
                __syncwarp();
                if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue (4 warps)
        const int q = warp & 3;                       // TMEM lane quadrant this warp may read
        float *stg = epi_stage + (warp - 2) * C::EPI_STAGE_WORDS;
        int as = 0;
        uint32_t aph = 0;
        for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
            const int c = item / P.n_tiles;
            const int tile = item - c * P.n_tiles;
            const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1], ncc = 4 * P.tiles[4 * tile + 2];
            const int i_base = mi * (C::BM / 2) + q * 16;       // first input of this warp's 16
            const float sc = kInt8 ? 1.0f : P.scale[c];
            ptx::mbar_wait(tfull_bar(as), aph);
            ptx::tc_fence_after();
            const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * BN);
            x_epilogue_tile<kInt8>(P, stg, t_row, c, i_base, nj * 64, ncc, sc, lane);
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
