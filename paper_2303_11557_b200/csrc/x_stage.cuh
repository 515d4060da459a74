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
// This file: the kernel parameters and the epilogue; the kernel itself (CTA pairs, tcgen05 cta_group::2) is in
// x_stage2.cuh.  (Round 1 also kept a single-CTA kernel here as a cross-check of the pair kernel; it was a second
// dispatch target behind an environment switch and is gone: the oracle is the check.)
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
    const uint8_t *tiles;     // [n_tiles][4] = (mi, nj, 0, 0) in units of 128 inputs (256 rows / columns of G), nj <= mi; device
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

}  // namespace mwax
