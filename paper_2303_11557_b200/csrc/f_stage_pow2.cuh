// f_stage_pow2.cuh — F stage for power-of-two frame lengths N = R1 * R2 in {64, 128, 256}: a register-resident
// two-pass FFT in which LANE = INPUT.
//
// One CTA transforms one frame of 32 adjacent inputs.  Thread (warp w, lane L) works on input i0 + L only, so
//   * every shared-memory exchange is [index][lane]: conflict free by construction;
//   * every global store writes 32 adjacent inputs of one (channel, time) row: one full 128-byte line,
//     i.e. the corner turn into Y[p][t][input] costs nothing (PAPER.md L274 did it as a separate pass).
// Pass 1 (in registers): for its residues r (mod R2) the thread computes A_r[k1] = sum_j x[r + R2 j] W_R1^{j k1};
// twiddle W_N^{r k1}; exchange through shared memory; pass 2 (in registers): for its k1 the thread computes
// X[k1 + R1 k2] = sum_r W_R2^{r k2} (W_N^{r k1} A_r[k1]).
// int8 -> fp32 promotion happens in registers with the power-of-two F-stage scale folded in.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>
#include "f_stage.cuh"

namespace mwax {

// exp(-2 pi i m / 32), m = 0..15
__device__ __forceinline__ float2 w32(int m)
{
    switch (m) {
        case 0: return make_float2(1.0f, -0.0f);
        case 1: return make_float2(0.98078528040323043f, -0.19509032201612825f);
        case 2: return make_float2(0.92387953251128674f, -0.38268343236508978f);
        case 3: return make_float2(0.83146961230254524f, -0.55557023301960218f);
        case 4: return make_float2(0.70710678118654757f, -0.70710678118654757f);
        case 5: return make_float2(0.55557023301960229f, -0.83146961230254524f);
        case 6: return make_float2(0.38268343236508984f, -0.92387953251128674f);
        case 7: return make_float2(0.19509032201612833f, -0.98078528040323043f);
        case 8: return make_float2(0.0f, -1.0f);
        case 9: return make_float2(-0.19509032201612820f, -0.98078528040323043f);
        case 10: return make_float2(-0.38268343236508973f, -0.92387953251128674f);
        case 11: return make_float2(-0.55557023301960196f, -0.83146961230254546f);
        case 12: return make_float2(-0.70710678118654746f, -0.70710678118654757f);
        case 13: return make_float2(-0.83146961230254535f, -0.55557023301960218f);
        case 14: return make_float2(-0.92387953251128674f, -0.38268343236508989f);
        default: return make_float2(-0.98078528040323043f, -0.19509032201612861f);
    }
}

// d * exp(-2 pi i m / 32) with the trivial cases folded (m is a compile-time constant after unrolling)
__device__ __forceinline__ float2 mul_w32(float2 d, int m)
{
    if (m == 0) return d;
    if (m == 8) return make_float2(d.y, -d.x);                       // * (-i)
    if (m == 4) {                                                    // * (1 - i)/sqrt(2)
        const float h = 0.70710678118654757f;
        return make_float2((d.x + d.y) * h, (d.y - d.x) * h);
    }
    if (m == 12) {                                                   // * (-1 - i)/sqrt(2)
        const float h = 0.70710678118654757f;
        return make_float2((d.y - d.x) * h, -(d.x + d.y) * h);
    }
    return cmul(d, w32(m));
}

// In-register radix-2 decimation-in-frequency FFT of length M (power of two <= 32), forward.
// Result in BIT-REVERSED order: X[k] is left in x[bitrev_M(k)].
template <int M>
__device__ __forceinline__ void fft_dif(float2 (&x)[M])
{
#pragma unroll
    for (int len = M; len >= 2; len >>= 1) {
#pragma unroll
        for (int blk = 0; blk < M; blk += len) {
#pragma unroll
            for (int i = 0; i < len / 2; ++i) {
                const float2 a = x[blk + i], b = x[blk + i + len / 2];
                x[blk + i] = make_float2(a.x + b.x, a.y + b.y);
                x[blk + i + len / 2] = mul_w32(make_float2(a.x - b.x, a.y - b.y), i * (32 / len));
            }
        }
    }
}

__host__ __device__ constexpr int bitrev(int v, int bits)
{
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((v >> b) & 1) << (bits - 1 - b);
    return r;
}
__host__ __device__ constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

template <int N, int R1, int PTS>
struct FPow2Config {
    static constexpr int R2 = N / R1;
    static constexpr int W = N / PTS;             // warps per CTA
    static constexpr int THREADS = 32 * W;
    static constexpr int RPT = PTS / R1;          // residues per thread in pass 1
    static constexpr int KPT = PTS / R2;          // k1 values per thread in pass 2
    static constexpr int RAW_WORDS = 32 * (N / 2);          // 32 inputs x N samples x 2 bytes
    static constexpr int SMEM_BYTES = RAW_WORDS * 4 + N * 32 * 8;
    static_assert(RPT >= 1 && KPT >= 1 && (RPT == 1 || RPT == 2), "unsupported split");
    static_assert(R1 * R2 == N && W * RPT == R2 && W * KPT == R1, "bad factorisation");
};

template <int N, int R1, int PTS>
__global__ void __launch_bounds__(FPow2Config<N, R1, PTS>::THREADS) f_stage_pow2_kernel(const FParams P)
{
    using C = FPow2Config<N, R1, PTS>;
    constexpr int R2 = C::R2;
    extern __shared__ uint32_t fsm[];
    uint32_t *raw = fsm;                                         // [32 rows][N/2 words], word index XOR lane
    float2 *ex = reinterpret_cast<float2 *>(fsm + C::RAW_WORDS); // [k1][r][lane]

    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i0 = blockIdx.x * 32;
    const int t = blockIdx.y;
    const long long s_off = P.sample0 + (long long)t * N;

    // ---- coalesced 16-byte loads of the 32 rows (2N bytes each), scattered into raw with a per-row XOR swizzle
    constexpr int VPR = N / 8;                                   // 16-byte vectors per row
    for (int v = threadIdx.x; v < 32 * VPR; v += C::THREADS) {
        const int row = v / VPR, c = v % VPR;
        const int i = i0 + row;
        int4 q = make_int4(0, 0, 0, 0);
        if (i < P.n_inputs) {
            const int8_t *src = P.volt + 2 * ((long long)i * P.row_pitch + s_off) + 16 * c;
            if (P.vec_ok) {
                q = __ldg(reinterpret_cast<const int4 *>(src));
            } else {
                const uint16_t *s16 = reinterpret_cast<const uint16_t *>(src);   // samples are 2-byte aligned
                uint32_t ww[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) ww[e] = (uint32_t)s16[2 * e] | ((uint32_t)s16[2 * e + 1] << 16);
                q = make_int4((int)ww[0], (int)ww[1], (int)ww[2], (int)ww[3]);
            }
        }
        uint32_t *dst = raw + row * (N / 2);
        dst[(4 * c + 0) ^ row] = (uint32_t)q.x;
        dst[(4 * c + 1) ^ row] = (uint32_t)q.y;
        dst[(4 * c + 2) ^ row] = (uint32_t)q.z;
        dst[(4 * c + 3) ^ row] = (uint32_t)q.w;
    }
    __syncthreads();

    // ---- pass 1: this thread's residues r = w*RPT + e; points x[r + R2 j], j < R1
    // int8 -> fp32 with the F-stage scale s = 2^-sh folded in (exact): byte b -> ((b ^ 0x80) + 2^23 - (2^23 + 128)) * s
    const float s = P.in_scale;
    const float bias = -8388736.0f * s;
    {
        float2 x[C::RPT][R1];
        const uint32_t *rrow = raw + lane * (N / 2);
#pragma unroll
        for (int j = 0; j < R1; ++j) {
            if (C::RPT == 2) {
                // samples q = 2w + R2 j and q + 1 share one 32-bit word
                const uint32_t word = rrow[(w + (R2 / 2) * j) ^ lane] ^ 0x80808080u;
                x[0][j] = make_float2(fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7440)), s, bias),
                                      fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7441)), s, bias));
                x[C::RPT - 1][j] = make_float2(fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7442)), s, bias),
                                               fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7443)), s, bias));
            } else {
                const int q = w + R2 * j;
                uint32_t word = rrow[(q >> 1) ^ lane] ^ 0x80808080u;
                if (q & 1) word >>= 16;
                x[0][j] = make_float2(fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7440)), s, bias),
                                      fmaf(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7441)), s, bias));
            }
        }
#pragma unroll
        for (int e = 0; e < C::RPT; ++e) {
            fft_dif<R1>(x[e]);
            const int r = w * C::RPT + e;
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) {
                float2 v = x[e][bitrev(k1, ilog2(R1))];
                if (k1 > 0) v = cmul(v, __ldg(&P.tw[r * k1]));           // W_N^{r k1}; warp-uniform address
                ex[(k1 * R2 + r) * 32 + lane] = v;
            }
        }
    }
    __syncthreads();

    // ---- pass 2: this thread's k1 = w*KPT + e; X[k1 + R1 k2] = FFT_R2 over r
    const int i = i0 + lane;
    const int half = P.K / 2;
#pragma unroll
    for (int e = 0; e < C::KPT; ++e) {
        const int k1 = w * C::KPT + e;
        float2 y[R2];
#pragma unroll
        for (int r = 0; r < R2; ++r) y[r] = ex[(k1 * R2 + r) * 32 + lane];
        fft_dif<R2>(y);
        if (i < P.n_inputs) {
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const int k = k1 + R1 * k2;
                const int u = (k < N / 2) ? k : k - N;                   // signed bin
                const int p = u + half;                                  // centre order
                if (p < 0 || p >= P.K) continue;                         // keep the central K channels (L611)
                float2 v = y[bitrev(k2, ilog2(R2))];
                if (P.chan_scale) {
                    const float f = __ldg(&P.sw[p]);                     // sqrt(w_p): shared edge / DC exclusion
                    v.x *= f;
                    v.y *= f;
                }
                P.Y[((long long)p * P.T + t) * P.pitch2 + i] = __floats2half2_rn(v.x, v.y);
            }
        }
    }
}

}  // namespace mwax
