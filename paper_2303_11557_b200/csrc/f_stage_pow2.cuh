// f_stage_pow2.cuh — F stage for power-of-two frame lengths N = R1 * R2 in {64, 128, 256, 512}: a register-resident
// two-pass FFT in which LANE = INPUT.
//
// One CTA owns 32 adjacent inputs and walks over a run of consecutive frames.  Thread (warp w, lane L) works on
// input i0 + L only, so
//   * every shared-memory exchange is [index][lane]: conflict free by construction;
//   * every global store writes 32 adjacent inputs of one (channel, time) row: one full 128-byte line,
//     i.e. the corner turn into Y[p][t][input] costs nothing (PAPER.md L274 did it as a separate pass).
// Pass 1 (in registers): for its residues r (mod R2) the thread computes A_r[k1] = sum_j x[r + R2 j] W_R1^{j k1};
// twiddle W_N^{r k1}; exchange through shared memory; pass 2 (in registers): for its k1 the thread computes
// X[k1 + R1 k2] = sum_r W_R2^{r k2} (W_N^{r k1} A_r[k1]).
// int8 -> fp32 promotion happens in registers with the power-of-two F-stage scale folded in.
//
// The kernel is co-limited by the issue slots, the L1 data pipe and the FMA pipe (ncu: profiles/r2_ncu_full.md), so everything that is not butterfly
// arithmetic is hoisted out of the frame loop: row pointers, the swizzle-free padded raw tile (row stride N/2+1
// words -> bank = row + word), inter-pass twiddles and per-position factors read from the kernel-parameter constant bank, and store addresses
// formed as base + k2 * stride with compile-time k2.  The raw bytes of frame t+1 are fetched into registers while
// frame t is being transformed.
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
                const int m = i * (32 / len);
                x[blk + i] = cadd(a, b);
                // m = 8 (times -i) swaps the halves: scalar subtractions write them where they are wanted
                x[blk + i + len / 2] = (m == 8) ? make_float2(a.y - b.y, b.x - a.x) : mul_w32(csub(a, b), m);
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
    static constexpr int MIN_CTAS = (N == 128) ? 4 : 0;   // N = 128: hold the kernel to 64 registers (four CTAs per SM); 0 = no constraint
    static constexpr int RPT = PTS / R1;          // residues per thread in pass 1
    static constexpr int KPT = PTS / R2;          // k1 values per thread in pass 2
    static constexpr int ROW_WORDS = N / 2 + 1;   // padded raw row: bank(row, word) = row + word (mod 32)
    static constexpr int RAW_WORDS = 32 * ROW_WORDS;
    static constexpr int EX_OFF_WORDS = ((RAW_WORDS + 3) / 4) * 4;
    static constexpr int SMEM_BYTES = (EX_OFF_WORDS + N * 32 * 2) * 4;   // raw tile + fp32 exchange buffer
    static constexpr int VPT = (32 * (N / 8)) / THREADS;   // 16-byte raw vectors per thread per frame
    static_assert(RPT >= 1 && KPT >= 1 && (RPT == 1 || RPT == 2), "unsupported split");
    static_assert(R1 * R2 == N && W * RPT == R2 && W * KPT == R1, "bad factorisation");
    static_assert(VPT * THREADS == 32 * (N / 8) && THREADS % 8 == 0, "raw tile must divide evenly over the threads");
    static_assert(R1 % 4 == 0, "twiddle rows are read as 16-byte pairs");
};

// FULL : K == N (every bin is kept; no range checks)          SCALE : multiply by sw[p] (averaging weights)
// DELAY: fractional-delay / phase gain per (input, frame) (PAPER.md 2.5.1 L266-272)
template <int N, int R1, int PTS, bool FULL, bool SCALE, bool DELAY = false>
__global__ void __launch_bounds__(FPow2Config<N, R1, PTS>::THREADS, FPow2Config<N, R1, PTS>::MIN_CTAS) f_stage_pow2_kernel(const FParams P)
{
    using C = FPow2Config<N, R1, PTS>;
    constexpr int R2 = C::R2;
    extern __shared__ __align__(16) uint32_t fsm[];
    uint32_t *raw = fsm;                                              // [32 rows][ROW_WORDS]
    float2 *ex = reinterpret_cast<float2 *>(fsm + C::EX_OFF_WORDS);  // [k1][r][lane]
    // inter-pass twiddles W_N^{r k1} and per-position factors sqrt(w_p): constant-bank tables in the kernel parameters (FParams)

    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i0 = blockIdx.x * 32;
    const int t_begin = blockIdx.y * P.frames_per_cta;
    const int t_end = min(P.T, t_begin + P.frames_per_cta);

    // ---- per-CTA setup: row pointers
    const int8_t *src[C::VPT];
    uint32_t *rdst[C::VPT];
    bool rok[C::VPT];
#pragma unroll
    for (int v = 0; v < C::VPT; ++v) {
        // a warp covers 4 rows x 8 vectors (128 contiguous bytes of each row): its four 32-bit stores of a stash go to the
        // words row * ROW_WORDS + 4 c + k = row + 4 c + k (mod 32), all 32 banks once (2 rows x 16 vectors had c and c + 8
        // collide: 8.7 M conflict wavefronts per C3 launch on the kernel's busiest unit, the L1 data pipe)
        const int idx = threadIdx.x + v * C::THREADS;
        const int row = (idx >> 3) & 31, c = ((idx >> 3) >> 5) * 8 + (idx & 7);
        rok[v] = (i0 + row) < P.n_inputs;
        src[v] = P.volt + 2 * ((long long)(rok[v] ? i0 + row : 0) * P.row_pitch + P.sample0) + 16 * c;
        rdst[v] = raw + row * C::ROW_WORDS + 4 * c;
    }
    auto fetch = [&](int t, int4 (&q)[C::VPT]) {
#pragma unroll
        for (int v = 0; v < C::VPT; ++v) {
            q[v] = make_int4(0, 0, 0, 0);
            if (rok[v]) {
                const int8_t *s = src[v] + 2ll * t * N;
                q[v] = __ldg(reinterpret_cast<const int4 *>(s));   // rows are 16-byte aligned here: the plan sends anything
            }                                                  // else to the generic kernel (a predicated scalar path
        }                                                      // would cost an issue slot per sample even when unused)
    };
    auto stash = [&](const int4 (&q)[C::VPT]) {
#pragma unroll
        for (int v = 0; v < C::VPT; ++v) {
            rdst[v][0] = (uint32_t)q[v].x;
            rdst[v][1] = (uint32_t)q[v].y;
            rdst[v][2] = (uint32_t)q[v].z;
            rdst[v][3] = (uint32_t)q[v].w;
        }
    };

    int4 q[C::VPT];
    if (t_begin < t_end) {
        fetch(t_begin, q);
        stash(q);
    }
    __syncthreads();

    // int8 -> fp32 with the F-stage scale s = 2^-sh folded in (exact): byte b -> ((b ^ 0x80) + 2^23 - (2^23 + 128)) * s
    const float s = P.in_scale;
    const float bias = -8388736.0f * s;
    const float2 ss = make_float2(s, s), bb = make_float2(bias, bias);
    const uint32_t *rrow = raw + lane * C::ROW_WORDS + (C::RPT == 2 ? w : (w >> 1));
    float2 *ex_w = ex + (w * C::RPT) * 32 + lane;                     // + (k1 * R2 + e) * 32
    const float2 *ex_r = ex + (w * C::KPT) * R2 * 32 + lane;          // + (e * R2 + r) * 32
    const float4 *tw_row = reinterpret_cast<const float4 *>(P.twc + (w * C::RPT) * R1);   // rows r = RPT w + e: warp-uniform

    // output addressing: position p of bin k = k1 + R1 k2 is k +- N/2 when K == N
    const int i = i0 + lane;
    const bool iok = i < P.n_inputs;
    const int half = P.K / 2;
    const unsigned chan_stride = (unsigned)P.T * (unsigned)P.pitch2;  // half2 elements between positions (< 2^32: checked at create)
    __half2 *ybase = P.Y + i;

    // store addressing: one pointer chain per k1 where a thread has ONE k1 (N <= 128: -1.4 % at N = 128); with two (N >= 256)
    // the extra live pointers spill under the two-CTA register budget and cost 4.6 %, so those keep (p, t) addressing
    constexpr bool CHAIN = (C::KPT == 1);
    unsigned cs_reg;                                                  // chan_stride in a general register for the whole loop (the
    asm volatile("mov.u32 %0, %1;" : "=r"(cs_reg) : "r"(chan_stride));   // compiler re-materialised it from the constant bank per store)
    const unsigned row_bytes = (unsigned)P.pitch2 * 4u;
    char *yq[C::KPT];
#pragma unroll
    for (int e = 0; e < C::KPT; ++e)
        yq[e] = reinterpret_cast<char *>(ybase + ((size_t)(w * C::KPT + e) * P.T + t_begin) * P.pitch2);
    for (int t = t_begin; t < t_end; ++t) {
        const bool more = (t + 1) < t_end;
        if (more) fetch(t + 1, q);                                    // in flight during both passes

        // ---- pass 1: this thread's residues r = w*RPT + e; points x[r + R2 j], j < R1
        {
            float2 x[C::RPT][R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                if (C::RPT == 2) {
                    // samples q = 2w + R2 j and q + 1 share one 32-bit word
                    const uint32_t word = rrow[(R2 / 2) * j] ^ 0x80808080u;
                    x[0][j] = fma2(make_float2(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7440)), __uint_as_float(__byte_perm(word, 0x4B000000u, 0x7441))), ss, bb);
                    x[C::RPT - 1][j] = fma2(make_float2(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7442)), __uint_as_float(__byte_perm(word, 0x4B000000u, 0x7443))), ss, bb);
                } else {
                    uint32_t word = rrow[(R2 / 2) * j] ^ 0x80808080u;
                    if (w & 1) word >>= 16;
                    x[0][j] = fma2(make_float2(__uint_as_float(__byte_perm(word, 0x4B000000u, 0x7440)), __uint_as_float(__byte_perm(word, 0x4B000000u, 0x7441))), ss, bb);
                }
            }
#pragma unroll
            for (int e = 0; e < C::RPT; ++e) {
                fft_dif<R1>(x[e]);
#pragma unroll
                for (int kk = 0; kk < R1; kk += 2) {
                    const float4 tw2 = tw_row[(e * R1 + kk) / 2];     // W_N^{r kk}, W_N^{r (kk+1)}: warp-uniform
                    float2 v0 = x[e][bitrev(kk, ilog2(R1))];
                    float2 v1 = x[e][bitrev(kk + 1, ilog2(R1))];
                    if (kk > 0) v0 = cmul(v0, make_float2(tw2.x, tw2.y));
                    v1 = cmul(v1, make_float2(tw2.z, tw2.w));
                    ex_w[(kk * R2 + e) * 32] = v0;
                    ex_w[((kk + 1) * R2 + e) * 32] = v1;
                }
            }
        }
        __syncthreads();                                              // ex complete; raw(t) no longer needed
        DelayGain gn = {0.f, 0.f};
        if (DELAY && iok) gn = load_delay_gain(P.delay, P.phase, (long long)i * P.d_stride + P.frame0 + t, 1.0f / (float)N);

        // ---- pass 2: this thread's k1 = w*KPT + e; X[k1 + R1 k2] = FFT_R2 over r
        // DELAY: the gains of the bins u = k1 + R1 k2 (k2 < R2/2) and u = k1 - N/2 + R1 (k2 - R2/2) are two geometric runs of
        // ratio gs; each run is walked as CH interleaved chains of ratio gs^CH (one dependent chain of complex multiplies in
        // the store loop of this latency-bound kernel cost more than the sine and cosine per bin it replaced)
        constexpr int CH = (R2 / 2 >= 4) ? 4 : R2 / 2;
        const float2 gs = DELAY ? delay_gain_at(0.0f, gn.st, R1) : make_float2(1.0f, 0.0f);
        const float2 gsc = DELAY ? delay_gain_at(0.0f, gn.st, R1 * CH) : make_float2(1.0f, 0.0f);
#pragma unroll
        for (int e = 0; e < C::KPT; ++e) {
            const int k1 = w * C::KPT + e;
            float2 y[R2];
#pragma unroll
            for (int r = 0; r < R2; ++r) y[r] = ex_r[(e * R2 + r) * 32];
            fft_dif<R2>(y);
            if (DELAY) {
                // gains in place, before the store loop: g[k2] for both runs
#pragma unroll
                for (int hrun = 0; hrun < 2; ++hrun) {
                    float2 gq[CH];
                    gq[0] = delay_gain_at(gn.pt, gn.st, hrun ? k1 - N / 2 : k1);
#pragma unroll
                    for (int j = 1; j < CH; ++j) gq[j] = cmul(gq[j - 1], gs);
#pragma unroll
                    for (int q = 0; q < R2 / 2; ++q) {
                        const int k2 = hrun * (R2 / 2) + q;
                        y[bitrev(k2, ilog2(R2))] = cmul(y[bitrev(k2, ilog2(R2))], gq[q % CH]);
                        if (q + CH < R2 / 2) gq[q % CH] = cmul(gq[q % CH], gsc);
                    }
                }
            }
            if (FULL && CHAIN) {
                // K == N: the thread's R2 bins k1 + R1 k2 land on the positions p = k1 + R1 j, j = (k2 + R2/2) mod R2: ONE chain of
                // R2 rows, R1 channel positions apart, from a per-thread pointer that moves one spectrum per frame.  (Forming
                // every address from (p, t) cost ~60 integer instructions per frame, an eighth of the kernel's issue slots.)
                const float *swp = P.swc + k1;
                char *dst = yq[e];
                if (iok) {
#pragma unroll
                    for (int jj = 0; jj < R2; ++jj) {
                        const int k2 = (jj + R2 / 2) % R2;
                        float2 v = y[bitrev(k2, ilog2(R2))];
                        if (SCALE) v = scale2(v, swp[R1 * jj]);
                        *reinterpret_cast<__half2 *>(dst) = __floats2half2_rn(v.x, v.y);
                        dst += (unsigned long long)cs_reg * (unsigned)(R1 * 4);       // one IMAD.WIDE.U32
                    }
                }
                yq[e] += row_bytes;
            } else if (FULL) {
                // k < N/2  <=>  k2 < R2/2:  p = k + N/2, else p = k - N/2
                __half2 *yp = ybase + ((size_t)(k1 + N / 2) * P.T + t) * P.pitch2;
                __half2 *yn = ybase + ((size_t)k1 * P.T + t) * P.pitch2;
                const float *swp = P.swc + k1;
                if (iok) {
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) {
                        float2 v = y[bitrev(k2, ilog2(R2))];
                        const int pk = (k2 < R2 / 2) ? (N / 2 + R1 * k2) : (R1 * k2 - N / 2);   // p - k1
                        if (SCALE) v = scale2(v, swp[pk]);
                        __half2 *dst = (k2 < R2 / 2) ? yp + (size_t)(unsigned)(R1 * k2) * chan_stride      // one IMAD.WIDE.U32
                                                     : yn + (size_t)(unsigned)(R1 * (k2 - R2 / 2)) * chan_stride;
                        *dst = __floats2half2_rn(v.x, v.y);
                    }
                }
            } else if (iok) {
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const int k = k1 + R1 * k2;
                    const int u = (k < N / 2) ? k : k - N;                   // signed bin
                    const int p = u + half;                                  // centre order
                    if (p < 0 || p >= P.K) continue;                         // keep the central K channels (L611)
                    float2 v = y[bitrev(k2, ilog2(R2))];
                    if (SCALE) v = scale2(v, P.swc[p]);                      // sqrt(w_p): shared edge / DC exclusion
                    ybase[((size_t)p * P.T + t) * P.pitch2] = __floats2half2_rn(v.x, v.y);
                }
            }
        }
        // the prefetched bytes of frame t + 1 go into the raw tile as LATE as possible (the tile is free from the first barrier
        // on): stashed right after pass 1, as in round 1, the store waited for the loads and held 28 % of the kernel's stall
        // samples (profiles/r2_ncu_full.md); here they have had both passes to arrive
        if (more) stash(q);
        __syncthreads();                                              // ex consumed; raw(t+1) visible
    }
}

}  // namespace mwax
