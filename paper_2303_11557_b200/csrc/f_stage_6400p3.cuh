// f_stage_6400p3.cuh — F stage for the paper's own frame length N = 6400 = 20 x 20 x 16 (§2.5,
// L264: "6400-point FFT", 200 Hz ultra-fine channels): a three-pass in-place shared-memory FFT with radix-20, 20
// and 16 sub-transforms in registers, 640 threads (20 warps) per CTA so that global-load latency is hidden by
// thread-level parallelism (a two-pass 80 x 80 variant needs 160 registers of data per thread, runs at 5 warps
// per SM and measured slower: DESIGN.md §5.1).
//
//   n = 320 n1 + 16 n2 + n3,   k = k1 + 20 k2 + 400 k3        (n1, n2, k1, k2 < 20;  n3, k3 < 16)
//   pass 1  task (n2, n3): A[k1]   = sum_{n1} x[320 n1 + 16 n2 + n3] W_20^{n1 k1},   times W_400^{n2 k1}
//   pass 2  task (k1, n3): B[k2]   = sum_{n2} A[k1; n2, n3] W_20^{n2 k2},            times s W_6400^{n3 (k1 + 20 k2)}
//   pass 3  task (k1, k2): X[k]    = sum_{n3} B[k1, k2; n3] W_16^{n3 k3}
//
// One CTA transforms one frame of G = 4 adjacent inputs; thread = (g = tid & 3, j = tid >> 2 in [0,160)).
// Every global LOAD of the steady state is the raw voltage itself: a thread owns the two adjacent samples
// n3 = 2 lo, 2 lo + 1 of its (n2 | k1) row, fetches them as one 32-bit word per n1 (a warp reads 32 contiguous
// bytes of each of its 4 inputs) into 20 registers, and does so one item AHEAD (issued when pass 3 starts, used
// by the next item's pass 1), so no pass waits on HBM.  All twiddles are small shared-memory tables:
//   W_400^{n2 k1} [n2][k1] (warp-uniform rows), s W_320^{n3 k2} [n3][k2] (rows padded to 21), and the factor
//   W_6400^{n3 k1}, which is a per-thread constant of pass 2 (two registers per task).
// Exchange buffer E[g][i1][i2][n3] fp32 complex, float2 strides (S1, 16, 1) = (322, 16, 1), input g at
// g * 6440 + {0,1,1,0}: the 16 lanes of a half warp (4 g x 4 consecutive lo, i.e. n3 step 2, in passes 1-2;
// 4 g x 4 consecutive k1, S1 = 2 mod 16, in pass 3) fall in 16 different 8-byte bank pairs: offsets
// {0,2,4,6} + {0,9,1,8} (mod 16).  No bank conflicts in any pass.
// Pass 3 stores fp16 results already corner-turned: lanes (g, 8 consecutive bins) write 8 rows x 16 bytes of
// Y[p][t][input]; all 128 input groups of a frame run in the same wave of persistent CTAs, so the eight 16-byte
// pieces of every 128-byte line meet in L2 before the line goes to HBM (ncu: dram write bytes = algorithmic).
#pragma once
#include <cuda_fp16.h>
#include <cstdint>
#include "f_stage.cuh"
#include "f_stage_pow2.cuh"
#include "ptx.cuh"

namespace mwax {

// exp(-2 pi i m / 20), m = 1..12 (the twiddles inside the 20-point transform)
__device__ __forceinline__ float2 w20(int m)
{
    switch (m) {
        case 1: return make_float2(9.510565163e-01f, -3.090169944e-01f);
        case 2: return make_float2(8.090169944e-01f, -5.877852523e-01f);
        case 3: return make_float2(5.877852523e-01f, -8.090169944e-01f);
        case 4: return make_float2(3.090169944e-01f, -9.510565163e-01f);
        case 5: return make_float2(0.0f, -1.0f);
        case 6: return make_float2(-3.090169944e-01f, -9.510565163e-01f);
        case 7: return make_float2(-5.877852523e-01f, -8.090169944e-01f);
        case 8: return make_float2(-8.090169944e-01f, -5.877852523e-01f);
        case 9: return make_float2(-9.510565163e-01f, -3.090169944e-01f);
        case 10: return make_float2(-1.0f, 0.0f);
        case 11: return make_float2(-9.510565163e-01f, 3.090169944e-01f);
        case 12: return make_float2(-8.090169944e-01f, 5.877852523e-01f);
        default: return make_float2(1.0f, 0.0f);
    }
}

// In-register 20-point forward DFT.  In: x[a][b] = sample index 4 a + b (a < 5, b < 4).
// Out: X[ka + 5 kb] in x[ka][kb]  (ka < 5, kb < 4).
__device__ __forceinline__ void fft20(float2 (&x)[5][4])
{
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        float2 v[5] = {x[0][b], x[1][b], x[2][b], x[3][b], x[4][b]};
        butterfly<5>(v);                                             // over a -> ka
#pragma unroll
        for (int ka = 0; ka < 5; ++ka) x[ka][b] = (b * ka == 0) ? v[ka] : cmul(v[ka], w20(b * ka));   // W_20^{b ka}
    }
#pragma unroll
    for (int ka = 0; ka < 5; ++ka) butterfly<4>(x[ka]);              // over b -> kb
}

struct F6400P3 {
    static constexpr int N = 6400, G = 4;
    static constexpr int THREADS = 640;                              // 160 per input
    static constexpr int S1 = 322, SG = 20 * S1;                     // float2 strides: S1 = 2, SG = 8 (mod 16)
    static constexpr int E_F2 = G * SG + 2;                          // + the per-input offsets {0,1,1,0}
    static constexpr int T1_OFF = E_F2;                              // W_400^{n2 k1} [n2][k1], 400 float2
    static constexpr int T2_OFF = T1_OFF + 400;                      // s W_320^{n3 k2} [n3][21], 336 float2
    static constexpr int CODE_OFF = T2_OFF + 336;                    // 400 x uint32 weight codes (as 200 float2)
    static constexpr int SMEM_BYTES = (CODE_OFF + 200) * 8;          // 213,584
    static_assert(S1 % 16 == 2 && SG % 16 == 8 && T1_OFF % 2 == 0, "bank-conflict-free strides, 16-byte aligned tables");
};


// ---- thread-block-cluster helpers (distributed shared memory)
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_count_x()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
// relaxed arrive: orders nothing; enough to tell the other CTAs "I have finished READING your shared memory"
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// shared::cluster address of local shared address `saddr` in CTA `rank` of this cluster
__device__ __forceinline__ uint32_t ld_dsmem_base(uint32_t saddr, uint32_t rank)
{
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(saddr), "r"(rank));
    return ra;
}
// 16 bytes from distributed shared memory
__device__ __forceinline__ uint4 ld_shared_cluster_v4(uint32_t caddr)
{
    uint4 v;
    asm volatile("ld.shared::cluster.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(caddr) : "memory");
    return v;
}

// FULL : K == N (every bin kept)          SCALE : multiply by sqrt(w_p) (averaging weights folded into the F stage)
// Q    : CTAs per cluster.  A cluster transforms one frame of 4 Q adjacent inputs (CTA rank r: inputs 4 r .. 4 r + 3)
//        and each CTA then STORES the rows of 16 / Q values of k3 for all 4 Q inputs, fetching the other CTAs'
//        fp16 results through distributed shared memory: every global store is 16 bytes wide and a row receives
//        16 Q contiguous bytes at once (Q = 2: whole 32-byte sectors, Q = 8: whole 128-byte lines).  With one CTA
//        per row piece (Q = 1) the 16-byte pieces of a sector arrive from different SMs at different times and L2
//        turns them into read-modify-write DRAM traffic (ncu: profiles/r1_f6400.md).
// DELAY: fractional-delay / phase gain per (input, frame) applied to the pass-3 results (PAPER.md 2.5.1 L266-272)
template <bool FULL, bool SCALE, int Q, bool DELAY = false>
__global__ void __launch_bounds__(F6400P3::THREADS, 1) f_stage_6400p3_kernel(const FParams P)
{
    using C = F6400P3;
    extern __shared__ __align__(16) float2 esm[];
    float2 *t1 = esm + C::T1_OFF;                                    // W_400^{n2 k1} = W_6400^{16 n2 k1}
    float2 *t2 = esm + C::T2_OFF;                                    // s W_320^{n3 k2} = s W_6400^{20 n3 k2}
    uint32_t *codes = reinterpret_cast<uint32_t *>(esm + C::CODE_OFF);
    for (int e = threadIdx.x; e < 400; e += C::THREADS) {
        t1[e] = __ldg(&P.tw[(16 * (e / 20) * (e % 20)) % C::N]);
        if (FULL && SCALE) codes[e] = __ldg(&P.swcode[e]);
    }
    for (int e = threadIdx.x; e < 320; e += C::THREADS) {
        const float2 w = __ldg(&P.tw[(20 * (e / 20) * (e % 20)) % C::N]);
        t2[(e / 20) * 21 + e % 20] = make_float2(w.x * P.in_scale, w.y * P.in_scale);
    }
    __syncthreads();

    // Q = 2: the partner's fp16 rows are PUSHED into this CTA by bulk copies (one per k1: its 20 slots are contiguous, 2560 bytes;
    // completion counted on `rx_bar`) into the slots of input 1, free once pass 3 has read them; the
    // store phase then reads local shared memory only.  Pulling the rows with ld.shared::cluster inside the store loop
    // left every store waiting on a remote load: 37 % of the kernel's stall samples (profiles/r1_ncu_full.md).
    constexpr bool PUSH = (Q == 2);
    // float2 index of the receive area of CTA r: 16-byte aligned, and 64 bytes (mod 128) away from that CTA's own staged
    // rows (input 0's slots for rank 0, input 3's for rank 1), so that the 16-byte reads of a row's two pieces never share banks
    auto rx_off = [](uint32_t r) { return C::SG + (r ? 8 : 0); };
    __shared__ __align__(8) unsigned long long rx_bar;
    const uint32_t rx_bar_a = ptx::smem_u32(&rx_bar);
    uint32_t rx_phase = 0;
    if (PUSH && threadIdx.x == 0) {
        ptx::mbar_init(rx_bar_a, 1);
        ptx::fence_mbar_init();
    }
    const uint32_t rank = cluster_ctarank();
    const int g = threadIdx.x & 3, j = threadIdx.x >> 2;             // j in [0,160)
    const int hi = j >> 3, lo = j & 7;                               // hi = warp index (warp-uniform), in [0,20)
    float2 *eg = esm + g * C::SG + ((g == 1 || g == 2) ? 1 : 0);
    const int groups = (P.n_inputs + C::G * Q - 1) / (C::G * Q);     // groups of 4 Q inputs
    const int n_items = groups * P.T;
    const int half = P.K / 2;
    const unsigned chan_stride = P.y_p_stride;                       // half2 elements between channel positions
    // pass-2 constants of this thread's two tasks (k1 = hi, n3 = 2 lo + rep): W_6400^{n3 k1}
    const float2 cw0 = __ldg(&P.tw[(2 * lo) * hi]), cw1 = __ldg(&P.tw[(2 * lo + 1) * hi]);

    // raw voltages of one item: samples 320 n1 + 16 hi + 2 lo + {0,1}, n1 < 20, one 32-bit word each
    uint32_t raw[20];
    auto fetch = [&](int item) {
        const int t = item / groups;
        const int i = ((item - t * groups) * Q + (int)rank) * C::G + g;
        if (item < n_items && i < P.n_inputs) {
            const int8_t *src = P.volt + 2 * ((long long)i * P.row_pitch + P.sample0 + (long long)t * C::N + 16 * hi + 2 * lo);
#pragma unroll
            for (int q = 0; q < 20; ++q) raw[q] = __ldg(reinterpret_cast<const unsigned *>(src + 640 * q));   // 4-byte aligned: the
                                                                     // plan sends misaligned buffers to the generic kernel
        } else {
#pragma unroll
            for (int q = 0; q < 20; ++q) raw[q] = 0u;                // absent input: zeros
        }
    };
    const int item0 = (int)cluster_id_x(), item_step = (int)cluster_count_x();
    fetch(item0);
    cluster_arrive_relaxed();                                        // pairs with the wait before the first E write

    for (int item = item0; item < n_items; item += item_step) {
        const int t = item / groups;
        const int grp = item - t * groups;

        // ---- pass 1: tasks (n2 = hi, n3 = 2 lo + rep): 20-point FFT over n1 of x[320 n1 + 16 n2 + n3], then W_400^{n2 k1}
        float2 x[5][4];
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const uint32_t w = raw[4 * a + b];               // int8 -> fp32 promotion
                    x[a][b] = rep == 0 ? make_float2((float)(signed char)(w & 0xffu), (float)(signed char)((w >> 8) & 0xffu))
                                       : make_float2((float)(signed char)((w >> 16) & 0xffu), (float)(signed char)(w >> 24));
                }
            fft20(x);
            if (rep == 0) cluster_wait();                            // the other CTAs have finished reading my staged rows
            const float4 *trow = reinterpret_cast<const float4 *>(t1 + hi * 20);   // warp-uniform: broadcast loads
            float2 *ew = eg + hi * 16 + 2 * lo + rep;
#pragma unroll
            for (int k1 = 0; k1 < 20; k1 += 2) {
                const float4 tw = trow[k1 / 2];
                const float2 v0 = x[k1 % 5][k1 / 5], v1 = x[(k1 + 1) % 5][(k1 + 1) / 5];
                ew[k1 * C::S1] = (k1 == 0) ? v0 : cmul(v0, make_float2(tw.x, tw.y));
                ew[(k1 + 1) * C::S1] = cmul(v1, make_float2(tw.z, tw.w));
            }
        }
        __syncthreads();

        // ---- pass 2 (in place): tasks (k1 = hi, n3 = 2 lo + rep): 20-point FFT over n2, then s W_6400^{n3 (k1 + 20 k2)}
#pragma unroll 1
        for (int rep = 0; rep < 2; ++rep) {
            const int n3 = 2 * lo + rep;
            float2 *e = eg + hi * C::S1 + n3;
            const float2 *trow = t2 + n3 * 21;
            const float2 cw = rep ? cw1 : cw0;
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) x[a][b] = e[(4 * a + b) * 16];
            fft20(x);
#pragma unroll
            for (int k2 = 0; k2 < 20; ++k2) e[k2 * 16] = cmul(x[k2 % 5][k2 / 5], cmul(trow[k2], cw));
        }
        __syncthreads();

        // the next item's voltages travel while pass 3 computes and stores
        fetch(item + item_step);

        DelayGain gn = {0.f, 0.f};
        if (DELAY) {
            const int i = (grp * Q + (int)rank) * C::G + g;
            if (i < P.n_inputs) gn = load_delay_gain(P.delay, P.phase, (long long)i * P.d_stride + P.frame0 + t, 1.0f / (float)C::N);
        }

        // ---- pass 3: tasks c = k1 + 20 k2 = j + 160 r: 16-point FFT over n3 -> bins k = c + 400 k3, rounded to fp16 and
        // staged in place as rows S(c, k3) = 4 inputs x 4 bytes, inside the slots of inputs 0 (k3 < 8) and 3 (k3 >= 8)
#pragma unroll 1
        for (int r = 0; r < 3; ++r) {
            const int c = j + 160 * r;
            if (c >= 400) break;                                     // warp-uniform
            const int k2 = c / 20, k1 = c - 20 * k2;
            const int slot = k1 * C::S1 + k2 * 16;
            const float2 *e = eg + slot;
            float2 z[16];
#pragma unroll
            for (int n3 = 0; n3 < 16; ++n3) z[n3] = e[n3];
            __syncwarp();                                            // the four slots of this c are now free
            fft_dif<16>(z);
            uint32_t *s_lo = reinterpret_cast<uint32_t *>(esm + slot) + g;
            uint32_t *s_hi = reinterpret_cast<uint32_t *>(esm + 3 * C::SG + slot) + g;
            const uint32_t code = (FULL && SCALE) ? codes[c] : 0u;   // 2 bits per k3: 0 -> 1, 1 -> sqrt(1/2), 2 -> 0
            if (DELAY) {
#pragma unroll
                for (int k3 = 0; k3 < 16; ++k3)
                    z[bitrev(k3, 4)] = apply_delay_gain(z[bitrev(k3, 4)], gn, c + 400 * k3 - (k3 < 8 ? 0 : C::N));
            }
            if (FULL && SCALE && code != 0u) {                       // rare: 8 + 1 of the 400 tasks at F = 50
#pragma unroll
                for (int k3 = 0; k3 < 16; ++k3) {
                    const uint32_t cd = (code >> (2 * k3)) & 3u;
                    const float f = cd == 0u ? 1.0f : (cd == 1u ? 0.70710678118654757f : 0.0f);
                    z[bitrev(k3, 4)].x *= f;
                    z[bitrev(k3, 4)].y *= f;
                }
            }
#pragma unroll
            for (int k3 = 0; k3 < 16; ++k3) {
                float2 v = z[bitrev(k3, 4)];
                if (!FULL && SCALE) {
                    const int k = c + 400 * k3;
                    const int p = ((k < C::N / 2) ? k : k - C::N) + half;
                    const float f = (p >= 0 && p < P.K) ? __ldg(&P.sw[p]) : 0.0f;
                    v.x *= f;
                    v.y *= f;
                }
                const __half2 hv = __floats2half2_rn(v.x, v.y);
                ((k3 < 8) ? s_lo : s_hi)[(k3 & 7) * 4] = *reinterpret_cast<const uint32_t *>(&hv);
            }
        }
        if (PUSH) {
            ptx::fence_proxy_async();                                // the staged rows will be read by bulk copies
            if (threadIdx.x == 0) ptx::mbar_arrive_expect_tx(rx_bar_a, 400u * 128u);   // this item's incoming rows
        }
        // PUSH: the staged rows are read by THIS CTA's own bulk copies, so CTA-level ordering (bar.sync) is enough, and the
        // cluster barrier only has to say "my pass 3 no longer reads the slots you are about to overwrite": a relaxed
        // arrive.  The release form compiles to MEMBAR.ALL.GPU + ERRBAR, which also waits for the 20 voltage loads of the
        // next item that were issued when pass 3 started - it turned the one-item-ahead prefetch into a blocking load.
        if (PUSH) {
            __syncthreads();
            cluster_arrive_relaxed();
        } else {
            cluster_arrive();
        }
        cluster_wait();                                              // every CTA of the cluster has staged its rows
        if (PUSH) {
            // rows of the OTHER CTA's k3 half: rank 0 sends its k3 >= 8 rows (input 3's slots), rank 1 its k3 < 8 rows
            // the 20 slots (k2) of one k1 are contiguous: 20 copies of 2560 bytes
            if (threadIdx.x < 20) {
                const int slot = threadIdx.x * C::S1;
                const uint32_t base = (uint32_t)__cvta_generic_to_shared(esm);
                const uint32_t src = base + (uint32_t)(((rank == 0 ? 3 * C::SG : 0) + slot) * 8);
                const uint32_t dst = ld_dsmem_base(base + (uint32_t)((rx_off(rank ^ 1u) + slot) * 8), rank ^ 1u);
                ptx::bulk_copy_to_cluster(dst, src, 20u * 128u, ld_dsmem_base(rx_bar_a, rank ^ 1u));
            }
            ptx::mbar_wait(rx_bar_a, rx_phase);                      // the partner's rows of MY k3 half have landed
            rx_phase ^= 1u;
        }

        // ---- corner-turned store: this CTA writes rows k3 in [rank 16/Q, (rank + 1) 16/Q) for all 4 Q inputs
        // Thread = (piece q = tid % Q of a row, row stream tid / Q + (640 / Q) it): 640 / Q is a multiple of 20, so k1 is
        // a per-thread constant and (c, k3) advance by additions.  Loads go out in batches of 4 (all of a batch's
        // remote reads in flight together), then the batch is stored: 16-byte pieces, Q adjacent lanes per row.
        {
            constexpr int RSTEP = C::THREADS / Q;                    // rows per iteration (320 / 160 / 80)
            const int q = threadIdx.x % Q;
            const uint32_t rbase = ld_dsmem_base((uint32_t)__cvta_generic_to_shared(esm), (uint32_t)q);
            const int col = (grp * Q + q) * C::G;
            const bool col_ok = col < P.pitch2;
            __half2 *ycol = P.Y + (size_t)t * P.y_t_stride + col;
            int c = threadIdx.x / Q, kl = 0;
            const int k1 = c % 20;
            constexpr int NB = 4;                                    // loads in flight per thread
#pragma unroll 1
            for (int b0 = 0; b0 < C::N / C::THREADS; b0 += NB) {
                uint4 pv[NB];
                int pk[NB];
#pragma unroll
                for (int e = 0; e < NB; ++e) {
                    if (b0 + e >= C::N / C::THREADS) break;
                    const int k3 = (int)rank * (16 / Q) + kl;
                    const int k2 = c / 20;
                    if (PUSH) {                                      // own piece: staged slot; partner's piece: receive area
                        const int area = (q == (int)rank) ? (k3 < 8 ? 0 : 3 * C::SG) : rx_off(rank);
                        pv[e] = *reinterpret_cast<const uint4 *>(reinterpret_cast<const uint8_t *>(esm) +
                                                                  (area + k1 * C::S1 + k2 * 16) * 8 + (k3 & 7) * 16);
                    } else {
                        const uint32_t so = (uint32_t)(((k3 < 8 ? 0 : 3 * C::SG) + k1 * C::S1 + k2 * 16) * 8 + (k3 & 7) * 16);
                        pv[e] = ld_shared_cluster_v4(rbase + so);
                    }
                    pk[e] = c + 400 * k3;
                    c += RSTEP;
                    if (c >= 400) { c -= 400; ++kl; }
                }
#pragma unroll
                for (int e = 0; e < NB; ++e) {
                    if (b0 + e >= C::N / C::THREADS) break;
                    const int p = ((pk[e] < C::N / 2) ? pk[e] : pk[e] - C::N) + half;   // centre order (L290); keep (L611)
                    if (col_ok && (FULL || (p >= 0 && p < P.K))) *reinterpret_cast<uint4 *>(ycol + (size_t)p * chan_stride) = pv[e];
                }
            }
        }
        cluster_arrive_relaxed();                                    // pairs with the wait inside the next pass 1
    }
    cluster_wait();                                                  // nobody may leave while its rows can still be read
}

}  // namespace mwax
