// f_stage_6400.cuh — F stage for the paper's own frame length N = 6400 = 20 x 20 x 16 (§2.5,
// L264: "6400-point FFT", 200 Hz ultra-fine channels): a three-pass in-place shared-memory FFT with radix-20, 20 and
// 16 sub-transforms in registers, 640 threads (20 warps) per CTA, one CTA per SM (the fp32 exchange buffer for four
// inputs is 206 KB).  Round 2's design: the passes of round 1's cluster kernel WITHOUT clusters, row staging or a
// separate store phase:
//
//   n = 320 n1 + 16 n2 + n3,   k = k1 + 20 k2 + 400 k3        (n1, n2, k1, k2 < 20;  n3, k3 < 16)
//   pass 1  task (n2, n3): A[k1]   = sum_{n1} x[320 n1 + 16 n2 + n3] W_20^{n1 k1},   times W_400^{n2 k1}
//   pass 2  task (k1, n3): B[k2]   = sum_{n2} A[k1; n2, n3] W_20^{n2 k2},            times s W_6400^{n3 (k1 + 20 k2)}
//   pass 3  task (k1, k2): X[k]    = sum_{n3} B[k1, k2; n3] W_16^{n3 k3}
//
// A CTA's natural output is 4 inputs x 4 bytes = 16 bytes of a Y[p][t][input] row; L2 turns such partial 32-byte
// sectors into read-modify-write DRAM traffic (profiles/r1_ncu_full.md), so round 1 exchanged rows between the two
// CTAs of a cluster (15 % of the kernel on the push + wait, 21 % on a separate store phase).  Here a work item is
// (frame t, group of EIGHT adjacent inputs), done as two sub-items of four inputs, thread g <-> input 2 g + s:
//   pass 3 of BOTH sub-items rounds its results to fp16 and PARKS them in tensor memory (tcgen05.st, thread-private
//   lanes: TMEM is 256 KB of otherwise idle on-chip storage in this kernel; 204 KB are used), sub-item 1 next to sub-item 0;
//   the item then leaves during passes 1 and 2 of the NEXT item's first sub-item: at twelve points of those passes every
//   thread reads four bins of both sub-items back (tcgen05.ld) and stores {input 2 g, input 2 g + 1} = 8 bytes per bin,
//   four adjacent lanes = one whole 32-byte sector.  Issued in one burst at the end of pass 3 the 6400 scattered sectors of
//   an item held 30 % of the kernel (2.38 ms, 1.66 ms with the stores removed: the LSU takes a cycle per 128-byte line an
//   instruction touches, eight per STG.64 here, and 20 warps x 16 stores queued at once); spread out they cost half of that.
// Every global LOAD of the steady state is the raw voltage itself, one sub-item ahead (see fetch()).
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

struct F6400 {
    static constexpr int N = 6400, G = 4, GI = 8;                    // inputs per sub-item / per work item
    static constexpr int THREADS = 640;                              // 160 per input
    // Exchange buffer E[g][k1][i2][n3] fp32 complex, float2 strides (SG, S1, S2, 1) = (6820, 341, 17, 1).  Passes 1 and 2:
    // a warp = ONE input x four values a of the middle index (n2 | k1) x eight sample pairs lo; the 16 lanes of a half warp
    // (a in {0,1} | {2,3}, lo) touch float2 offsets 17 a + 2 lo (pass 1) / 341 a + 2 lo (pass 2): 16 different 8-byte bank
    // pairs since 17 and 341 are odd.  Pass 3: a warp = four inputs g x eight consecutive k1; offsets 6820 g + 341 k1 =
    // 4 g + 5 k1 (mod 16), all different for g, k1 < 4.  No bank conflicts in any pass.
    static constexpr int S2 = 17;                                    // float2 stride of the middle index (n2 | k2)
    static constexpr int S1 = 20 * S2 + 1, SG = 20 * S1;             // float2 strides of k1 and of the input
    static constexpr int E_F2 = G * SG;
    static constexpr int T1_OFF = E_F2;                              // W_400^{n2 k1} [n2][k1], 400 float2
    static constexpr int T2_OFF = T1_OFF + 400;                      // s W_320^{n3 k2}: row pair (n3 = 2 lo, 2 lo + 1) at 42 lo, the odd row 22 in: 336 float2
    static constexpr int CODE_OFF = T2_OFF + 336;                    // 400 x uint32 weight codes (as 200 float2)
    static constexpr int SMEM_BYTES = (CODE_OFF + 200) * 8;          // 225,728
    static constexpr int TMEM_COLS = 512;                            // 5 warps per lane quadrant x 96 columns
    static constexpr int PARK_STRIDE = 96;                           // columns per warp: 2 sub-items x 3 rounds x 16 words
    static constexpr int PARK_SUB = 48;                              // column offset of sub-item 1's words
    static_assert(S2 % 2 == 1 && S1 % 16 == 5 && SG % 16 == 4 && T1_OFF % 2 == 0, "bank-conflict-free strides, 16-byte aligned tables");
    static_assert(5 * PARK_STRIDE <= TMEM_COLS, "parked rows of the five warps of a lane quadrant");
};

// TMEM as thread-private scratch: this warp's 32 lanes x 16 consecutive 32-bit columns (thread L <-> lane base + L)
__device__ __forceinline__ void tmem_st_32x32b_x16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
          "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tmem_ld_32x32b_x4(uint32_t taddr, uint32_t (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(taddr)
                 : "memory");
}
// streaming 4-byte load that does not allocate an L1 line (the shared tile leaves this kernel almost no L1)
__device__ __forceinline__ uint32_t ld_stream_u32(const void *p)
{
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// FULL : K == N (every bin kept)          SCALE : multiply by sqrt(w_p) (averaging weights folded into the F stage)
// DELAY: fractional-delay / phase gain per (input, frame) applied to the pass-3 results (PAPER.md 2.5.1 L266-272)
template <bool FULL, bool SCALE, bool DELAY = false>
__global__ void __launch_bounds__(F6400::THREADS, 1) f_stage_6400_kernel(const FParams P)
{
    using C = F6400;
    extern __shared__ __align__(16) float2 esm[];
    float2 *t1 = esm + C::T1_OFF;                                    // W_400^{n2 k1} = W_6400^{16 n2 k1}
    float2 *t2 = esm + C::T2_OFF;                                    // s W_320^{n3 k2} = s W_6400^{20 n3 k2}
    uint32_t *codes = reinterpret_cast<uint32_t *>(esm + C::CODE_OFF);
    __shared__ uint32_t tmem_slot;
    for (int e = threadIdx.x; e < 400; e += C::THREADS) {
        t1[e] = __ldg(&P.tw[(16 * (e / 20) * (e % 20)) % C::N]);
        if (FULL && SCALE) codes[e] = __ldg(&P.swcode[e]);
    }
    for (int e = threadIdx.x; e < 320; e += C::THREADS) {
        const float2 w = __ldg(&P.tw[(20 * (e / 20) * (e % 20)) % C::N]);
        t2[(e / 40) * 42 + 22 * ((e / 20) & 1) + e % 20] = make_float2(w.x * P.in_scale, w.y * P.in_scale);
    }
    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_slot), C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    // this thread's parking place: its own lane of the warp's quadrant, 96 columns per warp of the quadrant (two sub-items x 48)
    const uint32_t park = *reinterpret_cast<volatile uint32_t *>(&tmem_slot) + ((uint32_t)((warp & 3) * 32) << 16) +
                          (uint32_t)((warp >> 2) * C::PARK_STRIDE);

    float2 *eg = esm + (threadIdx.x & 3) * C::SG;
    // passes 1 and 2 (and the voltage loads): warp = (input gw, five groups v of four middle-index values), lane = (a, lo):
    // the 32 lanes of a load instruction read 128 CONTIGUOUS bytes of one input, one L2 request instead of the four
    // 32-byte ones of (4 inputs x 8 pairs) warps: 400 instead of 1600 read requests per sub-item (measured: -3.5 %)
    const int lane = threadIdx.x & 31;
    const int gw = warp / 5, hi = 4 * (warp % 5) + (lane >> 3), lo = lane & 7;   // hi = n2 (pass 1) = k1 (pass 2), in [0,20)
    float2 *egw = esm + gw * C::SG;
    const int groups = (P.n_inputs + C::GI - 1) / C::GI;             // groups of 8 inputs
    const int n_sub = 2 * groups * P.T;                              // sub-items: (frame t, group, s), s fastest
    const int half = P.K / 2;
    const unsigned chan_stride = P.y_p_stride;                       // half2 elements between channel positions
    // pass-2 constants of this thread's two tasks (k1 = hi, n3 = 2 lo + rep): W_6400^{n3 k1}
    const float2 cw0 = __ldg(&P.tw[(2 * lo) * hi]), cw1 = __ldg(&P.tw[(2 * lo + 1) * hi]);

    // raw voltages of one sub-item: samples 320 n1 + 16 hi + 2 lo + {0,1}, n1 < 20, one 32-bit word each.  (16-byte loads
    // by the four lanes that share a chunk + 4 x 4 lane transposes were measured SLOWER, 2.67 against 2.47 ms: a warp's load
    // touches the same number of 128-byte lines either way, and the shuffles come on top.)
    uint32_t raw[20];
    auto fetch = [&](int sub) {
        const int item = sub >> 1, s = sub & 1;
        const int t = item / groups;
        const int i = (item - t * groups) * C::GI + 2 * gw + s;
        if (sub < n_sub && i < P.n_inputs) {
            const int8_t *src = P.volt + 2 * ((long long)i * P.row_pitch + P.sample0 + (long long)t * C::N + 16 * hi + 2 * lo);
#pragma unroll
            for (int q = 0; q < 20; ++q) raw[q] = __ldg(reinterpret_cast<const unsigned *>(src + 640 * q));   // 4-byte aligned: the
                                                                     // plan sends misaligned buffers to the generic kernel
        } else {
#pragma unroll
            for (int q = 0; q < 20; ++q) raw[q] = 0u;                // absent input: zeros (pad columns of Y stay zero)
        }
    };
    const int sub0 = 2 * (int)blockIdx.x, sub_step = 2 * (int)gridDim.x;
    fetch(sub0);

    // Deferred stores.  Pass 3 of BOTH sub-items parks its fp16 rows in tensor memory; the 6400 sectors of item i leave
    // during passes 1 and 2 of the next item's first sub-item, four stores per thread at each of twelve points spread over
    // those passes (point pt: round r = pt / 4, bins k3 = 4 (pt % 4) ...+3).  Issued in one burst at the end of pass 3 they
    // cost 30 % of the kernel: the SM sends one 32-byte sector per clock to L2, 20 warps x 16 stores x 8 sectors queued at
    // once, and every warp sat on the full queue (profiles/r2_f6400.md).
    const unsigned cs_bytes = chan_stride * 4u;                      // bytes between channel positions (< 2^32: checked by the plan)
    const int g = threadIdx.x & 3, j = threadIdx.x >> 2;             // pass 3: thread = (input g of 4, task index j of 160)
    const char *yold = nullptr;                                      // column base of the parked item's rows (this thread's input pair)
    auto store_point = [&](int pt) {
        const int r = pt >> 2, k3b = (pt & 3) * 4;
        const int c = j + 160 * r;
        if (c >= 400) return;                                        // warp-uniform (r = 2: warps 0..9)
        uint32_t pa[4], pb[4];
        tmem_ld_32x32b_x4(park + (uint32_t)(16 * r + k3b), pa);
        tmem_ld_32x32b_x4(park + (uint32_t)(C::PARK_SUB + 16 * r + k3b), pb);
        ptx::tmem_ld_wait();
        // rows p = u + K/2 of the signed bins u = c + 400 k3 (k3 < 8), c - 3200 + 400 (k3 - 8) (k3 >= 8): centre order (L290), keep (L611)
        const int p0 = c + half + 400 * (k3b & 7) - (k3b < 8 ? 0 : C::N / 2);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int p = p0 + 400 * q;
            if (FULL || (p >= 0 && p < P.K))
                *reinterpret_cast<uint2 *>(const_cast<char *>(yold) + (size_t)(unsigned)p * cs_bytes) = make_uint2(pa[q], pb[q]);
        }
    };

    for (int sub_a = sub0; sub_a < n_sub; sub_a += sub_step) {
#pragma unroll 1
        for (int s = 0; s < 2; ++s) {
            const int item = sub_a >> 1;
            const int t = item / groups;
            const int grp = item - t * groups;

            // ---- pass 1: tasks (n2 = hi, n3 = 2 lo + rep): 20-point FFT over n1 of x[320 n1 + 16 n2 + n3], then W_400^{n2 k1}
            float2 x[5][4];
            const bool drain = (s == 0) && (yold != nullptr);        // this sub-item's passes 1-2 carry the previous item's stores
#pragma unroll
            for (int rep = 0; rep < 2; ++rep) {
                if (drain) store_point(3 * rep);
#pragma unroll
                for (int a = 0; a < 5; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        // int8 -> fp32 promotion on the ALU / FMA pipes: byte b ^ 0x80 placed in the mantissa
                        // of 2^23 gives 2^23 + b + 128 exactly (I2F.S8 runs on the quarter-rate XU pipe: 2 per sample made
                        // pass 1 XU bound, profiles/r2_f6400.md)
                        const uint32_t w = raw[4 * a + b] ^ 0x80808080u;
                        const float2 m = rep == 0 ? make_float2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7440)),
                                                                __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7441)))
                                                  : make_float2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7442)),
                                                                __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7443)));
                        x[a][b] = cadd(m, make_float2(-8388736.0f, -8388736.0f));
                    }
                fft20(x);
                if (drain) store_point(3 * rep + 1);
                const float4 *trow = reinterpret_cast<const float4 *>(t1 + hi * 20);   // four rows per warp, 160 bytes apart: one wavefront
                float2 *ew = egw + hi * C::S2 + 2 * lo + rep;
#pragma unroll
                for (int k1 = 0; k1 < 20; k1 += 2) {
                    if (k1 == 10 && drain) store_point(3 * rep + 2);
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
                float2 *e = egw + hi * C::S1 + n3;
                const float4 *trow = reinterpret_cast<const float4 *>(t2 + lo * 42 + 22 * rep);   // (k2, k2 + 1) pairs: 16-byte loads
                const float2 cw = rep ? cw1 : cw0;
#pragma unroll
                for (int a = 0; a < 5; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) x[a][b] = e[(4 * a + b) * C::S2];
                if (drain) store_point(6 + 3 * rep);
                fft20(x);
                if (drain) store_point(7 + 3 * rep);
#pragma unroll
                for (int k2 = 0; k2 < 20; k2 += 2) {
                    if (k2 == 10 && drain) store_point(8 + 3 * rep);
                    const float4 tw = trow[k2 / 2];
                    e[k2 * C::S2] = cmul(x[k2 % 5][k2 / 5], cmul(make_float2(tw.x, tw.y), cw));
                    e[(k2 + 1) * C::S2] = cmul(x[(k2 + 1) % 5][(k2 + 1) / 5], cmul(make_float2(tw.z, tw.w), cw));
                }
            }
            __syncthreads();

            // the next sub-item's voltages travel while pass 3 computes and stores.  They must be issued HERE: after the first
            // round of pass 3 they queue behind that round's stores in the LSU and pass 1 waits for them (measured 2.89 against
            // 2.43 ms); at the start of pass 2 they gain nothing (2.43)
            fetch(s == 0 ? sub_a + 1 : sub_a + sub_step);

            const int i_in = grp * C::GI + 2 * g + s;                // this thread's input in this sub-item
            DelayGain gn = {0.f, 0.f};
            if (DELAY && i_in < P.n_inputs)
                gn = load_delay_gain(P.delay, P.phase, (long long)i_in * P.d_stride + P.frame0 + t, 1.0f / (float)C::N);
            const float2 gs = DELAY ? delay_gain_at(0.0f, gn.st, 400) : make_float2(1.0f, 0.0f);
            // ---- pass 3: tasks c = k1 + 20 k2 = j + 160 r: 16-point FFT over n3 -> bins k = c + 400 k3, rounded to fp16 and
            // parked in TMEM (sub-item 1 next to sub-item 0: together they are the 8 bytes this thread stores per bin)
#pragma unroll 1
            for (int r = 0; r < 3; ++r) {
                const int c = j + 160 * r;
                if (c >= 400) break;                                 // warp-uniform (r = 2: warps 0..9)
                const int k2 = c / 20, k1 = c - 20 * k2;
                const float2 *e = eg + k1 * C::S1 + k2 * C::S2;
                float2 z[16];
#pragma unroll
                for (int n3 = 0; n3 < 16; ++n3) z[n3] = e[n3];
                fft_dif<16>(z);
                const uint32_t code = (FULL && SCALE) ? codes[c] : 0u;   // 2 bits per k3: 0 -> 1, 1 -> sqrt(1/2), 2 -> 0
                if (DELAY) {
                    // bins u = c + 400 k3 (k3 < 8) and u = c - 3200 + 400 (k3 - 8): two geometric runs of ratio gs
                    float2 gq = delay_gain_at(gn.pt, gn.st, c);
                    const float2 gneg = delay_gain_at(gn.pt, gn.st, c - C::N / 2);
#pragma unroll
                    for (int k3 = 0; k3 < 16; ++k3) {
                        if (k3 == 8) gq = gneg;
                        z[bitrev(k3, 4)] = cmul(z[bitrev(k3, 4)], gq);
                        if (k3 != 7 && k3 != 15) gq = cmul(gq, gs);
                    }
                }
                if (FULL && SCALE && code != 0u) {                   // rare: 8 + 1 of the 400 tasks at F = 50
#pragma unroll
                    for (int k3 = 0; k3 < 16; ++k3) {
                        const uint32_t cd = (code >> (2 * k3)) & 3u;
                        const float f = cd == 0u ? 1.0f : (cd == 1u ? 0.70710678118654757f : 0.0f);
                        z[bitrev(k3, 4)].x *= f;
                        z[bitrev(k3, 4)].y *= f;
                    }
                }
                uint32_t hv[16];
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
                    const __half2 h2 = __floats2half2_rn(v.x, v.y);
                    hv[k3] = *reinterpret_cast<const uint32_t *>(&h2);
                }
                tmem_st_32x32b_x16(park + (uint32_t)(C::PARK_SUB * s + 16 * r), hv);
            }
            tmem_st_wait();
            if (s != 0) {                                            // the item is complete in TMEM: its rows leave during the next passes 1-2
                const int col = grp * C::GI + 2 * g;                 // complex column of this thread's input pair (< pitch2: 8 | 32)
                yold = reinterpret_cast<const char *>(P.Y + (size_t)t * P.y_t_stride + col);
            }
            __syncthreads();                                         // pass 3 has read E: the next pass 1 may overwrite it
        }
    }
    if (yold != nullptr) {                                           // the CTA's last item
#pragma unroll 1
        for (int pt = 0; pt < 12; ++pt) store_point(pt);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(*reinterpret_cast<volatile uint32_t *>(&tmem_slot), C::TMEM_COLS);
    }
}

}  // namespace mwax
