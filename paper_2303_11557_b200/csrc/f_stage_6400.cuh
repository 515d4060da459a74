// f_stage_6400.cuh — F stage for the paper's own frame length N = 6400 = 80 x 80 (§2.5:
// "6400-point FFT", 200 Hz ultra-fine channels): a two-pass FFT whose 80-point sub-transforms live entirely in
// registers, with ONE shared-memory exchange between the passes.
//
//   n = 80 n1 + n2,  k = k1 + 80 k2:
//   X[k1 + 80 k2] = sum_{n2} W_80^{n2 k2} ( W_6400^{n2 k1} sum_{n1} x[80 n1 + n2] W_80^{n1 k1} )
//
// One CTA (320 threads) transforms one frame of G = 4 adjacent inputs; thread = (g = tid & 3, idx = tid >> 2).
//   pass 1  thread (g, n2) gathers its 80 stride-80 samples straight from global memory (int8 pairs, promoted in
//           registers), runs the 80-point FFT, multiplies by the pre-scaled inter-pass twiddles
//           tw2[k1][n2] = s W_6400^{n2 k1} (one table row read shared by the four g lanes) and writes the
//           exchange buffer E[g][k1][n2] (fp32; 4 x 80 x 81 float2 = 207 KB: the whole SM).
//   pass 2  thread (g, k1) reads E[g][k1][0..79], runs the 80-point FFT over n2 and stores fp16 results for bins
//           k1 + 80 k2 already corner-turned: lanes (g, 8 consecutive k1) write 8 rows x 16 bytes of
//           Y[p][t][input].  All 128 input groups of a frame run in the same wave of persistent CTAs, so the
//           eight 16-byte pieces of every 128-byte line meet in L2 before the line goes to HBM.
// Strides of E are padded (row 81, group 6484 float2) so both the pass-1 writes and the pass-2 reads are
// bank-conflict free for 64-bit accesses: index mod 16 = 4 g + idx + const.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>
#include "f_stage.cuh"
#include "f_stage_pow2.cuh"

namespace mwax {

// exp(-2 pi i m / 80), m = 0..60
__device__ __forceinline__ float2 w80(int m)
{
    switch (m) {
        case 0: return make_float2(1.000000000e+00f, 0.000000000e+00f);
        case 1: return make_float2(9.969173337e-01f, -7.845909573e-02f);
        case 2: return make_float2(9.876883406e-01f, -1.564344650e-01f);
        case 3: return make_float2(9.723699204e-01f, -2.334453639e-01f);
        case 4: return make_float2(9.510565163e-01f, -3.090169944e-01f);
        case 5: return make_float2(9.238795325e-01f, -3.826834324e-01f);
        case 6: return make_float2(8.910065242e-01f, -4.539904997e-01f);
        case 7: return make_float2(8.526401644e-01f, -5.224985647e-01f);
        case 8: return make_float2(8.090169944e-01f, -5.877852523e-01f);
        case 9: return make_float2(7.604059656e-01f, -6.494480483e-01f);
        case 10: return make_float2(7.071067812e-01f, -7.071067812e-01f);
        case 11: return make_float2(6.494480483e-01f, -7.604059656e-01f);
        case 12: return make_float2(5.877852523e-01f, -8.090169944e-01f);
        case 13: return make_float2(5.224985647e-01f, -8.526401644e-01f);
        case 14: return make_float2(4.539904997e-01f, -8.910065242e-01f);
        case 15: return make_float2(3.826834324e-01f, -9.238795325e-01f);
        case 16: return make_float2(3.090169944e-01f, -9.510565163e-01f);
        case 17: return make_float2(2.334453639e-01f, -9.723699204e-01f);
        case 18: return make_float2(1.564344650e-01f, -9.876883406e-01f);
        case 19: return make_float2(7.845909573e-02f, -9.969173337e-01f);
        case 20: return make_float2(0.000000000e+00f, -1.000000000e+00f);
        case 21: return make_float2(-7.845909573e-02f, -9.969173337e-01f);
        case 22: return make_float2(-1.564344650e-01f, -9.876883406e-01f);
        case 23: return make_float2(-2.334453639e-01f, -9.723699204e-01f);
        case 24: return make_float2(-3.090169944e-01f, -9.510565163e-01f);
        case 25: return make_float2(-3.826834324e-01f, -9.238795325e-01f);
        case 26: return make_float2(-4.539904997e-01f, -8.910065242e-01f);
        case 27: return make_float2(-5.224985647e-01f, -8.526401644e-01f);
        case 28: return make_float2(-5.877852523e-01f, -8.090169944e-01f);
        case 29: return make_float2(-6.494480483e-01f, -7.604059656e-01f);
        case 30: return make_float2(-7.071067812e-01f, -7.071067812e-01f);
        case 31: return make_float2(-7.604059656e-01f, -6.494480483e-01f);
        case 32: return make_float2(-8.090169944e-01f, -5.877852523e-01f);
        case 33: return make_float2(-8.526401644e-01f, -5.224985647e-01f);
        case 34: return make_float2(-8.910065242e-01f, -4.539904997e-01f);
        case 35: return make_float2(-9.238795325e-01f, -3.826834324e-01f);
        case 36: return make_float2(-9.510565163e-01f, -3.090169944e-01f);
        case 37: return make_float2(-9.723699204e-01f, -2.334453639e-01f);
        case 38: return make_float2(-9.876883406e-01f, -1.564344650e-01f);
        case 39: return make_float2(-9.969173337e-01f, -7.845909573e-02f);
        case 40: return make_float2(-1.000000000e+00f, 0.000000000e+00f);
        case 41: return make_float2(-9.969173337e-01f, 7.845909573e-02f);
        case 42: return make_float2(-9.876883406e-01f, 1.564344650e-01f);
        case 43: return make_float2(-9.723699204e-01f, 2.334453639e-01f);
        case 44: return make_float2(-9.510565163e-01f, 3.090169944e-01f);
        case 45: return make_float2(-9.238795325e-01f, 3.826834324e-01f);
        case 46: return make_float2(-8.910065242e-01f, 4.539904997e-01f);
        case 47: return make_float2(-8.526401644e-01f, 5.224985647e-01f);
        case 48: return make_float2(-8.090169944e-01f, 5.877852523e-01f);
        case 49: return make_float2(-7.604059656e-01f, 6.494480483e-01f);
        case 50: return make_float2(-7.071067812e-01f, 7.071067812e-01f);
        case 51: return make_float2(-6.494480483e-01f, 7.604059656e-01f);
        case 52: return make_float2(-5.877852523e-01f, 8.090169944e-01f);
        case 53: return make_float2(-5.224985647e-01f, 8.526401644e-01f);
        case 54: return make_float2(-4.539904997e-01f, 8.910065242e-01f);
        case 55: return make_float2(-3.826834324e-01f, 9.238795325e-01f);
        case 56: return make_float2(-3.090169944e-01f, 9.510565163e-01f);
        case 57: return make_float2(-2.334453639e-01f, 9.723699204e-01f);
        case 58: return make_float2(-1.564344650e-01f, 9.876883406e-01f);
        case 59: return make_float2(-7.845909573e-02f, 9.969173337e-01f);
        case 60: return make_float2(0.000000000e+00f, 1.000000000e+00f);
        default: return make_float2(1.0f, 0.0f);
    }
}

__device__ __forceinline__ float2 mul_w80(float2 d, int m)
{
    if (m == 0) return d;
    if (m == 20) return make_float2(d.y, -d.x);                      // * (-i)
    if (m == 40) return make_float2(-d.x, -d.y);                     // * (-1)
    if (m == 60) return make_float2(-d.y, d.x);                      // * (+i)
    if (m == 10) {                                                   // * (1 - i)/sqrt(2)
        const float h = 0.70710678118654757f;
        return make_float2((d.x + d.y) * h, (d.y - d.x) * h);
    }
    if (m == 30) {                                                   // * (-1 - i)/sqrt(2)
        const float h = 0.70710678118654757f;
        return make_float2((d.y - d.x) * h, -(d.x + d.y) * h);
    }
    return cmul(d, w80(m));
}

// In-register 80-point forward DFT.  In: x[a][b] = sample index 16 a + b (a < 5, b < 16).
// Out: X[ka + 5 kb] is left in x[ka][bitrev4(kb)]  (ka < 5, kb < 16).
__device__ __forceinline__ void fft80(float2 (&x)[5][16])
{
#pragma unroll
    for (int b = 0; b < 16; ++b) {
        float2 v[5] = {x[0][b], x[1][b], x[2][b], x[3][b], x[4][b]};
        butterfly<5>(v);                                             // over a, output index ka
#pragma unroll
        for (int ka = 0; ka < 5; ++ka) x[ka][b] = mul_w80(v[ka], b * ka);   // W_80^{b ka}
    }
#pragma unroll
    for (int ka = 0; ka < 5; ++ka) fft_dif<16>(x[ka]);               // over b, output index kb (bit reversed)
}

struct F6400 {
    static constexpr int N = 6400, R = 80, G = 4;
    static constexpr int THREADS = R * G;                            // 320
    static constexpr int ROW = R + 1;                                // 81 float2 per k1 row
    static constexpr int GRP = R * ROW + 4;                          // 6484 float2 per input (mod 16 == 4)
    static constexpr int SMEM_BYTES = G * GRP * 8;                   // 207,488
};

// FULL : K == N (every bin kept)          SCALE : multiply by sw[p] (averaging weights folded into the F stage)
// TPT : 80-point transforms per thread and pass (1 -> 320 threads / 168 registers, 2 -> 160 threads / 255 registers)
template <bool FULL, bool SCALE, int TPT>
__global__ void __launch_bounds__(F6400::THREADS / TPT, 1) f_stage_6400_kernel(const FParams P)
{
    using C = F6400;
    extern __shared__ __align__(16) float2 f64ex[];
    const int g = threadIdx.x & 3;
    const int groups = (P.n_inputs + C::G - 1) / C::G;
    const int n_items = groups * P.T;
    const int half = P.K / 2;
    const unsigned chan_stride = (unsigned)P.T * (unsigned)P.pitch2; // half2 elements between channel positions

    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int t = item / groups;
        const int i = (item - t * groups) * C::G + g;
        const bool iok = i < P.n_inputs;

        // ---- pass 1: 80-point FFT over n1 of x[80 n1 + n2], n2 = idx
#pragma unroll 1
        for (int rep = 0; rep < TPT; ++rep) {
            const int idx = (threadIdx.x >> 2) + rep * (C::R / TPT);
            float2 *ew = f64ex + g * C::GRP + idx;                   // E[g][k1][n2 = idx]: + k1 * ROW
            const float2 *twp = P.tw2 + idx;                         // tw2[k1][n2 = idx]: + k1 * 80
            float2 x[5][16];
            const int8_t *src = P.volt + 2 * ((long long)(iok ? i : 0) * P.row_pitch + P.sample0 + (long long)t * C::N + idx);
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 16; ++b) {
                    const unsigned w = __ldg(reinterpret_cast<const unsigned short *>(src + 160 * (16 * a + b)));
                    x[a][b] = make_float2((float)(signed char)(w & 0xffu), (float)(signed char)(w >> 8));   // L264
                }
            if (!iok) {
#pragma unroll
                for (int a = 0; a < 5; ++a)
#pragma unroll
                    for (int b = 0; b < 16; ++b) x[a][b] = make_float2(0.f, 0.f);
            }
            fft80(x);
#pragma unroll
            for (int kb = 0; kb < 16; ++kb)
#pragma unroll
                for (int ka = 0; ka < 5; ++ka) {
                    const int k1 = ka + 5 * kb;
                    ew[k1 * C::ROW] = cmul(x[ka][bitrev(kb, 4)], __ldg(twp + k1 * C::R));
                }
        }
        __syncthreads();

        // ---- pass 2: 80-point FFT over n2 for k1 = idx; bins k = k1 + 80 k2
#pragma unroll 1
        for (int rep = 0; rep < TPT; ++rep) {
            const int idx = (threadIdx.x >> 2) + rep * (C::R / TPT);
            const float2 *er = f64ex + g * C::GRP + idx * C::ROW;    // E[g][k1 = idx][n2]: + n2
            float2 y[5][16];
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 16; ++b) y[a][b] = er[16 * a + b];
            fft80(y);
            if (iok) {
                if (FULL) {
                    // k2 < 40 <=> k < N/2: p = k + N/2, else p = k - N/2 (centre order)
                    __half2 *yp = P.Y + i + (size_t)t * P.pitch2 + (size_t)(idx + C::N / 2) * chan_stride;
                    __half2 *yn = P.Y + i + (size_t)t * P.pitch2 + (size_t)idx * chan_stride;
                    const float *swp = P.sw + idx;
#pragma unroll
                    for (int kb = 0; kb < 16; ++kb)
#pragma unroll
                        for (int ka = 0; ka < 5; ++ka) {
                            const int k2 = ka + 5 * kb;
                            float2 v = y[ka][bitrev(kb, 4)];
                            if (SCALE) {
                                const float f = __ldg(swp + ((k2 < 40) ? (C::N / 2 + C::R * k2) : (C::R * k2 - C::N / 2)));
                                v.x *= f;
                                v.y *= f;
                            }
                            __half2 *dst = (k2 < 40) ? yp + (size_t)(unsigned)(C::R * k2) * chan_stride
                                                     : yn + (size_t)(unsigned)(C::R * (k2 - 40)) * chan_stride;
                            *dst = __floats2half2_rn(v.x, v.y);
                        }
                } else {
#pragma unroll
                    for (int kb = 0; kb < 16; ++kb)
#pragma unroll
                        for (int ka = 0; ka < 5; ++ka) {
                            const int k = idx + C::R * (ka + 5 * kb);
                            const int u = (k < C::N / 2) ? k : k - C::N;         // signed bin
                            const int p = u + half;
                            if (p < 0 || p >= P.K) continue;                     // keep the central K channels (L611)
                            float2 v = y[ka][bitrev(kb, 4)];
                            if (SCALE) {
                                const float f = __ldg(&P.sw[p]);
                                v.x *= f;
                                v.y *= f;
                            }
                            P.Y[((size_t)p * P.T + t) * P.pitch2 + i] = __floats2half2_rn(v.x, v.y);
                        }
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace mwax
