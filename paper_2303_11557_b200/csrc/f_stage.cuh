// f_stage.cuh — F stage: int8 complex voltages -> FFT -> keep/centre-order -> scale -> fp16, written already
// corner-turned into the X stage's operand layout Y[p][t][input][re,im] (no separate transpose pass).
//
// PAPER.md §2.5, §2.5.1 L264 (promote 8-bit to float, FFT), L274 (transpose), L290/L611 (centre order,
// keep); DESIGN.md §5.1.
//
// Generic kernel (any N = 2^a 5^b): one CTA transforms one frame of G adjacent inputs with a Stockham autosort
// FFT in shared memory, radix 4/2/5 passes, fp32.  The G transforms are interleaved in shared memory
// ([index][g], g fastest) so that a warp's accesses are conflict free and the final store writes G*4
// contiguous bytes per (channel, time) row.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>

namespace mwax {

struct FParams {
    const int8_t *volt;      // [input][row_pitch samples][re,im]
    long long row_pitch;     // samples
    long long sample0;       // first sample of this dump in every row
    int n_inputs, N, K, T;
    int G;                   // inputs per CTA
    int frames_per_cta;      // consecutive frames one CTA of the power-of-two kernel walks over
    int n_pass;
    int radix[16];
    int vec_ok;              // 16-byte loads allowed
    const float2 *tw;        // [N] exp(-2 pi i m / N)
    const unsigned *swcode;  // N = 6400 three-pass kernel, K == N: [c = k mod 400] 2 bits per k3 = k / 400: 0 -> 1, 1 -> sqrt(1/2), 2 -> 0
    const float *sw;         // [K] per-position factor sqrt(w_p): 1, sqrt(1/2) on a shared edge, 0 for excluded DC
    float in_scale;          // s: power-of-two F-stage scale (keeps fp16 in range)
    int chan_scale;          // 0 when every sw[p] == 1
    // fractional-delay / phase correction (PAPER.md 2.5.1 L266-272): entry (input i, frame f) at i * d_stride + f; the
    // kernel's frame t is table frame frame0 + t.  NULL = zero.  Applied only by the DELAY kernel variants.
    const float *delay;      // samples
    const float *phase;      // radians
    long long d_stride;
    int frame0;
    __half2 *Y;              // [K][T][pitch2]
    int pitch2;              // half2 (complex) elements per Y row
    unsigned y_p_stride, y_t_stride;   // half2 elements between channel positions / between spectra (N = 6400 kernel)
    // Register kernels (N = 64 .. 512) only: their two small tables travel in the KERNEL-PARAMETER constant bank, so that the
    // warp-uniform reads of them are constant-cache loads and not wavefronts of the L1 data pipe, the busiest unit of those
    // kernels (profiles/r2_ncu_full.md).  twc[r * R1 + k1] = W_N^{r k1} (R1 = 8 for N <= 128, else 16); swc[p] = sw[p].
    float2 twc[512];
    float swc[512];
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// Packed fp32 pairs (sm_100 add/sub/fma .f32x2 -> FADD2 / FFMA2): one issue slot for the real and the imaginary part.
// The F kernels are issue bound, not FP32-lane bound (profiles/r1_ncu_full.md), so complex adds and subtractions, which
// are most of an FFT's instructions, go through these.  Same IEEE round-to-nearest results as the scalar forms.
__device__ __forceinline__ unsigned long long pack2(float2 a)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ float2 unpack2(unsigned long long r)
{
    float2 a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
// (a.x * f, a.y * f) in one issue slot
__device__ __forceinline__ float2 scale2(float2 a, float f)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(make_float2(f, f))));
    return unpack2(r);
}
// (a.x * b.x + c.x, a.y * b.y + c.y)
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)), "l"(pack2(c)));
    return unpack2(r);
}

// Delay/phase gain of one (input, frame): applying a delay of d samples multiplies signed bin u by
// exp(i (phase - 2 pi u d / N)) (shift theorem; reading Q19).  Kept in TURNS so that the argument of the
// fast sine/cosine is reduced exactly: turns(u) = pt + u * st, pt = phase / 2 pi, st = -d / N.
struct DelayGain {
    float pt, st;
};
__device__ __forceinline__ DelayGain load_delay_gain(const float *delay, const float *phase, long long idx, float inv_n)
{
    DelayGain gn;
    gn.pt = phase ? __ldg(phase + idx) * 0.15915494309189535f : 0.0f;
    gn.st = delay ? -__ldg(delay + idx) * inv_n : 0.0f;
    return gn;
}
__device__ __forceinline__ float2 apply_delay_gain(float2 v, DelayGain gn, int u)
{
    float tr = fmaf((float)u, gn.st, gn.pt);
    tr -= rintf(tr);                                                 // [-0.5, 0.5] turns
    float sn, cs;
    __sincosf(tr * 6.283185307179586f, &sn, &cs);
    return make_float2(fmaf(v.x, cs, -v.y * sn), fmaf(v.x, sn, v.y * cs));
}

// The gain along a run of bins u0, u0 + du, u0 + 2 du, ... is a geometric sequence: the register kernels take the sine
// and cosine once per run (delay_gain_at) and once per (input, frame) for the ratio (delay_gain_at with pt = 0) and walk
// the run with one complex multiply per bin.  Runs are 8 bins long (16 at most), so the walk adds a few 1e-7 of error;
// round 1's sine + cosine per bin kept the quarter-rate XU pipe busier than the FFT kept the FMA pipe.
__device__ __forceinline__ float2 delay_gain_at(float pt, float st, int u)
{
    float tr = fmaf((float)u, st, pt);
    tr -= rintf(tr);                                                 // [-0.5, 0.5] turns, exact
    float sn, cs;
    __sincosf(tr * 6.283185307179586f, &sn, &cs);
    return make_float2(cs, sn);
}

// y_k = sum_j x_j w_R^{jk}, forward (w_R = exp(-2 pi i / R))
template <int R>
__device__ __forceinline__ void butterfly(float2 (&x)[R]);

template <>
__device__ __forceinline__ void butterfly<2>(float2 (&x)[2])
{
    const float2 a = x[0], b = x[1];
    x[0] = cadd(a, b);
    x[1] = csub(a, b);
}
template <>
__device__ __forceinline__ void butterfly<4>(float2 (&x)[4])
{
    const float2 a = cadd(x[0], x[2]);
    const float2 b = csub(x[0], x[2]);
    const float2 c = cadd(x[1], x[3]);
    const float2 d = csub(x[1], x[3]);
    x[0] = cadd(a, c);
    x[2] = csub(a, c);
    x[1] = make_float2(b.x + d.y, b.y - d.x);   // b - i d
    x[3] = make_float2(b.x - d.y, b.y + d.x);   // b + i d
}
template <>
__device__ __forceinline__ void butterfly<5>(float2 (&x)[5])
{
    const float c1 = 0.30901699437494742f, c2 = -0.80901699437494742f;   // cos(2pi/5), cos(4pi/5)
    const float s1 = 0.95105651629515357f, s2 = 0.58778525229247313f;    // sin(2pi/5), sin(4pi/5)
    const float2 t1 = cadd(x[1], x[4]);
    const float2 t2 = cadd(x[2], x[3]);
    const float2 t3 = csub(x[1], x[4]);
    const float2 t4 = csub(x[2], x[3]);
    const float2 C1 = make_float2(c1, c1), C2 = make_float2(c2, c2), S1 = make_float2(s1, s1), S2 = make_float2(s2, s2);
    const float2 m1 = fma2(C2, t2, fma2(C1, t1, x[0]));
    const float2 m2 = fma2(C1, t2, fma2(C2, t1, x[0]));
    const float2 n1 = fma2(S2, t4, make_float2(s1 * t3.x, s1 * t3.y));
    const float2 n2 = fma2(make_float2(-s1, -s1), t4, make_float2(s2 * t3.x, s2 * t3.y));
    x[0] = cadd(cadd(x[0], t1), t2);
    x[1] = make_float2(m1.x + n1.y, m1.y - n1.x);   // m1 - i n1
    x[4] = make_float2(m1.x - n1.y, m1.y + n1.x);   // m1 + i n1
    x[2] = make_float2(m2.x + n2.y, m2.y - n2.x);
    x[3] = make_float2(m2.x - n2.y, m2.y + n2.x);
}

// One Stockham pass over G interleaved transforms:
//   y[q + s(R p + k)] = w_n^{p k} * sum_j x[q + s(p + m j)] w_R^{j k},  n = current sub-length, m = n/R, b = q + s p
template <int R>
__device__ __forceinline__ void stockham_pass(const float2 *__restrict__ src, float2 *__restrict__ dst, int N, int G,
                                              int n_cur, int s, const float2 *__restrict__ tw)
{
    const int nb = N / R;
    const int tw_step = N / n_cur;
    for (int w = threadIdx.x; w < nb * G; w += blockDim.x) {
        const int g = w % G, b = w / G;
        const int p = b / s, q = b - p * s;
        float2 x[R];
#pragma unroll
        for (int j = 0; j < R; ++j) x[j] = src[(b + j * nb) * G + g];
        butterfly<R>(x);
        const int o = q + s * R * p;
        dst[o * G + g] = x[0];
#pragma unroll
        for (int k = 1; k < R; ++k) dst[(o + s * k) * G + g] = cmul(x[k], __ldg(&tw[p * k * tw_step]));
    }
}

__global__ void __launch_bounds__(256) f_stage_generic_kernel(const FParams P)
{
    extern __shared__ float2 fbuf[];
    const int G = P.G, N = P.N;
    float2 *buf0 = fbuf, *buf1 = fbuf + (size_t)G * N;
    const int i0 = blockIdx.x * G;
    const int t = blockIdx.y;
    const long long s_off = P.sample0 + (long long)t * N;

    // ---- load + promote int8 -> fp32, transposing into [q][g]
    if (P.vec_ok) {
        const int nv = N / 8;
        for (int w = threadIdx.x; w < nv * G; w += blockDim.x) {
            const int g = w % G, v = w / G;
            const int i = i0 + g;
            int4 raw = make_int4(0, 0, 0, 0);
            if (i < P.n_inputs)
                raw = __ldg(reinterpret_cast<const int4 *>(P.volt + 2 * ((long long)i * P.row_pitch + s_off + 8 * v)));
            const int wd[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int x = wd[e];
                buf0[(8 * v + 2 * e) * G + g] = make_float2((float)(int8_t)(x & 0xff), (float)(int8_t)((x >> 8) & 0xff));
                buf0[(8 * v + 2 * e + 1) * G + g] =
                    make_float2((float)(int8_t)((x >> 16) & 0xff), (float)(int8_t)((x >> 24) & 0xff));
            }
        }
    } else {
        for (int w = threadIdx.x; w < N * G; w += blockDim.x) {
            const int g = w % G, qq = w / G;
            const int i = i0 + g;
            float2 v = make_float2(0.f, 0.f);
            if (i < P.n_inputs) {
                const int8_t *s = P.volt + 2 * ((long long)i * P.row_pitch + s_off + qq);
                v = make_float2((float)s[0], (float)s[1]);
            }
            buf0[qq * G + g] = v;
        }
    }
    __syncthreads();

    // ---- FFT passes
    float2 *src = buf0, *dst = buf1;
    int n_cur = N, s = 1;
    for (int ps = 0; ps < P.n_pass; ++ps) {
        const int R = P.radix[ps];
        if (R == 4) stockham_pass<4>(src, dst, N, G, n_cur, s, P.tw);
        else if (R == 2) stockham_pass<2>(src, dst, N, G, n_cur, s, P.tw);
        else stockham_pass<5>(src, dst, N, G, n_cur, s, P.tw);
        n_cur /= R;
        s *= R;
        float2 *tmp = src; src = dst; dst = tmp;
        __syncthreads();
    }

    // ---- keep the central K channels in signed order, scale, fp16 (round to nearest even), corner-turned store
    const int half = P.K / 2;
    for (int w = threadIdx.x; w < P.K * G; w += blockDim.x) {
        const int g = w % G, p = w / G;
        const int i = i0 + g;
        if (i >= P.n_inputs) continue;
        int k = p - half;
        if (k < 0) k += N;
        const float f = __ldg(&P.sw[p]) * P.in_scale;
        float2 v = src[k * G + g];
        if (P.delay || P.phase)
            v = apply_delay_gain(v, load_delay_gain(P.delay, P.phase, (long long)i * P.d_stride + P.frame0 + t, 1.0f / (float)N),
                                 p - half);
        P.Y[((long long)p * P.T + t) * P.pitch2 + i] = __floats2half2_rn(v.x * f, v.y * f);
    }
}

}  // namespace mwax
