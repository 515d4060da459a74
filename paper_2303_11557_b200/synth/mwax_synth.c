/*
 * mwax_synth.c — seeded, counter-based generator of synthetic MWA-like voltages.
 *
 * This module holds NONE of the correlator's arithmetic (no DFT, no cross-multiply, no averaging).
 * It only draws numbers.  Both the float64 oracle (oracle/) and the CUDA path (csrc/) are fed the
 * bytes it writes; neither of them includes or links it.
 *
 * Stand-in for the paper's telescope data (8-bit complex samples; L260: 1.28 MSPS per
 * coarse channel; L527: 512 signal paths "manufactured by duplicating signal paths").  Recipe: DESIGN.md §4.
 *
 * Every value is a pure function of (seed, stream, coarse, input, sample), so any sub-range can be
 * regenerated independently and generation parallelises over host threads.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>

#define SYNTH_STREAM_NOISE  1u   /* g_i[m]  : independent per input             */
#define SYNTH_STREAM_COMMON 2u   /* s[m]    : shared by all inputs of a coarse  */
#define SYNTH_STREAM_UNIF   3u   /* uniform integers, independent per input     */
#define SYNTH_STREAM_USHARE 4u   /* uniform integers, shared component          */

static inline uint64_t splitmix64(uint64_t x)
{
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

/* one 64-bit draw per (seed, stream, coarse, input, index) */
static inline uint64_t draw(uint64_t seed, uint32_t stream, uint32_t coarse, uint32_t input, uint64_t index)
{
    uint64_t h = splitmix64(seed ^ (0xA5A5A5A5ull * stream));
    h = splitmix64(h ^ (((uint64_t)coarse << 32) | input));
    return splitmix64(h ^ index);
}

/* two independent standard normals from one draw (Box-Muller on two 32-bit halves) */
static inline void normal_pair(uint64_t r, double *z0, double *z1)
{
    const double two_pi = 6.283185307179586476925286766559;
    double u1 = ((double)(uint32_t)(r >> 32) + 1.0) * (1.0 / 4294967296.0); /* (0,1] */
    double u2 = ((double)(uint32_t)r) * (1.0 / 4294967296.0);               /* [0,1) */
    double rad = sqrt(-2.0 * log(u1));
    *z0 = rad * cos(two_pi * u2);
    *z1 = rad * sin(two_pi * u2);
}

static inline int8_t clip_round(double v, int lim)
{
    double r = rint(v);
    if (r > lim) r = lim;
    if (r < -lim) r = -lim;
    return (int8_t)r;
}

/*
 * Gaussian voltages: out[(i - input0) * row_pitch + (m - sample0)][re,im], int8,
 *   x_i[m] = clip(rint( sqrt(1-rho)*g_i[m] + sqrt(rho)*s[m] + sum_tones a*exp(2*pi*j*(k*m/N + mult*i/n_total)) ), +-127)
 * per component; g_i, s complex Gaussians with per-component standard deviation sigma.
 * Tones: tone_bin[k] (signed integer DFT bin for frame length tone_nfft), tone_amp[k], tone_phase_mult[k].
 */
void mwax_synth_gauss(uint64_t seed, uint32_t coarse,
                      int input0, int n_gen, int n_total,
                      int64_t sample0, int64_t n_samples, int64_t row_pitch,
                      double sigma, double rho,
                      int n_tones, const int *tone_bin, const double *tone_amp, const int *tone_phase_mult,
                      int tone_nfft, int8_t *out)
{
    const double two_pi = 6.283185307179586476925286766559;
    const double a_noise = sqrt(1.0 - rho) * sigma, a_common = sqrt(rho) * sigma;
    const int use_common = (rho != 0.0);
    /* the common signal s[m] is the same for every input: draw it once */
    double *cs = NULL;
    if (use_common) {
        cs = (double *)malloc(sizeof(double) * 2 * (size_t)n_samples);
        if (!cs) return;
#pragma omp parallel for schedule(static)
        for (int64_t mm = 0; mm < n_samples; ++mm)
            normal_pair(draw(seed, SYNTH_STREAM_COMMON, coarse, 0u, (uint64_t)(sample0 + mm)), &cs[2 * mm], &cs[2 * mm + 1]);
    }
#pragma omp parallel
    {
        /* per-input tone sum over one frame (tones are on integer bins, so they repeat every tone_nfft samples) */
        double *tt = (n_tones > 0) ? (double *)malloc(sizeof(double) * 2 * (size_t)tone_nfft) : NULL;
#pragma omp for schedule(dynamic, 1)
        for (int ii = 0; ii < n_gen; ++ii) {
            const int i = input0 + ii;
            if (tt) {
                for (int r = 0; r < tone_nfft; ++r) {
                    double re = 0.0, im = 0.0;
                    for (int k = 0; k < n_tones; ++k) {
                        int64_t km = ((int64_t)tone_bin[k] * r) % tone_nfft;
                        if (km < 0) km += tone_nfft;
                        int64_t ph_i = ((int64_t)tone_phase_mult[k] * i) % n_total;
                        double ph = two_pi * ((double)km / (double)tone_nfft + (double)ph_i / (double)n_total);
                        re += tone_amp[k] * cos(ph);
                        im += tone_amp[k] * sin(ph);
                    }
                    tt[2 * r] = re;
                    tt[2 * r + 1] = im;
                }
            }
            for (int64_t mm = 0; mm < n_samples; ++mm) {
                const int64_t m = sample0 + mm;
                double gr, gi;
                normal_pair(draw(seed, SYNTH_STREAM_NOISE, coarse, (uint32_t)i, (uint64_t)m), &gr, &gi);
                double re = a_noise * gr, im = a_noise * gi;
                if (use_common) {
                    re += a_common * cs[2 * mm];
                    im += a_common * cs[2 * mm + 1];
                }
                if (tt) {
                    const int r = (int)(m % tone_nfft);
                    re += tt[2 * r];
                    im += tt[2 * r + 1];
                }
                int8_t *o = out + 2 * ((int64_t)ii * row_pitch + mm);
                o[0] = clip_round(re, 127);
                o[1] = clip_round(im, 127);
            }
        }
        free(tt);
    }
    free(cs);
}

/*
 * Uniform integer voltages for the pre-channelised X-only path (BASELINE.json configs[1]):
 * out[chan][time][input][re,im] int8, re/im ~ U{-8..7}; inputs < n_shared add a shared U{-8..7}
 * component per (chan, time).
 */
void mwax_synth_uniform(uint64_t seed, int n_chan, int n_time, int n_inputs, int n_shared, int8_t *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int c = 0; c < n_chan; ++c) {
        for (int t = 0; t < n_time; ++t) {
            uint64_t rs = draw(seed, SYNTH_STREAM_USHARE, (uint32_t)c, 0u, (uint64_t)t);
            int sh_re = (int)(rs & 15u) - 8, sh_im = (int)((rs >> 4) & 15u) - 8;
            int8_t *o = out + 2 * (((int64_t)c * n_time + t) * n_inputs);
            for (int i = 0; i < n_inputs; ++i) {
                uint64_t r = draw(seed, SYNTH_STREAM_UNIF, (uint32_t)c, (uint32_t)i, (uint64_t)t);
                int re = (int)(r & 15u) - 8, im = (int)((r >> 4) & 15u) - 8;
                if (i < n_shared) { re += sh_re; im += sh_im; }
                o[2 * i] = (int8_t)re;
                o[2 * i + 1] = (int8_t)im;
            }
        }
    }
}
