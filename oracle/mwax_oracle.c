/*
 * mwax_oracle.c — float64 CPU oracle for the MWAX FX-correlator hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product (paper_2303_11557_b200/csrc)
 * shares no code, header, table or helper with it and never routes through it.
 *
 * It is the plain definition of what the path computes, written from PAPER.md (Morrison et al., "MWAX: A New
 * Correlator for the Murchison Widefield Array", arXiv 2303.11557) in the paper's order; every step cites the
 * passage it follows.  No blocking, fusion or reordering.  OpenMP is used only across independent outputs
 * (frames, channels); every individual output is accumulated sequentially in index order.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): brute-force DFT, numpy.fft on special cases, tone ->
 * bin/position, Parseval, Hermitian symmetry, phase closure, additivity, weight-table invariants stated in
 * the paper (L290-306), the K=8,F=2 worked table, Fig.14 data rates, common-signal correlation coefficient.
 * Steps 3b/3c/7/8 (delay, de-ripple gains, MWAX_ORDER, occupancy weights): shift theorem vs numpy.roll, numpy-scaled
 * channels and a numpy.fft-made passband ripple flattened by its inverse, Fig. 8 row order, numpy counts.
 * "parity unpinned" items (no instrument data in the container): which operand is conjugated (reading Q2),
 * absolute scale of the DFT and sum-vs-mean over time (Q1, Q5) — DESIGN.md §3.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define ORACLE_OK 0
#define ORACLE_ERR_ARG -1
#define ORACLE_ERR_NOMEM -2
#define ORACLE_ERR_OVERFLOW -3

#define AVG_CENTRE_SYMMETRIC 0
#define AVG_BLOCK 1
#define AVG_KEEP_DC 2 /* flag, OR-ed into the centre-symmetric mode: do NOT exclude the DC ultra-fine channel */

static const double TWO_PI = 6.283185307179586476925286766559;

/* w[m] = exp(-2*pi*i*m/N), m in [0,N): "twiddles from cos/sin(2*pi*((k*q) mod N)/N) in double" (reading Q1:
 * forward transform, negative exponent, unnormalised — the cuFFT forward convention the paper relies on,
 * PAPER.md L249, L264). */
static cplx *twiddle_table(int N)
{
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    if (!w) return NULL;
    for (int m = 0; m < N; ++m) {
        double a = TWO_PI * (double)m / (double)N;
        w[m] = cos(a) - I * sin(a);
    }
    return w;
}

/* Step 2 (definition): X[k] = sum_q f[q] * exp(-2*pi*i*k*q/N).  O(N^2). */
int mwax_oracle_dft_naive(int N, const double *in_ri, double *out_ri)
{
    if (N < 1 || !in_ri || !out_ri) return ORACLE_ERR_ARG;
    const cplx *f = (const cplx *)in_ri;
    cplx *X = (cplx *)out_ri;
    cplx *w = twiddle_table(N);
    if (!w) return ORACLE_ERR_NOMEM;
    for (int k = 0; k < N; ++k) {
        cplx acc = 0.0;
        for (int q = 0; q < N; ++q) acc += f[q] * w[(int)(((int64_t)k * q) % N)];
        X[k] = acc;
    }
    free(w);
    return ORACLE_OK;
}

static int smallest_prime_factor(int N)
{
    for (int r = 2; (int64_t)r * r <= N; ++r)
        if (N % r == 0) return r;
    return N;
}

/* Textbook recursive decimation-in-time Cooley-Tukey: split N = r*M by the smallest prime factor r,
 *   X[k] = sum_{a<r} w_N^{a*k} * DFT_M{ f[q*r + a] }[k mod M],
 * naive DFT at prime length.  wN is the table for the TOP-level length Ntop; w_N^m = wN[m * (Ntop/N)]. */
static void fft_rec(int N, const cplx *in, int stride, cplx *out, cplx *scratch, const cplx *wtop, int Ntop)
{
    const int step = Ntop / N;
    int r = smallest_prime_factor(N);
    if (r == N) { /* prime (or 1): the definition itself */
        for (int k = 0; k < N; ++k) {
            cplx acc = 0.0;
            for (int q = 0; q < N; ++q) acc += in[(size_t)q * stride] * wtop[(size_t)((k * q) % N) * step];
            out[k] = acc;
        }
        return;
    }
    const int M = N / r;
    /* sub-transforms of the r decimated sequences, results in scratch[a*M + k'] */
    for (int a = 0; a < r; ++a)
        fft_rec(M, in + (size_t)a * stride, stride * r, scratch + (size_t)a * M, out, wtop, Ntop);
    for (int k = 0; k < N; ++k) {
        cplx acc = 0.0;
        for (int a = 0; a < r; ++a)
            acc += wtop[(size_t)(((int64_t)a * k) % N) * step] * scratch[(size_t)a * M + (k % M)];
        out[k] = acc;
    }
}

/* NOTE on scratch use in fft_rec: the children write their results into `scratch + a*M` and use `out` as
 * THEIR scratch; `out` is only written by this level after all children are done, and a child's own scratch
 * region (length M inside `out`) never overlaps what a sibling returned (those live in `scratch`). */

int mwax_oracle_fft(int N, const double *in_ri, double *out_ri)
{
    if (N < 1 || !in_ri || !out_ri) return ORACLE_ERR_ARG;
    cplx *w = twiddle_table(N);
    cplx *scratch = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    if (!w || !scratch) { free(w); free(scratch); return ORACLE_ERR_NOMEM; }
    fft_rec(N, (const cplx *)in_ri, 1, (cplx *)out_ri, scratch, w, N);
    free(w);
    free(scratch);
    return ORACLE_OK;
}

/* Step 5: averaging weights W[c][p], C = K/F rows, K columns (readings Q4-Q8).
 *  - output channels are centre-symmetric: c0 = floor(C/2) is centred on DC (L296);
 *  - channel c is centred on signed bin u_c = (c - c0)*F; taps u_c + delta, cyclic mod K (Q8);
 *  - F odd: delta in [-(F-1)/2, (F-1)/2], weight 1; F even: F+1 taps, the two outermost weighted 0.5 (L298);
 *  - F > 1: the DC ultra-fine channel is excluded from the centre channel and that channel re-scaled by
 *    F/(F-1) (L290-294; Q6, Q7);
 *  - finally a mean: all weights divided by F (Q5).
 *  BLOCK mode (legacy adjacent grouping, Fig 6a): W[c][p] = 1/F for p in [cF,(c+1)F).
 *  AVG_KEEP_DC (flag on the centre-symmetric mode; SURVEY.md 8(b) MWAX_OPT_DC_EXCLUDE = 0): L290-294 describe the
 *  exclusion as something the averaging step DOES ("That centre ultra-fine channel is excluded ... and the output
 *  re-scaled accordingly"); with the flag the step is left out: the DC tap keeps weight 1 and the centre channel is a
 *  plain mean like every other channel (no F/(F-1)).
 *  Position p <-> signed bin u = p - floor(K/2) (step 3). */
int mwax_oracle_weights(int K, int F, int mode, double *W)
{
    if (K < 1 || F < 1 || K % F != 0 || !W) return ORACLE_ERR_ARG;
    const int C = K / F;
    memset(W, 0, sizeof(double) * (size_t)C * K);
    if (mode == AVG_BLOCK) {
        for (int c = 0; c < C; ++c)
            for (int p = c * F; p < (c + 1) * F; ++p) W[(size_t)c * K + p] = 1.0 / F;
        return ORACLE_OK;
    }
    if (mode != AVG_CENTRE_SYMMETRIC && mode != (AVG_CENTRE_SYMMETRIC | AVG_KEEP_DC)) return ORACLE_ERR_ARG;
    const int dc_exclude = !(mode & AVG_KEEP_DC);
    const int c0 = C / 2, half = K / 2;
    for (int c = 0; c < C; ++c) {
        const int uc = (c - c0) * F;
        const int dmax = (F % 2 == 1) ? (F - 1) / 2 : F / 2;
        for (int delta = -dmax; delta <= dmax; ++delta) {
            double wt = 1.0;
            if (F % 2 == 0 && (delta == -dmax || delta == dmax)) wt = 0.5;
            int u = uc + delta;
            int p = ((u + half) % K + K) % K;
            if (dc_exclude && F > 1 && c == c0 && delta == 0) wt = 0.0; /* DC excluded */
            W[(size_t)c * K + p] += wt;
        }
        if (dc_exclude && F > 1 && c == c0)
            for (int p = 0; p < K; ++p) W[(size_t)c * K + p] *= (double)F / (double)(F - 1);
        for (int p = 0; p < K; ++p) W[(size_t)c * K + p] /= (double)F;
    }
    return ORACLE_OK;
}

/* Steps 1-3 for a selection of inputs and one dump:
 *  1. frame t of input i: f[q] = x_i[(dump*T + t)*N + q], contiguous, no window;
 *  2. forward DFT of each frame (L247-249, L264); naive for N <= 64, recursive FFT otherwise;
 *  3. keep the K channels centred on DC in ascending signed frequency: u in [-floor(K/2), ceil(K/2)),
 *     Y[p] = X[u mod N], p = u + floor(K/2) (L290 centre-symmetric; L611 discard the rest).
 * volt: [input][row_pitch samples][re,im] int8.  Y: [K][T][n_sel] complex double. */
int mwax_oracle_spectra(int n_sel, const int *sel, int N, int K, int T, int dump, const int8_t *volt,
                        int64_t row_pitch, double *Y_ri)
{
    if (n_sel < 1 || !sel || N < 1 || K < 1 || K > N || T < 1 || dump < 0 || !volt || !Y_ri) return ORACLE_ERR_ARG;
    cplx *Y = (cplx *)Y_ri;
    cplx *w = twiddle_table(N);
    if (!w) return ORACLE_ERR_NOMEM;
    int err = ORACLE_OK;
#pragma omp parallel
    {
        cplx *f = (cplx *)malloc(sizeof(cplx) * (size_t)N);
        cplx *X = (cplx *)malloc(sizeof(cplx) * (size_t)N);
        cplx *scratch = (cplx *)malloc(sizeof(cplx) * (size_t)N);
        if (!f || !X || !scratch) {
#pragma omp atomic write
            err = ORACLE_ERR_NOMEM;
        } else {
#pragma omp for collapse(2) schedule(static)
            for (int s = 0; s < n_sel; ++s) {
                for (int t = 0; t < T; ++t) {
                    const int8_t *x = volt + 2 * ((int64_t)sel[s] * row_pitch + ((int64_t)dump * T + t) * N);
                    for (int q = 0; q < N; ++q) f[q] = (double)x[2 * q] + I * (double)x[2 * q + 1];
                    if (N <= 64) {
                        for (int k = 0; k < N; ++k) {
                            cplx acc = 0.0;
                            for (int q = 0; q < N; ++q) acc += f[q] * w[(k * q) % N];
                            X[k] = acc;
                        }
                    } else {
                        fft_rec(N, f, 1, X, scratch, w, N);
                    }
                    for (int p = 0; p < K; ++p) {
                        int u = p - K / 2;
                        int k = ((u % N) + N) % N;
                        Y[((size_t)p * T + t) * n_sel + s] = X[k];
                    }
                }
            }
        }
        free(f);
        free(X);
        free(scratch);
    }
    free(w);
    return err;
}

/* Step 3b (PAPER.md 2.5.1 L266-272, 2.4.1 L221, 4.3 L585): fractional-delay / phase
 * correction.  "any remaining fractional sample delay components can be applied by multiplying the frequency-domain
 * samples of each signal path by a phase gradient ... gradients can differ in both their slope and phase offset.
 * The slopes depend only on the delays to be applied, while the phase offsets [are supplied per path]"; one value
 * per signal path per frame ("5 ms update rate", 1600 values per 8 s at N = 6400).  Reading Q19:
 * APPLYING a delay of d samples to a signal multiplies bin u of its spectrum by exp(-2 pi i u d / N) (shift
 * theorem, forward transform of reading Q1); the phase offset phi (radians) multiplies by exp(+i phi):
 *     Y[p][t][s] *= exp(i * (phase[i][f] - 2 pi u d[i][f] / N)),  u = p - floor(K/2),  i = sel[s],  f = dump*T + t.
 * The paper takes the gains from a pre-computed look-up table; here they are computed directly (cos/sin in double).
 * delay, phase: [n_inputs][row_stride] doubles (NULL = all zero). */
int mwax_oracle_apply_delays(int n_sel, const int *sel, int N, int K, int T, int dump, const double *delay,
                             const double *phase, int64_t row_stride, double *Y_ri)
{
    if (n_sel < 1 || !sel || N < 1 || K < 1 || K > N || T < 1 || dump < 0 || !Y_ri) return ORACLE_ERR_ARG;
    cplx *Y = (cplx *)Y_ri;
#pragma omp parallel for schedule(static)
    for (int p = 0; p < K; ++p) {
        const int u = p - K / 2;
        for (int t = 0; t < T; ++t)
            for (int s = 0; s < n_sel; ++s) {
                const int64_t o = (int64_t)sel[s] * row_stride + (int64_t)dump * T + t;
                const double d = delay ? delay[o] : 0.0, ph = phase ? phase[o] : 0.0;
                const double th = ph - TWO_PI * (double)u * d / (double)N;
                Y[((size_t)p * T + t) * n_sel + s] *= cos(th) + I * sin(th);
            }
    }
    return ORACLE_OK;
}

/* Step 3c ("PFB de-ripple magnitude"; PAPER.md 4.2 L561-567): the gain table of the
 * fractional-delay stage "could be combined with a spectral magnitude response that represents the inverse of the
 * receiver PFB's passband response.  As the delays are applied, the spectral samples will then simultaneously be
 * magnitude-adjusted to provide a flattened overall frequency response."  One real, non-negative magnitude per kept
 * fine channel, the same for every signal path (one passband response; per-receiver-type tables are "not currently
 * supported", L571) and every frame (reading Q23):
 *     Y[p][t][s] *= gain[p],   p = channel position of step 3 (ascending signed frequency, DC at floor(K/2)). */
int mwax_oracle_apply_channel_gains(int n_sel, int K, int T, const double *gain, double *Y_ri)
{
    if (n_sel < 1 || K < 1 || T < 1 || !gain || !Y_ri) return ORACLE_ERR_ARG;
    cplx *Y = (cplx *)Y_ri;
    for (int p = 0; p < K; ++p)
        for (int t = 0; t < T; ++t)
            for (int s = 0; s < n_sel; ++s) Y[((size_t)p * T + t) * n_sel + s] *= gain[p];
    return ORACLE_OK;
}

/* Step 4: R[p][a(a+1)/2 + b] = sum_{t<T} Y_a[p][t] * conj(Y_b[p][t]) for all a >= b (autos included):
 * "cross-multiply every input pair", summed (not averaged) over the integration
 * (L280; reading Q5).  Direct per-pair multiply-accumulate.  Reading Q2: the SECOND index is conjugated. */
int mwax_oracle_correlate(int n_sel, int K, int T, const double *Y_ri, double *R_ri)
{
    if (n_sel < 1 || K < 1 || T < 1 || !Y_ri || !R_ri) return ORACLE_ERR_ARG;
    const cplx *Y = (const cplx *)Y_ri;
    cplx *R = (cplx *)R_ri;
    const size_t B = (size_t)n_sel * (n_sel + 1) / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int p = 0; p < K; ++p) {
        for (int a = 0; a < n_sel; ++a) {
            for (int b = 0; b <= a; ++b) {
                cplx acc = 0.0;
                for (int t = 0; t < T; ++t) {
                    const cplx *row = Y + ((size_t)p * T + t) * n_sel;
                    acc += row[a] * conj(row[b]);
                }
                R[(size_t)p * B + (size_t)a * (a + 1) / 2 + b] = acc;
            }
        }
    }
    return ORACLE_OK;
}

/* Steps 5-6: V[c][bl] = sum_p W[c][p] * R[p][bl], then Im V_aa := 0 exactly for autos
 * (reading Q13; L475 reports tiny non-zero values from xGPU where exactly zero was predicted). */
int mwax_oracle_average(int n_sel, int K, int F, int mode, const double *R_ri, double *V_ri)
{
    if (n_sel < 1 || K < 1 || F < 1 || K % F != 0 || !R_ri || !V_ri) return ORACLE_ERR_ARG;
    const cplx *R = (const cplx *)R_ri;
    cplx *V = (cplx *)V_ri;
    const int C = K / F;
    const size_t B = (size_t)n_sel * (n_sel + 1) / 2;
    double *W = (double *)malloc(sizeof(double) * (size_t)C * K);
    if (!W) return ORACLE_ERR_NOMEM;
    int rc = mwax_oracle_weights(K, F, mode, W);
    if (rc != ORACLE_OK) { free(W); return rc; }
#pragma omp parallel for schedule(static)
    for (int c = 0; c < C; ++c) {
        for (size_t bl = 0; bl < B; ++bl) {
            cplx acc = 0.0;
            for (int p = 0; p < K; ++p) {
                double wt = W[(size_t)c * K + p];
                if (wt != 0.0) acc += wt * R[(size_t)p * B + bl];
            }
            V[(size_t)c * B + bl] = acc;
        }
        for (int a = 0; a < n_sel; ++a) {
            size_t bl = (size_t)a * (a + 1) / 2 + a;
            V[(size_t)c * B + bl] = creal(V[(size_t)c * B + bl]);
        }
    }
    free(W);
    return ORACLE_OK;
}

/* Whole float path for one dump and a selection of inputs (steps 1-6 in order).
 * vis: [C][n_sel(n_sel+1)/2][re,im] float64; pair (a,b), a >= b, refers to inputs sel[a], sel[b].
 * The _delay form inserts step 3b between steps 3 and 4, the _gain form steps 3b and 3c. */
int mwax_oracle_fx_gain(int n_sel, const int *sel, int N, int K, int T, int F, int mode, int dump,
                        const int8_t *volt, int64_t row_pitch, const double *delay, const double *phase,
                        int64_t row_stride, const double *gain, double *vis_ri)
{
    if (n_sel < 1 || K < 1 || F < 1 || K % F != 0 || T < 1) return ORACLE_ERR_ARG;
    const size_t B = (size_t)n_sel * (n_sel + 1) / 2;
    double *Y = (double *)malloc(sizeof(double) * 2 * (size_t)K * T * n_sel);
    double *R = (double *)malloc(sizeof(double) * 2 * (size_t)K * B);
    if (!Y || !R) { free(Y); free(R); return ORACLE_ERR_NOMEM; }
    int rc = mwax_oracle_spectra(n_sel, sel, N, K, T, dump, volt, row_pitch, Y);
    if (rc == ORACLE_OK && (delay || phase))
        rc = mwax_oracle_apply_delays(n_sel, sel, N, K, T, dump, delay, phase, row_stride, Y);
    if (rc == ORACLE_OK && gain) rc = mwax_oracle_apply_channel_gains(n_sel, K, T, gain, Y);
    if (rc == ORACLE_OK) rc = mwax_oracle_correlate(n_sel, K, T, Y, R);
    if (rc == ORACLE_OK) rc = mwax_oracle_average(n_sel, K, F, mode, R, vis_ri);
    free(Y);
    free(R);
    return rc;
}

int mwax_oracle_fx_delay(int n_sel, const int *sel, int N, int K, int T, int F, int mode, int dump,
                         const int8_t *volt, int64_t row_pitch, const double *delay, const double *phase,
                         int64_t row_stride, double *vis_ri)
{
    return mwax_oracle_fx_gain(n_sel, sel, N, K, T, F, mode, dump, volt, row_pitch, delay, phase, row_stride, NULL, vis_ri);
}

int mwax_oracle_fx(int n_sel, const int *sel, int N, int K, int T, int F, int mode, int dump,
                   const int8_t *volt, int64_t row_pitch, double *vis_ri)
{
    return mwax_oracle_fx_delay(n_sel, sel, N, K, T, F, mode, dump, volt, row_pitch, NULL, NULL, 0, vis_ri);
}

/* Step 7 (PAPER.md 2.7 L318-326, Fig. 8, Fig. 9): MWAX_ORDER,
 * "(slowest-to-fastest changing): [time][baseline][channel][polarisation]", baselines listed as antA <= antB row by
 * row (0-0, 0-1, ..., 0-(n-1), 1-1, ...), polarisation products xx, xy, yx, yy, each value complex.
 * Readings: Q20 signal path i = 2*tile + pol with pol x = 0, y = 1 (the xGPU input order
 * "[tile][polarisation]", L274); Q21 element (antA, antB, ch, pq) = sum X_{antA,p} * conj(X_{antB,q}) -- the
 * first-named antenna unconjugated, as in step 4 (Q2; which antenna the instrument conjugates is unpinned).
 * With the native packed triangle V[ch][i(i+1)/2 + j] (i >= j) that is V[i][j] when i >= j, else conj(V[j][i]).
 * in:  V  [C][n(n+1)/2] complex double, n = 2*n_tiles signal paths.
 * out: M  [n_tiles(n_tiles+1)/2][C][4] complex double;  W [n_tiles(n_tiles+1)/2][4] weights, all 1.0 (L328: "these
 * weights are not utilised and all values are set to 1.0"). */
int mwax_oracle_mwax_order(int n_tiles, int C, const double *V_ri, double *M_ri, double *W)
{
    if (n_tiles < 1 || C < 1 || !V_ri || !M_ri) return ORACLE_ERR_ARG;
    const cplx *V = (const cplx *)V_ri;
    cplx *M = (cplx *)M_ri;
    const size_t n = 2 * (size_t)n_tiles, B = n * (n + 1) / 2;
    size_t row = 0;
    for (int a = 0; a < n_tiles; ++a)
        for (int b = a; b < n_tiles; ++b, ++row)
            for (int ch = 0; ch < C; ++ch)
                for (int p = 0; p < 2; ++p)
                    for (int q = 0; q < 2; ++q) {
                        const size_t i = 2 * (size_t)a + p, j = 2 * (size_t)b + q;
                        const cplx v = (i >= j) ? V[(size_t)ch * B + i * (i + 1) / 2 + j]
                                                : conj(V[(size_t)ch * B + j * (j + 1) / 2 + i]);
                        M[(row * C + ch) * 4 + 2 * p + q] = v;
                    }
    if (W)
        for (size_t r = 0; r < row * 4; ++r) W[r] = 1.0;
    return ORACLE_OK;
}

/* Step 8 (PAPER.md 4.1 L557-559, 2.4.2 L225, 2.6 L288): visibility weights = "the fraction of
 * the integration time for that visibility set that contained fully populated 50 ms sub-blocks in both signal paths
 * for that baseline/polarisation", from the zeroing flags (1 = that sub-block of that signal path was zeroed), and the
 * optional normalisation "such that missing packets do not cause variations in visibility magnitudes".
 * Reading Q22: weight(antA, antB, pq) = (1/S) * #{s : both paths valid in sub-block s}; normalising divides the
 * visibility by its weight; a weight of 0 leaves the (necessarily zero) visibility untouched.
 * flags: [2*n_tiles][S] bytes.  W: [n_tiles(n_tiles+1)/2][4].  M (optional, normalised in place): [rows][C][4] complex. */
int mwax_oracle_occupancy(int n_tiles, int S, const uint8_t *flags, int C, int normalise, double *W, double *M_ri)
{
    if (n_tiles < 1 || S < 1 || !flags || !W) return ORACLE_ERR_ARG;
    cplx *M = (cplx *)M_ri;
    size_t row = 0;
    for (int a = 0; a < n_tiles; ++a)
        for (int b = a; b < n_tiles; ++b, ++row)
            for (int p = 0; p < 2; ++p)
                for (int q = 0; q < 2; ++q) {
                    const uint8_t *fa = flags + (size_t)(2 * a + p) * S, *fb = flags + (size_t)(2 * b + q) * S;
                    int both = 0;
                    for (int sb = 0; sb < S; ++sb) both += (!fa[sb] && !fb[sb]);
                    const double w = (double)both / (double)S;
                    W[row * 4 + 2 * p + q] = w;
                    if (normalise && M && w > 0.0)
                        for (int ch = 0; ch < C; ++ch) M[(row * C + ch) * 4 + 2 * p + q] /= w;
                }
    return ORACLE_OK;
}

/* Integer X-only path (BASELINE.json configs[1]; the same contraction as step 4 on pre-channelised int8
 * samples z = a + ib, layout [chan][time][input][re,im]):
 *   Re V_ab = sum_t (a_a a_b + b_a b_b),  Im V_ab = sum_t (b_a a_b - a_a b_b)      (z_a * conj(z_b))
 * accumulated in int64, checked to fit int32, written as int32 [chan][a(a+1)/2+b][re,im]. */
int mwax_oracle_xcorr_i8(int n_sel, const int *sel, int n_inputs, int n_chan, int n_time, const int8_t *z,
                         int32_t *vis)
{
    if (n_sel < 1 || !sel || n_inputs < 1 || n_chan < 1 || n_time < 1 || !z || !vis) return ORACLE_ERR_ARG;
    const size_t B = (size_t)n_sel * (n_sel + 1) / 2;
    int err = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int c = 0; c < n_chan; ++c) {
        for (int a = 0; a < n_sel; ++a) {
            for (int b = 0; b <= a; ++b) {
                int64_t re = 0, im = 0;
                for (int t = 0; t < n_time; ++t) {
                    const int8_t *row = z + 2 * (((int64_t)c * n_time + t) * n_inputs);
                    int64_t ar = row[2 * sel[a]], ai = row[2 * sel[a] + 1];
                    int64_t br = row[2 * sel[b]], bi = row[2 * sel[b] + 1];
                    re += ar * br + ai * bi;
                    im += ai * br - ar * bi;
                }
                if (re > INT32_MAX || re < INT32_MIN || im > INT32_MAX || im < INT32_MIN) {
#pragma omp atomic write
                    err = ORACLE_ERR_OVERFLOW;
                }
                size_t o = 2 * ((size_t)c * B + (size_t)a * (a + 1) / 2 + b);
                vis[o] = (int32_t)re;
                vis[o + 1] = (int32_t)im;
            }
        }
    }
    return err;
}

#ifdef _OPENMP
#include <omp.h>
int mwax_oracle_threads(void) { return omp_get_max_threads(); }
/* timing infrastructure only (bench.py's single-thread run of config C1); no arithmetic depends on it */
void mwax_oracle_set_threads(int n) { if (n >= 1) omp_set_num_threads(n); }
#else
int mwax_oracle_threads(void) { return 1; }
void mwax_oracle_set_threads(int n) { (void)n; }
#endif
