/*
 * mwax_corr.h — C ABI of the B200-native MWAX FX-correlator hot path.
 *
 * What the library computes (PAPER.md = Morrison et al., "MWAX: A New Correlator for the Murchison
 * Widefield Array", arXiv 2303.11557; readings Q1-Q18 are listed in DESIGN.md §3):
 *
 *   F stage   PAPER.md §2.5, §2.5.1: every signal path's complex 8-bit voltage stream is cut
 *             into non-overlapping frames of n_fft samples and each frame is Fourier transformed (forward,
 *             unnormalised) into n_fft fine channels.  The n_keep channels centred on DC are kept, in
 *             ascending signed frequency (L290 centre-symmetric; §4.5 L611 discard the rest).
 *   X stage   §2.1, §2.5.2: for every fine channel, every pair of signal paths (autos
 *             included) is cross-multiplied, V_ij = sum_t X_i(t) * conj(X_j(t)), and accumulated over the
 *             integration time (t_int spectra, L280).
 *   Averaging §2.6: f_avg adjacent fine channels are averaged into one output channel with the
 *             paper's centre-symmetric grouping (the DC fine channel excluded and its channel re-scaled;
 *             f_avg+1 taps with half-weighted ends when f_avg is even), or plain adjacent blocks
 *             (MWAX_AVG_BLOCK, the legacy grouping of Fig. 6a).
 *
 * Everything runs in hand-written sm_100a kernels (no cuFFT, no xGPU, no CPU fallback).  All entry points
 * are plain C: pointers are DEVICE pointers unless the name says `_host`; sizes are in the units stated.
 * Calls return MWAX_OK (0) or a negative error code; nothing throws, aborts or prints.
 *
 * Threading/streams: all device work of a call is enqueued on `stream` (a cudaStream_t passed as void*;
 * NULL = the legacy default stream) and the call returns after enqueueing.  One call in flight per handle
 * (the handle owns a workspace); different handles may run on different streams and threads.
 * Devices: a handle belongs to the CUDA device that was current when it was created (any sm_100 device of the
 * process; the library is built for sm_100a only, other architectures get MWAX_ERR_ARCH).  Every call must be made
 * with that device current, otherwise it returns MWAX_ERR_INVALID_ARG without enqueueing anything.
 * The library reads no environment variables: every knob is an argument or a mwax_corr_set_option key below.
 */
#ifndef MWAX_CORR_H
#define MWAX_CORR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mwax_corr mwax_corr_t;   /* opaque FX plan + workspace */
typedef struct mwax_xcorr mwax_xcorr_t; /* opaque X-only integer plan */

enum {
    MWAX_OK = 0,
    MWAX_ERR_NULL = -1,        /* a required pointer was NULL                                   */
    MWAX_ERR_INVALID_ARG = -2, /* argument out of range (sizes < 1, misaligned pointer, ...)    */
    MWAX_ERR_UNSUPPORTED = -3, /* n_fft not 2^a*5^b or > 6400, n_keep > n_fft, f_avg !| n_keep  */
    MWAX_ERR_NOMEM = -4,       /* host or device allocation failed                              */
    MWAX_ERR_CUDA = -5,        /* a CUDA runtime/driver call failed; see mwax_corr_last_cuda_error */
    MWAX_ERR_ARCH = -6,        /* no CUDA device, or the current device is not sm_100           */
    MWAX_ERR_TOO_LARGE = -7    /* mwax_corr_process_static: spectra exceed the static workspace */
};

/* options for mwax_corr_set_option */
enum { MWAX_OPT_AVG_MODE = 1, MWAX_OPT_ACCUMULATE = 2, MWAX_OPT_DC_EXCLUDE = 3, MWAX_OPT_X_EDGE_RUNS = 4 };
enum { MWAX_AVG_CENTRE_SYMMETRIC = 0, MWAX_AVG_BLOCK = 1 };

/* ------------------------------------------------------------------------------------------------------
 * FX path (BASELINE.json north star).
 *
 * mwax_corr_create(n_inputs, n_fft, n_keep, t_int, f_avg)
 *   n_inputs  number of signal paths n (tiles x 2 polarisations), >= 1
 *   n_fft     frame / FFT length N; must be 2^a * 5^b, 1 <= N <= 6400 (the paper uses 6400, L264)
 *   n_keep    K <= N fine channels kept, centred on DC: signed bins u in [-floor(K/2), ceil(K/2)),
 *             output position p = u + floor(K/2)
 *   t_int     T >= 1 spectra summed into one integration (seconds never cross the ABI: T = t * 1.28e6 / N)
 *   f_avg     F >= 1 fine channels per output channel, F | K; C = K/F output channels
 * Returns a handle owning its tables and an fp16 workspace of mwax_corr_workspace_bytes() on the current
 * CUDA device, or NULL; the reason is then returned by mwax_corr_last_error() (thread-local).
 * ---------------------------------------------------------------------------------------------------- */
mwax_corr_t *mwax_corr_create(int n_inputs, int n_fft, int n_keep, int t_int, int f_avg);
int mwax_corr_last_error(void);

/* MWAX_OPT_AVG_MODE: averaging geometry; call before the first process().  Default MWAX_AVG_CENTRE_SYMMETRIC (L290).
 * MWAX_OPT_DC_EXCLUDE (1/0, default 1; centre-symmetric mode, f_avg > 1): "That centre ultra-fine channel
 *   is excluded ... and the output re-scaled accordingly".  With 1 the DC fine channel gets weight 0 in the centre output
 *   channel, which is multiplied by F/(F-1); with 0 the step is left out: the DC fine channel is averaged in like any
 *   other and the centre channel is a plain mean.  Rebuilds the small device tables (synchronous).
 * MWAX_OPT_X_EDGE_RUNS (default -1): schedule of the X stage when f_avg is even (see mwax_corr_x_edge_runs): -1 = the
 *   library decides from its cost model, 0 = never use the shared-edge schedule, r >= 1 = use it with r runs of adjacent
 *   output channels per tile (clamped to C) whenever the geometry allows it (even f_avg, centre-symmetric, t_int >= 64).
 *   A scheduling knob only: every setting computes the same sums (in a different fp32 order).
 * MWAX_OPT_ACCUMULATE (0/1, default 0): streaming integration (§2.5, §2.5.2:
 *   50 ms blocks aggregated into the integration).  With 1, process()/process_batch()/x_stage() ADD their result to
 *   what d_vis already holds, so an integration of any length is the sum of calls over its pieces (t_int = spectra per
 *   piece, e.g. 10 for one 50 ms block at n_fft = 6400) without keeping the voltages: first piece with 0, the rest
 *   with 1.  Sums of fp32 partial results; the pieces need not be equal in content but each has t_int spectra. */
int mwax_corr_set_option(mwax_corr_t *h, int key, int value);

/* Fractional-delay / phase correction (§2.5.1, §2.4.1, §4.3):
 * before cross-correlation every signal path's spectrum is multiplied by a phase gradient whose slope is the
 * fractional-sample delay to apply and by a phase offset, one pair of values per signal path per frame (the paper's
 * 5 ms cadence: 1600 values per 8 s at n_fft = 6400).  Signed bin u of frame f of input i is multiplied by
 *     exp(i * (phase[i][f] - 2 pi u delay[i][f] / n_fft))          (delay in samples, phase in radians;
 * applying a delay of d samples; reading Q19).  The gains are computed in the F kernel (no look-up table).
 *   d_delay, d_phase  DEVICE float tables, entry (coarse c, input i, frame f) at c*coarse_stride + i*row_stride + f;
 *                     frame f counts the frames of the row handed to process()/process_batch()/process_host()
 *                     (dump d uses frames d*T .. d*T+T-1).  Either may be NULL (= zeros); both NULL switches the
 *                     correction off.  Caller-owned; must stay valid while calls that use them are in flight.
 *   row_stride >= frames per row (T * n_dumps), else MWAX_ERR_INVALID_ARG (checked again by the process calls). */
int mwax_corr_set_delays(mwax_corr_t *h, const float *d_delay, const float *d_phase, size_t row_stride,
                         size_t coarse_stride);

/* Per-channel magnitude gains — "PFB de-ripple" (§4.2): the gain table of
 * the delay stage "could be combined with a spectral magnitude response that represents the inverse of the receiver
 * PFB's passband response", so that the spectra are "magnitude-adjusted to provide a flattened overall frequency
 * response".  Every spectral sample of kept channel position p (ascending signed frequency, DC at n_keep/2) of every
 * signal path and frame is multiplied by gain[p] before cross-correlation, so fine channel p's products carry
 * gain[p]^2 into the average (reading Q23).  Folded into the F kernels' per-channel factor: no extra pass.
 *   gain  HOST float [n_keep], each in [0, 4] (fp16 headroom), copied by the call; NULL switches the gains off.
 * Synchronous (rebuilds the small device tables); call between, not during, process calls.
 * MWAX_ERR_INVALID_ARG for a value outside [0, 4] or NaN. */
int mwax_corr_set_channel_gains(mwax_corr_t *h, const float *gain);

/* One integration:
 *   d_volt  in : int8 [n_inputs][T*N][re,im] — row i is signal path i's contiguous sample stream
 *                (PAPER.md L260), row pitch exactly T*N samples; two's-complement, -128 accepted.
 *                Must be 16-byte aligned.  mwax_corr_input_bytes() = n*T*N*2.
 *   d_vis   out: float [C][n(n+1)/2][re,im], baseline index i*(i+1)/2 + j for i >= j,
 *                V_ij = sum X_i conj(X_j); autos have Im == 0 exactly; sum (not mean) over time, weighted
 *                MEAN over the averaged fine channels; DFT unnormalised.  mwax_corr_output_bytes() = C*B*8.
 * Caller owns both buffers; they must stay valid until the stream has drained.
 */
int mwax_corr_process(mwax_corr_t *h, const int8_t *d_volt, float *d_vis, void *stream);

/* Several integrations / coarse channels from one resident buffer, no copies:
 *   sample (coarse c, input i, time m) is at d_volt + 2*(c*coarse_pitch + i*row_pitch + m) bytes;
 *   dump d uses samples [d*T*N, (d+1)*T*N) of every row.  Pitches are in complex samples and must keep
 *   every frame start 16-byte aligned (even pitches when N is a multiple of 8).
 *   d_vis: float [n_coarse][n_dumps][C][B][2].
 */
int mwax_corr_process_batch(mwax_corr_t *h, const int8_t *d_volt, size_t row_pitch, size_t coarse_pitch,
                            int n_dumps, int n_coarse, float *d_vis, void *stream);

/* Same as process_batch but with HOST buffers (pinned memory recommended): the call copies the voltages
 * host->device, runs the path, copies the visibilities device->host and synchronises `stream` before
 * returning.  The kernels run on `stream`, after whatever the caller has queued there; the copies run on two
 * streams of the handle so that dump d + 1 arrives and dump d - 1 leaves while dump d is correlated (the last
 * dump leaves in channel ranges).  Staging buffers are owned by the handle (allocated on first use).
 * Errors: MWAX_ERR_NULL, MWAX_ERR_INVALID_ARG (pitch shorter than n_dumps integrations), MWAX_ERR_NOMEM
 * (staging), MWAX_ERR_CUDA. */
int mwax_corr_process_host(mwax_corr_t *h, const int8_t *h_volt, size_t row_pitch, size_t coarse_pitch,
                           int n_dumps, int n_coarse, float *h_vis, void *stream);

/* F stage / X stage on their own (used by the per-stage benchmarks and tests).
 * f_stage writes the handle's workspace; x_stage consumes it.  Same argument meaning as process(). */
int mwax_corr_f_stage(mwax_corr_t *h, const int8_t *d_volt, size_t row_pitch, void *stream);
int mwax_corr_x_stage(mwax_corr_t *h, float *d_vis, void *stream);

/* MWAX_ORDER emitter (§2.7, Figs 8-9): re-index one dump from the native
 * packed triangle into the instrument's output order, on the device.
 *   d_vis      in : float [C][n(n+1)/2][re,im], as written by process() (n_inputs must be even: signal path
 *                   i = 2*tile + pol, pol x = 0, y = 1, reading Q20)
 *   d_out      out: float [n_tiles(n_tiles+1)/2][C][xx,xy,yx,yy][re,im], baselines antA <= antB row by row
 *                   (0-0, 0-1, ..., 0-(nt-1), 1-1, ...); element (antA, antB, ch, pq) = sum X_{antA,p} conj(X_{antB,q})
 *                   (reading Q21).  mwax_corr_mwax_order_bytes() bytes.
 *   d_weights  out: float [n_tiles(n_tiles+1)/2][4] visibility weights, all 1.0 (L328), or NULL
 * Pure data movement: the values are bit copies (sign of Im flipped where the conjugate is taken).
 * CAVEAT (readings Q2, Q21, both "parity unpinned"): PAPER.md does not say which antenna of a baseline is
 * conjugated nor how Fig. 8's xx, xy, yx, yy map onto (antA, antB); nothing in the container pins it.  The output may
 * therefore be the complex conjugate (and xy/yx swapped) of what the real instrument writes. */
int mwax_corr_to_mwax_order(mwax_corr_t *h, const float *d_vis, float *d_out, float *d_weights, void *stream);
size_t mwax_corr_mwax_order_bytes(const mwax_corr_t *h);

/* Same with occupancy weights (§4.1, §2.4.2):
 *   d_flags    in : uint8 [n_inputs][n_sub] zeroing flags of this integration, 1 = that sub-block (50 ms in the paper)
 *                   of that signal path was zero-filled; NULL = nothing was (weights 1.0)
 *   normalise     : non-zero divides every visibility by its weight (weight 0 leaves the zero visibility as it is)
 *   d_weights  out: weight(antA, antB, pq) = fraction of the n_sub sub-blocks in which BOTH signal paths were valid */
int mwax_corr_to_mwax_order_weighted(mwax_corr_t *h, const float *d_vis, const uint8_t *d_flags, int n_sub, int normalise,
                                     float *d_out, float *d_weights, void *stream);

size_t mwax_corr_input_bytes(const mwax_corr_t *h);
size_t mwax_corr_output_bytes(const mwax_corr_t *h);
size_t mwax_corr_workspace_bytes(const mwax_corr_t *h);
/* Caller-owned workspace (e.g. a torch tensor) instead of the one create() allocated: d_ws is DEVICE memory of at
 * least mwax_corr_workspace_bytes() bytes, 256-byte aligned; it is zeroed here, the library's own buffer is released,
 * and the memory must outlive the handle's last call.  Synchronises the device; not to be called with work in flight. */
int mwax_corr_set_workspace(mwax_corr_t *h, void *d_ws, size_t bytes);
/* X-stage schedule of this plan: with even f_avg and the centre-symmetric averaging of PAPER.md L290-298
 * the outermost fine channel of an output channel is shared, at half weight, with its neighbour; when it pays, a CTA
 * pair walks a run of adjacent output channels and contracts each shared channel once.  Returns the number of such runs
 * per tile (> 0), 0 for the plain schedule (every output channel on its own), or a negative MWAX_ERR_* code. */
int mwax_corr_x_edge_runs(mwax_corr_t *h);
/* total number of kernels this handle has enqueued since create() (F, X and MWAX_ORDER kernels of every entry point) */
long long mwax_corr_launch_count(const mwax_corr_t *h);
int mwax_corr_last_cuda_error(const mwax_corr_t *h);
int mwax_corr_destroy(mwax_corr_t *h); /* NULL is a no-op returning MWAX_OK */

/* ------------------------------------------------------------------------------------------------------
 * Allocation-free entry (no handle): one integration through the same F and X kernels as
 * mwax_corr_create(n_inputs, n_fft, n_fft, t_int, f_avg) + mwax_corr_process with default options (every bin kept,
 * centre-symmetric averaging, DC excluded), for callers that may not call cudaMalloc: code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid allocation.  The call makes NO cudaMalloc / cudaFree / host-to-
 * device copy: the fp16 spectra Y[n_fft][t_int][pitch] (pitch = 2 n_inputs rounded up to 64) that the path keeps
 * between its two kernels live in a static device array inside the library, MWAX_STATIC_Y_BYTES = 32 MiB (plus 64 KiB
 * of tables filled on the device), which every GPU that loads the library holds until the process exits.
 *   d_volt in : int8 [n_inputs][t_int * n_fft][re,im], contiguous rows, 16-byte aligned (else MWAX_ERR_INVALID_ARG)
 *   d_vis  out: float [n_fft / f_avg][n(n+1)/2][re,im]  (caller-owned, as for mwax_corr_process)
 *   n_fft  in {64, 128, 256, 512} (the kernels whose tables travel in the kernel parameters; else MWAX_ERR_UNSUPPORTED),
 *   f_avg divides n_fft, n_inputs <= 8128.
 * Limit: n_fft * t_int * pitch * 2 bytes <= mwax_corr_static_workspace_max() = MWAX_STATIC_Y_BYTES, otherwise
 * MWAX_ERR_TOO_LARGE is returned and nothing is enqueued (e.g. 128 inputs x 128 channels x 512 spectra = 32 MiB fits).
 * The array is SHARED by every call on a device and keeps the last call's contents (the call clears what it needs
 * zero): two calls that overlap on the GPU (different streams or threads without an ordering between them) race.
 * Work is enqueued on `stream` (3-4 operations: optional clear, table kernel, F kernel, X kernel); the call is
 * asynchronous like mwax_corr_process.  The first call on a device sets kernel attributes and looks the array's
 * address up (cudaGetSymbolAddress); make it once outside a graph capture.
 * ---------------------------------------------------------------------------------------------------- */
#define MWAX_STATIC_Y_BYTES (32u * 1024u * 1024u)
#define MWAX_STATIC_TABLE_BYTES (64u * 1024u)
size_t mwax_corr_static_workspace_max(void);
int mwax_corr_process_static(const int8_t *d_volt, float *d_vis, int n_inputs, int n_fft, int t_int, int f_avg, void *stream);

/* ------------------------------------------------------------------------------------------------------
 * X-only integer path (BASELINE.json configs[1]): the X-stage contraction on pre-channelised int8
 * samples, exact int32 accumulation, no FFT, no averaging.
 *   d_z   in : int8 [n_chan][n_time][n_inputs][re,im], any n_inputs >= 1.  The kernel reads the buffer in place through a
 *              TMA tensor map when rows are 16-byte multiples (n_inputs % 8 == 0) and d_z is 16-byte aligned; otherwise
 *              the call first copies it, on the device, into an internal buffer with rows padded to 16 bytes (one extra
 *              pass over the input; allocated on first use, MWAX_ERR_NOMEM if that fails).  Partial tiles are padded by
 *              the tensor map's out-of-bounds zero fill.
 *   d_vis out: int32 [n_chan][n(n+1)/2][re,im],  Re = sum(a_i a_j + b_i b_j), Im = sum(b_i a_j - a_i b_j)
 * The caller guarantees 2*128*128*n_time < 2^31 (n_time <= 65535, else MWAX_ERR_UNSUPPORTED) so int32 cannot overflow.
 * process_host: the same with HOST buffers (pinned recommended); channels travel in 4 ranges so that range q + 1 goes
 * host->device and range q - 1 device->host while range q is correlated; synchronises `stream` before returning.
 * ---------------------------------------------------------------------------------------------------- */
mwax_xcorr_t *mwax_xcorr_i8_create(int n_inputs, int n_chan, int n_time);
int mwax_xcorr_i8_process(mwax_xcorr_t *h, const int8_t *d_z, int32_t *d_vis, void *stream);
int mwax_xcorr_i8_process_host(mwax_xcorr_t *h, const int8_t *h_z, int32_t *h_vis, void *stream);
int mwax_xcorr_i8_destroy(mwax_xcorr_t *h);

const char *mwax_corr_strerror(int code);
/* "sm_100a tcgen05/TMA; built <date>" — identifies the native library in logs */
const char *mwax_corr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MWAX_CORR_H */
