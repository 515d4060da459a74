// mwax_api.cu — the C ABI (include/mwax_corr.h): plan construction (tables, workspace, TMA tensor maps,
// triangle tile schedule) and kernel launches.  No CPU fallback: without an sm_100 device create() fails with
// MWAX_ERR_ARCH.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <algorithm>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/mwax_corr.h"
#include "f_stage.cuh"
#include "f_stage_pow2.cuh"
#include "f_stage_6400.cuh"
#include "x_stage.cuh"
#include "x_stage2.cuh"
#include "mwax_order.cuh"

namespace {

thread_local int g_last_error = MWAX_OK;

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

PFN_encodeTiled get_encode_fn()
{
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_encodeTiled>(p);
    }
    return fn;
}

// 3-D map over rows of `row_bytes` bytes: dims (inner elements, rows per channel, channels); box = 128 bytes x
// box_rows x 1, SWIZZLE_128B, out-of-bounds elements read as zero (that is what pads partial tiles and the
// last contraction block of a channel).
int encode_z_map(CUtensorMap *m, bool int8, const void *base, uint64_t inner_elems, uint64_t row_bytes, uint64_t rows,
                 uint64_t chans, uint32_t box_rows)
{
    PFN_encodeTiled fn = get_encode_fn();
    if (!fn) return MWAX_ERR_CUDA;
    cuuint64_t dims[3] = {inner_elems, rows, chans};
    cuuint64_t strides[2] = {row_bytes, row_bytes * rows};
    cuuint32_t box[3] = {int8 ? 128u : 64u, box_rows, 1u};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(m, int8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3,
                    const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? MWAX_OK : MWAX_ERR_CUDA;
}

bool factor_2_5(int N, std::vector<int> &radix)
{
    radix.clear();
    while (N % 4 == 0) { radix.push_back(4); N /= 4; }
    while (N % 2 == 0) { radix.push_back(2); N /= 2; }
    while (N % 5 == 0) { radix.push_back(5); N /= 5; }
    return N == 1;
}

// The library is built for sm_100a only (arch-specific code, not forward compatible): any other device, sm_103 included,
// is refused here instead of failing at the first launch with "no kernel image".
int check_device(int *sm_count, int *device)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MWAX_ERR_ARCH;
    int major = 0, minor = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return MWAX_ERR_ARCH;
    if (major != 10 || minor != 0) return MWAX_ERR_ARCH;
    *sm_count = sms;
    *device = dev;
    return MWAX_OK;
}

// every entry point that launches work checks that the caller is on the device the handle was created on
bool on_device(int device)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == device;
}

// tile list of the CTA-pair kernel: (mi, nj, 0, 0) in units of 128 inputs, nj <= mi
void build_pair_tiles(int n, std::vector<uint8_t> &tiles)
{
    tiles.clear();
    for (int mi = 0; mi * 128 < n; ++mi)
        for (int nj = 0; nj <= mi; ++nj) {
            tiles.push_back((uint8_t)mi);
            tiles.push_back((uint8_t)nj);
            tiles.push_back(0);
            tiles.push_back(0);
        }
}

template <typename T>
int upload(T **dptr, const std::vector<T> &h)
{
    if (*dptr) { cudaFree(*dptr); *dptr = nullptr; }
    if (cudaMalloc(reinterpret_cast<void **>(dptr), h.size() * sizeof(T)) != cudaSuccess) return MWAX_ERR_NOMEM;
    if (cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return MWAX_ERR_CUDA;
    return MWAX_OK;
}

// ------------------------------------------------------------------------------------------------ per-device setup
// cudaFuncSetAttribute and the occupancy queries are per DEVICE, a handle may be created on any sm_100 device of the
// process and handles may be used from different threads: the attributes of every kernel are set once per device, under
// a mutex, before create() returns; the launch paths only read what the handle copied from here.
constexpr int HOST_PARTS = 4;                      // channel ranges of the host-buffer entries' pipelines
constexpr int GENERIC_SMEM_MAX = 200 * 1024;       // the generic F kernel's largest plan (two fp32 ping-pong buffers)

struct DevicePlan {
    int pairs_f16, pairs_f16_edge, pairs_i8;       // CTA pairs the device holds at once (persistent X grids)
};

template <typename K>
bool set_smem(K kern, int bytes)
{
    return cudaFuncSetAttribute(reinterpret_cast<const void *>(kern), cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess;
}

template <int N, int R1, int PTS>
bool prep_f_pow2()
{
    using C = mwax::FPow2Config<N, R1, PTS>;
    return set_smem(mwax::f_stage_pow2_kernel<N, R1, PTS, true, false, false>, C::SMEM_BYTES) &&
           set_smem(mwax::f_stage_pow2_kernel<N, R1, PTS, true, true, false>, C::SMEM_BYTES) &&
           set_smem(mwax::f_stage_pow2_kernel<N, R1, PTS, false, true, false>, C::SMEM_BYTES) &&
           set_smem(mwax::f_stage_pow2_kernel<N, R1, PTS, true, true, true>, C::SMEM_BYTES) &&
           set_smem(mwax::f_stage_pow2_kernel<N, R1, PTS, false, true, true>, C::SMEM_BYTES);
}

// CTA pairs the device can hold at once for this kernel (GPCs with an odd SM count leave one SM unpaired); 0 on error
template <bool kInt8, bool kEdge>
int prep_x_pair(int sm_count)
{
    using C = mwax::XPairConfig<kInt8, kEdge>;
    auto kern = mwax::x_stage_pair_kernel<kInt8, kEdge>;
    if (!set_smem(kern, C::SMEM_BYTES)) return 0;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(C::THREADS); cfg.dynamicSmemBytes = C::SMEM_BYTES;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cfg.gridDim = dim3(2);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n < 1) n = sm_count / 2;
    return n < sm_count / 2 ? n : sm_count / 2;
}

int prepare_device(int dev, int sm_count, DevicePlan *out)
{
    static std::mutex mu;
    static std::map<int, DevicePlan> done;
    std::lock_guard<std::mutex> lock(mu);
    auto it = done.find(dev);
    if (it != done.end()) { *out = it->second; return MWAX_OK; }
    using F64 = mwax::F6400;
    bool ok = prep_f_pow2<64, 8, 16>() && prep_f_pow2<128, 8, 16>() && prep_f_pow2<256, 16, 32>() && prep_f_pow2<512, 16, 32>() &&
              set_smem(mwax::f_stage_6400_kernel<true, false, false>, F64::SMEM_BYTES) &&
              set_smem(mwax::f_stage_6400_kernel<true, true, false>, F64::SMEM_BYTES) &&
              set_smem(mwax::f_stage_6400_kernel<false, true, false>, F64::SMEM_BYTES) &&
              set_smem(mwax::f_stage_6400_kernel<true, true, true>, F64::SMEM_BYTES) &&
              set_smem(mwax::f_stage_6400_kernel<false, true, true>, F64::SMEM_BYTES) &&
              set_smem(mwax::f_stage_generic_kernel, GENERIC_SMEM_MAX);
    DevicePlan dp;
    dp.pairs_f16 = prep_x_pair<false, false>(sm_count);
    dp.pairs_f16_edge = prep_x_pair<false, true>(sm_count);
    dp.pairs_i8 = prep_x_pair<true, false>(sm_count);
    if (!ok || dp.pairs_f16 < 1 || dp.pairs_f16_edge < 1 || dp.pairs_i8 < 1) { cudaGetLastError(); return MWAX_ERR_CUDA; }
    done[dev] = dp;
    *out = dp;
    return MWAX_OK;
}

// power-of-two register kernel: (N, R1, PTS) per supported length; FULL = every bin kept, SCALE = sw[] applied
template <int N, int R1, int PTS>
int launch_f_pow2(const mwax::FParams &fp, bool full, bool scale, bool delay, int groups, int chunks, cudaStream_t st)
{
    using C = mwax::FPow2Config<N, R1, PTS>;
    dim3 grid(groups, chunks);
    if (delay) {   // the delay variants always take the (all-ones when unused) weight table
        if (full) mwax::f_stage_pow2_kernel<N, R1, PTS, true, true, true><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
        else mwax::f_stage_pow2_kernel<N, R1, PTS, false, true, true><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
    } else if (full && !scale)
        mwax::f_stage_pow2_kernel<N, R1, PTS, true, false, false><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
    else if (full)
        mwax::f_stage_pow2_kernel<N, R1, PTS, true, true, false><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
    else
        mwax::f_stage_pow2_kernel<N, R1, PTS, false, true, false><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
    return MWAX_OK;
}

template <bool FULL, bool SCALE, bool DELAY>
int launch_f_6400_v(const mwax::FParams &fp, int sm_count, cudaStream_t st)
{
    using C = mwax::F6400;
    // persistent CTAs, one per SM; item = (frame t, group of 8 inputs), groups fastest
    const long long items = (long long)((fp.n_inputs + C::GI - 1) / C::GI) * fp.T;
    const int grid = (int)(items < sm_count ? items : sm_count);
    mwax::f_stage_6400_kernel<FULL, SCALE, DELAY><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(fp);
    return MWAX_OK;
}

int launch_f_6400(const mwax::FParams &fp, bool full, bool scale, bool delay, int sm_count, cudaStream_t st)
{
    if (delay) {   // the delay variants always take the weight codes / table
        if (full) return launch_f_6400_v<true, true, true>(fp, sm_count, st);
        return launch_f_6400_v<false, true, true>(fp, sm_count, st);
    }
    if (full && !scale) return launch_f_6400_v<true, false, false>(fp, sm_count, st);
    if (full) return launch_f_6400_v<true, true, false>(fp, sm_count, st);
    return launch_f_6400_v<false, true, false>(fp, sm_count, st);
}

// persistent grid of CTA pairs: never more pairs than run concurrently on this device (max_pairs from prepare_device)
template <bool kInt8, bool kEdge = false>
int launch_x_pair(const CUtensorMap &tmap, const CUtensorMap &tmap_flat, const mwax::XParams &xp, int max_pairs, cudaStream_t st)
{
    using C = mwax::XPairConfig<kInt8, kEdge>;
    auto kern = mwax::x_stage_pair_kernel<kInt8, kEdge>;
    if (max_pairs < 1) return MWAX_ERR_CUDA;
    const int n_items = (kEdge ? xp.edge_runs : xp.n_out) * xp.n_tiles;   // units of the persistent loop
    if (n_items <= 0) return MWAX_OK;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(C::THREADS); cfg.dynamicSmemBytes = C::SMEM_BYTES; cfg.stream = st;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const int pairs = n_items < max_pairs ? n_items : max_pairs;
    cfg.gridDim = dim3(2 * pairs);
    return cudaLaunchKernelEx(&cfg, kern, tmap, tmap_flat, xp) == cudaSuccess ? MWAX_OK : MWAX_ERR_CUDA;
}

// Shared-edge schedule (x_stage.cuh): how many runs of adjacent output channels per tile, or 0 when the
// plain schedule is at least as good.  Cost model = waves of the persistent grid x cost of the longest unit, in contraction
// rows: an accumulator costs max(its rows, its epilogue), the epilogues measured on B200 as ~860 rows' worth of MMA time for
// one that stores a 256 x 256 tile and ~770 for one that only updates the running sums (n = 512, F = 2, T = 64..512:
// the plain schedule levels off at 0.09 ms below T = 256, the shared-edge one at 0.17 ms below T = 512).  A run of L channels
// costs max(T, 770) + L max(F T, 860 + 770), the plain schedule max((F + 1) T, 860) per channel; the shared-edge kernel also
// has 4 instead of 6 pipeline stages (F = 50: 3 % slower than the model says), hence the 4 % handicap and the 8 % margin.
// `want` is MWAX_OPT_X_EDGE_RUNS: -1 = decide here (default), 0 = never, r >= 1 = r runs (at most C) whenever the geometry allows.
int choose_edge_runs(int C, int F, int T, int n_tiles, int pairs, int want)
{
    if (want == 0 || F < 2 || (F & 1) || T < 64 || pairs < 1) return 0;
    if (want >= 1) return want < C ? want : C;
    const long long e_out = 860, e_add = 770;
    const long long per_chan_plain = std::max<long long>((long long)(F + 1) * T, e_out);
    const long long per_chan_edge = std::max<long long>((long long)F * T, e_out + e_add);
    const long long init = std::max<long long>(T, e_add);
    const long long plain = (((long long)C * n_tiles + pairs - 1) / pairs) * per_chan_plain;
    long long best = -1;
    int best_r = 0;
    for (int r = 1; r <= C; ++r) {
        const long long waves = ((long long)r * n_tiles + pairs - 1) / pairs;
        const long long cost = waves * (init + (long long)((C + r - 1) / r) * per_chan_edge);
        if (best < 0 || cost < best) { best = cost; best_r = r; }
    }
    return (best * 104 <= plain * 92) ? best_r : 0;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ handles
struct mwax_corr {
    int n, N, K, T, F, C;
    int device;        // CUDA device the handle lives on; every call checks that it is the current one
    DevicePlan dp;
    int avg_mode;
    int dc_exclude;    // MWAX_OPT_DC_EXCLUDE, default 1
    int accumulate;    // MWAX_OPT_ACCUMULATE: process() adds into d_vis
    int want_edge_runs;   // MWAX_OPT_X_EDGE_RUNS: -1 = auto
    int pitch;         // fp16 elements per Y row (2n rounded up to 64)
    int sm_count;
    int last_cuda;
    long long launches;   // kernels enqueued through this handle so far
    bool tables_ready;
    // F plan
    int f_kind;        // 0 = generic Stockham kernel, else the specialised kernel for that N (64, 128, 256, 512, 6400)
    float in_scale;
    int chan_scale;
    int G;
    size_t f_smem;
    std::vector<int> radix;
    // device tables
    float2 *d_tw;
    unsigned *d_swcode;
    float *d_sw;
    std::vector<float> h_sw;            // host copy of sw[] for the register kernels' parameter-bank table
    std::vector<float2> h_twc;          // W_N^{r k1} as [r][k1], computed once at create() for the same table
    int *d_tap_start;
    float *d_scale;
    uint8_t *d_ptiles;  // CTA-pair tile list
    int n_ptiles;
    int n_taps;
    int edge_runs;      // shared-edge schedule of the pair kernel: runs per tile, 0 = off, -1 = not chosen yet
    __half *d_Y;
    bool y_owned;      // false after mwax_corr_set_workspace: the caller owns the memory
    size_t y_bytes;
    CUtensorMap tmap;       // Y as [p][t][2n]: one channel position per box (rows past T read as zero)
    CUtensorMap tmap_flat;  // Y as [p T + t][2n]: boxes may run across adjacent channel positions
    // staging for process_host
    int8_t *d_in;
    size_t in_bytes;
    float *d_out;
    size_t out_bytes;
    const float *d_delay, *d_phase;        // caller-owned delay / phase tables (mwax_corr_set_delays), NULL = off
    std::vector<float> gains;              // per-channel magnitude gains (mwax_corr_set_channel_gains); empty = off
    size_t d_row_stride, d_coarse_stride;
    cudaStream_t s_in, s_out;              // copy streams of process_host
    cudaEvent_t ev_start, ev_copied;
    cudaEvent_t ev_part[8];                // channel ranges of the last dump of process_host
    std::vector<cudaEvent_t> ev_in, ev_done;
};

struct mwax_xcorr {
    int n, n_chan, n_time;
    int device;
    DevicePlan dp;
    int sm_count;
    int last_cuda;
    int pitch;          // bytes per (channel, time) row as the kernel reads it: 2n rounded up to 16 (TMA row pitch)
    int *d_tap_start;
    uint8_t *d_ptiles;
    int n_ptiles;
    int8_t *d_pad;      // [chan][time][pitch] copy of a ragged (2n % 16 != 0) input, allocated on first use
    int8_t *d_in;
    int32_t *d_out;
    cudaStream_t s_in, s_out;              // copy streams of process_host
    cudaEvent_t ev_start, ev_in[HOST_PARTS], ev_done[HOST_PARTS], ev_copied;
};

static int note_cuda(int *slot)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { *slot = (int)e; return MWAX_ERR_CUDA; }
    return MWAX_OK;
}

static void free_tables(mwax_corr *h)
{
    cudaFree(h->d_sw); h->d_sw = nullptr;
    cudaFree(h->d_swcode); h->d_swcode = nullptr;
    cudaFree(h->d_tap_start); h->d_tap_start = nullptr;
    cudaFree(h->d_scale); h->d_scale = nullptr;
    cudaFree(h->d_ptiles); h->d_ptiles = nullptr;
    h->tables_ready = false;
}

// Averaging geometry -> per-position factor sw[p], per-channel first tap and epilogue scale.
// The weights of PAPER.md L290-298 are folded as  W[c][p] = scale_c * s^2-normalised sw[p]^2 :
//   sw[p]   = sqrt(w_p) (the F stage also applies the power-of-two scale s), w_p = 1 inside a group, 1/2 on a shared edge (even F), 0 for the DC fine channel (F > 1)
//   scale_c = 1/(s^2 F), times F/(F-1) for the centre channel when F > 1.
static int build_tables(mwax_corr *h)
{
    free_tables(h);
    const int K = h->K, F = h->F, C = h->C;
    const int lg = (int)std::ceil(std::log2((double)h->N) / 2.0);
    const double s = std::ldexp(1.0, -lg);   // power of two near 1/sqrt(N): keeps fp16 in range, epilogue exact
    h->in_scale = (float)s;
    h->chan_scale = 0;
    std::vector<float> sw(K, 1.0f), scale(C, (float)(1.0 / (s * s * F)));
    std::vector<int> tap(C);
    if (h->avg_mode == MWAX_AVG_BLOCK || F == 1) {
        h->n_taps = F;
        for (int c = 0; c < C; ++c) tap[c] = c * F;
    } else {
        const int c0 = C / 2, half = K / 2;
        const int dmax = (F % 2) ? (F - 1) / 2 : F / 2;
        h->n_taps = 2 * dmax + 1;
        for (int c = 0; c < C; ++c) {
            const int u0 = (c - c0) * F - dmax;
            tap[c] = ((u0 + half) % K + K) % K;
        }
        if (F % 2 == 0)
            for (int p = 0; p < K; ++p) {
                const int u = p - half;
                if ((((u - F / 2) % F) + F) % F == 0) sw[p] = (float)std::sqrt(0.5);
            }
        h->chan_scale = (F % 2 == 0) ? 1 : 0;
        if (h->dc_exclude) {                                        // DC excluded, centre channel re-scaled (L290-294)
            sw[half] = 0.0f;
            h->chan_scale = 1;
            scale[c0] = (float)((1.0 / (s * s * F)) * (double)F / (double)(F - 1));
        }
    }
    std::vector<uint8_t> tiles;
    h->edge_runs = -1;
    int rc;
    if ((rc = upload(&h->d_sw, sw)) != MWAX_OK) return rc;
    h->h_sw = sw;
    if (h->N == 6400 && K == 6400) {
        // the three-pass kernel takes sqrt(w_p) as 2-bit codes, one word per c = k mod 400, field k3 = k / 400
        std::vector<unsigned> code(400, 0u);
        for (int k = 0; k < 6400; ++k) {
            const float v = sw[k < 3200 ? k + 3200 : k - 3200];
            const unsigned cd = v == 1.0f ? 0u : (v == 0.0f ? 2u : 1u);
            code[k % 400] |= cd << (2 * (k / 400));
        }
        if ((rc = upload(&h->d_swcode, code)) != MWAX_OK) return rc;
    }
    if (!h->gains.empty()) {
        // PFB de-ripple magnitudes (PAPER.md 4.2): folded into the same per-position factor; the 2-bit codes above no
        // longer describe it, so the N = 6400 kernel is launched in its table-reading (non-FULL) form while gains are set
        for (int p = 0; p < K; ++p) sw[p] *= h->gains[p];
        h->chan_scale = 1;
        cudaFree(h->d_sw); h->d_sw = nullptr;
        if ((rc = upload(&h->d_sw, sw)) != MWAX_OK) return rc;
        h->h_sw = sw;
    }
    if ((rc = upload(&h->d_tap_start, tap)) != MWAX_OK) return rc;
    if ((rc = upload(&h->d_scale, scale)) != MWAX_OK) return rc;
    build_pair_tiles(h->n, tiles);
    h->n_ptiles = (int)tiles.size() / 4;
    if ((rc = upload(&h->d_ptiles, tiles)) != MWAX_OK) return rc;
    h->tables_ready = true;
    return MWAX_OK;
}

extern "C" {

int mwax_corr_last_error(void) { return g_last_error; }

const char *mwax_corr_strerror(int code)
{
    switch (code) {
        case MWAX_OK: return "ok";
        case MWAX_ERR_NULL: return "null pointer";
        case MWAX_ERR_INVALID_ARG: return "invalid argument";
        case MWAX_ERR_UNSUPPORTED: return "unsupported configuration";
        case MWAX_ERR_NOMEM: return "out of memory";
        case MWAX_ERR_CUDA: return "CUDA error";
        case MWAX_ERR_ARCH: return "no sm_100 CUDA device";
        case MWAX_ERR_TOO_LARGE: return "spectra exceed the static workspace (MWAX_STATIC_Y_BYTES, see mwax_corr_static_workspace_max)";
        default: return "unknown error";
    }
}

const char *mwax_corr_version(void) { return "mwax_corr sm_100a tcgen05/TMA; built " __DATE__ " " __TIME__; }

mwax_corr_t *mwax_corr_create(int n_inputs, int n_fft, int n_keep, int t_int, int f_avg)
{
    g_last_error = MWAX_OK;
    if (n_inputs < 1 || n_fft < 1 || n_keep < 1 || t_int < 1 || f_avg < 1) { g_last_error = MWAX_ERR_INVALID_ARG; return nullptr; }
    std::vector<int> radix;
    if (n_fft > 6400 || !factor_2_5(n_fft, radix) || n_keep > n_fft || n_keep % f_avg != 0 || n_inputs > 8128) {
        g_last_error = MWAX_ERR_UNSUPPORTED;
        return nullptr;
    }
    int sm = 0, dev = 0;
    if ((g_last_error = check_device(&sm, &dev)) != MWAX_OK) return nullptr;
    DevicePlan dp;
    if ((g_last_error = prepare_device(dev, sm, &dp)) != MWAX_OK) return nullptr;
    mwax_corr *h = new (std::nothrow) mwax_corr();
    if (!h) { g_last_error = MWAX_ERR_NOMEM; return nullptr; }
    h->n = n_inputs; h->N = n_fft; h->K = n_keep; h->T = t_int; h->F = f_avg; h->C = n_keep / f_avg;
    h->device = dev; h->dp = dp;
    h->avg_mode = MWAX_AVG_CENTRE_SYMMETRIC;
    h->dc_exclude = 1;
    h->want_edge_runs = -1;
    h->pitch = ((2 * n_inputs + 63) / 64) * 64;
    if ((unsigned long long)t_int * (unsigned long long)(h->pitch / 2) >= (1ull << 32)) {   // kernels keep this stride in 32 bits
        g_last_error = MWAX_ERR_UNSUPPORTED; delete h; return nullptr;
    }
    h->sm_count = sm;
    h->last_cuda = 0;
    h->radix = radix;
    // F plan: specialised kernels for N in {64,128,256,512,6400}; otherwise the generic Stockham kernel with as
    // many adjacent inputs per CTA as fit (two fp32 ping-pong buffers), up to 32 (128-byte segments)
    int G = 32;
    while (G > 1 && (size_t)2 * G * n_fft * sizeof(float2) > (size_t)GENERIC_SMEM_MAX) G >>= 1;
    h->G = G;
    h->f_smem = (size_t)2 * G * n_fft * sizeof(float2);
    h->f_kind = 0;
    if (n_fft == 64 || n_fft == 128 || n_fft == 256 || n_fft == 512 || n_fft == 6400) h->f_kind = n_fft;
    // the N = 6400 kernel forms store addresses from a 32-bit byte stride between channel positions
    if (n_fft == 6400 && (unsigned long long)t_int * (unsigned long long)(h->pitch / 2) >= (1ull << 30)) h->f_kind = 0;
    // twiddles exp(-2 pi i m / N), computed in double
    std::vector<float2> tw(n_fft);
    for (int m = 0; m < n_fft; ++m) {
        const double a = 2.0 * M_PI * (double)m / (double)n_fft;
        tw[m] = make_float2((float)std::cos(a), (float)(-std::sin(a)));
    }
    if ((g_last_error = upload(&h->d_tw, tw)) != MWAX_OK) { mwax_corr_destroy(h); return nullptr; }
    if (h->f_kind && h->f_kind != 6400) {
        const int R1 = h->f_kind <= 128 ? 8 : 16, R2 = h->f_kind / R1;
        h->h_twc.resize((size_t)h->f_kind);
        for (int r = 0; r < R2; ++r)
            for (int k1 = 0; k1 < R1; ++k1) {
                const double a = 2.0 * M_PI * (double)((r * k1) % h->f_kind) / (double)h->f_kind;
                h->h_twc[(size_t)r * R1 + k1] = make_float2((float)std::cos(a), (float)(-std::sin(a)));
            }
    }
    // workspace Y[K][T][pitch] fp16, zeroed once (pad columns stay zero)
    h->y_bytes = (size_t)n_keep * t_int * h->pitch * sizeof(__half);
    if (cudaMalloc(reinterpret_cast<void **>(&h->d_Y), h->y_bytes) != cudaSuccess) {
        g_last_error = MWAX_ERR_NOMEM; mwax_corr_destroy(h); return nullptr;
    }
    h->y_owned = true;
    cudaMemset(h->d_Y, 0, h->y_bytes);
    if ((g_last_error = encode_z_map(&h->tmap, false, h->d_Y, (uint64_t)h->pitch, (uint64_t)h->pitch * 2,
                                     (uint64_t)t_int, (uint64_t)n_keep, 64)) != MWAX_OK) {
        mwax_corr_destroy(h); return nullptr;
    }
    if ((g_last_error = encode_z_map(&h->tmap_flat, false, h->d_Y, (uint64_t)h->pitch, (uint64_t)h->pitch * 2,
                                     (uint64_t)t_int * n_keep, 1, 64)) != MWAX_OK) {
        mwax_corr_destroy(h); return nullptr;
    }
    if ((g_last_error = build_tables(h)) != MWAX_OK) { mwax_corr_destroy(h); return nullptr; }
    if (cudaDeviceSynchronize() != cudaSuccess) { g_last_error = MWAX_ERR_CUDA; mwax_corr_destroy(h); return nullptr; }
    return h;
}

int mwax_corr_set_option(mwax_corr_t *h, int key, int value)
{
    if (!h) return MWAX_ERR_NULL;
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    switch (key) {
        case MWAX_OPT_AVG_MODE:
            if (value != MWAX_AVG_CENTRE_SYMMETRIC && value != MWAX_AVG_BLOCK) return MWAX_ERR_INVALID_ARG;
            h->avg_mode = value;
            return build_tables(h);
        case MWAX_OPT_DC_EXCLUDE:
            if (value != 0 && value != 1) return MWAX_ERR_INVALID_ARG;
            h->dc_exclude = value;
            return build_tables(h);
        case MWAX_OPT_ACCUMULATE:
            if (value != 0 && value != 1) return MWAX_ERR_INVALID_ARG;
            h->accumulate = value;
            return MWAX_OK;
        case MWAX_OPT_X_EDGE_RUNS:
            if (value < -1) return MWAX_ERR_INVALID_ARG;
            h->want_edge_runs = value;
            h->edge_runs = -1;       // chosen again at the next call
            return MWAX_OK;
        default:
            return MWAX_ERR_INVALID_ARG;
    }
}

int mwax_corr_set_channel_gains(mwax_corr_t *h, const float *gain)
{
    if (!h) return MWAX_ERR_NULL;
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    if (!gain) {
        if (h->gains.empty()) return MWAX_OK;
        h->gains.clear();
        return build_tables(h);
    }
    // |Y| <= 127 sqrt(2) N s gain with s ~ 1/sqrt(N) must stay inside fp16: gain <= 4 leaves a factor > 1.1 at N = 6400
    for (int p = 0; p < h->K; ++p)
        if (!(gain[p] >= 0.0f && gain[p] <= 4.0f)) return MWAX_ERR_INVALID_ARG;
    h->gains.assign(gain, gain + h->K);
    return build_tables(h);
}

static int f_stage_impl(mwax_corr_t *h, const int8_t *d_volt, size_t row_pitch, int frame0, int coarse, void *stream)
{
    if (!h || !d_volt) return MWAX_ERR_NULL;
    if (!h->tables_ready || !on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    mwax::FParams fp;
    fp.volt = d_volt; fp.row_pitch = (long long)row_pitch; fp.sample0 = 0;
    fp.n_inputs = h->n; fp.N = h->N; fp.K = h->K; fp.T = h->T; fp.G = h->G; fp.frames_per_cta = 1;
    fp.n_pass = (int)h->radix.size();
    for (int i = 0; i < fp.n_pass; ++i) fp.radix[i] = h->radix[i];
    fp.vec_ok = (h->N % 8 == 0) && (row_pitch % 8 == 0) && ((reinterpret_cast<uintptr_t>(d_volt) & 15u) == 0);
    fp.tw = h->d_tw; fp.swcode = h->d_swcode; fp.sw = h->d_sw; fp.in_scale = h->in_scale; fp.chan_scale = h->chan_scale;
    fp.Y = reinterpret_cast<__half2 *>(h->d_Y); fp.pitch2 = h->pitch / 2;
    const bool delay = h->d_delay || h->d_phase;
    fp.delay = h->d_delay ? h->d_delay + (size_t)coarse * h->d_coarse_stride : nullptr;
    fp.phase = h->d_phase ? h->d_phase + (size_t)coarse * h->d_coarse_stride : nullptr;
    fp.d_stride = (long long)h->d_row_stride; fp.frame0 = frame0;
    fp.y_p_stride = (unsigned)h->T * (unsigned)(h->pitch / 2); fp.y_t_stride = (unsigned)(h->pitch / 2);
    cudaStream_t st = (cudaStream_t)stream;
    const int f_kind = fp.vec_ok ? h->f_kind : 0;          // misaligned rows: generic kernel (scalar loads)
    if (f_kind == 6400) {
        const bool full = (h->K == h->N) && h->gains.empty(), scale = (h->chan_scale != 0) || !full;
        int rc = launch_f_6400(fp, full, scale, delay, h->sm_count, st);
        if (rc != MWAX_OK) return rc;
    } else if (f_kind) {
        // the register kernels read their twiddles and per-position factors from the kernel parameters (constant bank)
        std::memcpy(fp.twc, h->h_twc.data(), h->h_twc.size() * sizeof(float2));
        std::memcpy(fp.swc, h->h_sw.data(), (size_t)h->K * sizeof(float));
        // frames per CTA: enough CTAs for ~8 waves of 3 resident CTAs per SM, at most 32 frames each
        const int groups = (h->n + 31) / 32;
        long long fpc = ((long long)groups * h->T) / ((long long)h->sm_count * 24);
        if (fpc < 1) fpc = 1;
        if (fpc > 32) fpc = 32;
        fp.frames_per_cta = (int)fpc;
        const int chunks = (h->T + (int)fpc - 1) / (int)fpc;
        const bool full = (h->K == h->N), scale = (h->chan_scale != 0) || !full;
        int rc;
        switch (f_kind) {
            case 64: rc = launch_f_pow2<64, 8, 16>(fp, full, scale, delay, groups, chunks, st); break;
            case 128: rc = launch_f_pow2<128, 8, 16>(fp, full, scale, delay, groups, chunks, st); break;
            case 256: rc = launch_f_pow2<256, 16, 32>(fp, full, scale, delay, groups, chunks, st); break;
            default: rc = launch_f_pow2<512, 16, 32>(fp, full, scale, delay, groups, chunks, st); break;
        }
        if (rc != MWAX_OK) return rc;
    } else {
        dim3 grid((h->n + h->G - 1) / h->G, h->T);
        mwax::f_stage_generic_kernel<<<grid, 256, h->f_smem, st>>>(fp);
    }
    ++h->launches;
    return note_cuda(&h->last_cuda);
}

int mwax_corr_f_stage(mwax_corr_t *h, const int8_t *d_volt, size_t row_pitch, void *stream)
{
    return f_stage_impl(h, d_volt, row_pitch, 0, 0, stream);
}

int mwax_corr_set_delays(mwax_corr_t *h, const float *d_delay, const float *d_phase, size_t row_stride, size_t coarse_stride)
{
    if (!h) return MWAX_ERR_NULL;
    if ((d_delay || d_phase) && row_stride < (size_t)h->T) return MWAX_ERR_INVALID_ARG;
    h->d_delay = d_delay; h->d_phase = d_phase; h->d_row_stride = row_stride; h->d_coarse_stride = coarse_stride;
    return MWAX_OK;
}

int mwax_corr_x_edge_runs(mwax_corr_t *h)
{
    if (!h) return MWAX_ERR_NULL;
    if (!h->tables_ready) return MWAX_ERR_INVALID_ARG;
    if (h->edge_runs < 0)
        h->edge_runs = (h->avg_mode == MWAX_AVG_CENTRE_SYMMETRIC && h->n_taps == h->F + 1)
                           ? choose_edge_runs(h->C, h->F, h->T, h->n_ptiles, h->dp.pairs_f16_edge, h->want_edge_runs) : 0;
    return h->edge_runs;
}

// X stage over the output channels [c0, c0 + cnt) of one dump (d_vis = the dump's base).  The kernels index their
// per-channel tables and the output by channel number, so a sub-range is the same launch on offset pointers; the
// shared-edge schedule walks runs of the whole channel axis and is used for the full range only.
static int x_stage_range(mwax_corr_t *h, float *d_vis, int c0, int cnt, void *stream)
{
    if (!h || !d_vis) return MWAX_ERR_NULL;
    if (!h->tables_ready || c0 < 0 || cnt < 1 || c0 + cnt > h->C || !on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    const bool whole = (c0 == 0 && cnt == h->C);
    mwax::XParams xp;
    xp.n_inputs = h->n; xp.T = h->T; xp.K = h->K; xp.n_out = cnt; xp.n_tiles = h->n_ptiles;
    xp.tiles = h->d_ptiles; xp.tap_start = h->d_tap_start + c0; xp.n_taps = h->n_taps; xp.scale = h->d_scale + c0;
    xp.out_chan_stride = (long long)h->n * (h->n + 1) / 2;
    xp.out = d_vis + (size_t)c0 * (size_t)xp.out_chan_stride * 2;
    xp.accumulate = h->accumulate;
    xp.edge_runs = whole ? mwax_corr_x_edge_runs(h) : 0;
    int rc = xp.edge_runs > 0 ? launch_x_pair<false, true>(h->tmap, h->tmap_flat, xp, h->dp.pairs_f16_edge, (cudaStream_t)stream)
                              : launch_x_pair<false>(h->tmap, h->tmap_flat, xp, h->dp.pairs_f16, (cudaStream_t)stream);
    if (rc != MWAX_OK) note_cuda(&h->last_cuda);
    else ++h->launches;
    return rc;
}

int mwax_corr_x_stage(mwax_corr_t *h, float *d_vis, void *stream)
{
    if (!h) return MWAX_ERR_NULL;
    return x_stage_range(h, d_vis, 0, h->C, stream);
}

int mwax_corr_process_batch(mwax_corr_t *h, const int8_t *d_volt, size_t row_pitch, size_t coarse_pitch, int n_dumps,
                            int n_coarse, float *d_vis, void *stream)
{
    if (!h || !d_volt || !d_vis) return MWAX_ERR_NULL;
    if (n_dumps < 1 || n_coarse < 1 || row_pitch < (size_t)n_dumps * h->T * h->N) return MWAX_ERR_INVALID_ARG;
    if ((h->d_delay || h->d_phase) && h->d_row_stride < (size_t)n_dumps * h->T) return MWAX_ERR_INVALID_ARG;
    const size_t dump_samples = (size_t)h->T * h->N;
    const size_t vis_floats = (size_t)h->C * ((size_t)h->n * (h->n + 1) / 2) * 2;
    for (int c = 0; c < n_coarse; ++c)
        for (int d = 0; d < n_dumps; ++d) {
            int rc = f_stage_impl(h, d_volt + 2 * (c * coarse_pitch + d * dump_samples), row_pitch, d * h->T, c, stream);
            if (rc != MWAX_OK) return rc;
            rc = mwax_corr_x_stage(h, d_vis + ((size_t)c * n_dumps + d) * vis_floats, stream);
            if (rc != MWAX_OK) return rc;
        }
    return MWAX_OK;
}

int mwax_corr_process(mwax_corr_t *h, const int8_t *d_volt, float *d_vis, void *stream)
{
    if (!h) return MWAX_ERR_NULL;
    return mwax_corr_process_batch(h, d_volt, (size_t)h->T * h->N, 0, 1, 1, d_vis, stream);
}

int mwax_corr_process_host(mwax_corr_t *h, const int8_t *h_volt, size_t row_pitch, size_t coarse_pitch, int n_dumps,
                           int n_coarse, float *h_vis, void *stream)
{
    if (!h || !h_volt || !h_vis) return MWAX_ERR_NULL;
    // every argument check comes before the first enqueue; with MWAX_OPT_ACCUMULATE the sum would go into the staging
    // buffer, not into h_vis: refused rather than silently wrong
    if (n_dumps < 1 || n_coarse < 1 || row_pitch < (size_t)n_dumps * h->T * h->N || h->accumulate || !h->tables_ready ||
        !on_device(h->device))
        return MWAX_ERR_INVALID_ARG;
    if ((h->d_delay || h->d_phase) && h->d_row_stride < (size_t)n_dumps * h->T) return MWAX_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t dump_samples = (size_t)h->T * h->N;
    const size_t row_samples = (size_t)n_dumps * dump_samples;
    const size_t in_bytes = (size_t)h->n * row_samples * 2;
    const size_t dump_out = mwax_corr_output_bytes(h);
    const size_t out_bytes = (size_t)n_dumps * dump_out;
    if (h->in_bytes < in_bytes) {
        cudaFree(h->d_in); h->d_in = nullptr; h->in_bytes = 0;
        if (cudaMalloc(reinterpret_cast<void **>(&h->d_in), in_bytes) != cudaSuccess) { cudaGetLastError(); return MWAX_ERR_NOMEM; }
        h->in_bytes = in_bytes;
    }
    if (h->out_bytes < out_bytes) {
        cudaFree(h->d_out); h->d_out = nullptr; h->out_bytes = 0;
        if (cudaMalloc(reinterpret_cast<void **>(&h->d_out), out_bytes) != cudaSuccess) { cudaGetLastError(); return MWAX_ERR_NOMEM; }
        h->out_bytes = out_bytes;
    }
    // Three streams so that PCIe runs in both directions under the kernels: dump d + 1 travels host -> device and
    // dump d - 1 device -> host while dump d is correlated on the caller's stream.
    if (!h->s_in && cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking) != cudaSuccess) return note_cuda(&h->last_cuda);
    if (!h->s_out && cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking) != cudaSuccess) return note_cuda(&h->last_cuda);
    const int n_ev = n_dumps * n_coarse;
    while ((int)h->ev_in.size() < n_ev) {
        cudaEvent_t a, b;
        if (cudaEventCreateWithFlags(&a, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&b, cudaEventDisableTiming) != cudaSuccess)
            return note_cuda(&h->last_cuda);
        h->ev_in.push_back(a);
        h->ev_done.push_back(b);
    }
    if (!h->ev_start) {
        if (cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->ev_copied, cudaEventDisableTiming) != cudaSuccess)
            return note_cuda(&h->last_cuda);
        for (int q = 0; q < 8; ++q)
            if (cudaEventCreateWithFlags(&h->ev_part[q], cudaEventDisableTiming) != cudaSuccess) return note_cuda(&h->last_cuda);
    }
    // once work is in flight an error must not return while copies still reference the caller's host buffers
    auto fail = [&](int rc) {
        cudaStreamSynchronize(h->s_in);
        cudaStreamSynchronize(h->s_out);
        cudaStreamSynchronize(st);
        if (rc == MWAX_ERR_CUDA) note_cuda(&h->last_cuda);
        return rc;
    };
    // the copy streams start after whatever the caller has already queued on `stream`
    cudaEventRecord(h->ev_start, st);
    cudaStreamWaitEvent(h->s_in, h->ev_start, 0);
    cudaStreamWaitEvent(h->s_out, h->ev_start, 0);
    const size_t vis_floats = dump_out / sizeof(float);
    for (int c = 0; c < n_coarse; ++c)
        for (int d = 0; d < n_dumps; ++d) {
            const int e = c * n_dumps + d;
            // staging is reused by the next coarse channel: its dump d may be overwritten once it has been correlated
            if (c > 0) cudaStreamWaitEvent(h->s_in, h->ev_done[e - n_dumps], 0);
            if (cudaMemcpy2DAsync(h->d_in + 2 * d * dump_samples, row_samples * 2,
                                  h_volt + 2 * (c * coarse_pitch + d * dump_samples), row_pitch * 2, dump_samples * 2, h->n,
                                  cudaMemcpyHostToDevice, h->s_in) != cudaSuccess)
                return fail(MWAX_ERR_CUDA);
            cudaEventRecord(h->ev_in[e], h->s_in);
            cudaStreamWaitEvent(st, h->ev_in[e], 0);
            if (c > 0) cudaStreamWaitEvent(st, h->ev_copied, 0);   // previous channel's visibilities have left d_out
            int rc = f_stage_impl(h, h->d_in + 2 * d * dump_samples, row_samples, d * h->T, c, st);
            if (rc != MWAX_OK) return fail(rc);
            // Nothing hides the device -> host copy of the LAST dump: it is correlated in HOST_PARTS channel ranges and each
            // range leaves while the next is computed (plain schedule only; earlier dumps travel under the next dump's work).
            int parts = 1;
            if (e == n_ev - 1 && h->C >= 8 && mwax_corr_x_edge_runs(h) <= 0) parts = HOST_PARTS;
            for (int q = 0; q < parts; ++q) {
                const int c0 = (int)(((long long)q * h->C) / parts), c1 = (int)(((long long)(q + 1) * h->C) / parts);
                rc = x_stage_range(h, h->d_out + (size_t)d * vis_floats, c0, c1 - c0, st);
                if (rc != MWAX_OK) return fail(rc);
                cudaEventRecord(q == parts - 1 ? h->ev_done[e] : h->ev_part[q], st);
                cudaStreamWaitEvent(h->s_out, q == parts - 1 ? h->ev_done[e] : h->ev_part[q], 0);
                const size_t off = (size_t)c0 * (dump_out / h->C), len = (size_t)(c1 - c0) * (dump_out / h->C);
                if (cudaMemcpyAsync(reinterpret_cast<char *>(h_vis) + (size_t)c * out_bytes + (size_t)d * dump_out + off,
                                    reinterpret_cast<char *>(h->d_out + (size_t)d * vis_floats) + off, len, cudaMemcpyDeviceToHost,
                                    h->s_out) != cudaSuccess)
                    return fail(MWAX_ERR_CUDA);
            }
            if (d == n_dumps - 1) cudaEventRecord(h->ev_copied, h->s_out);
        }
    // join: the caller's stream continues after the last copy; the call itself returns when everything has landed
    cudaEventRecord(h->ev_copied, h->s_out);
    cudaStreamWaitEvent(st, h->ev_copied, 0);
    if (cudaStreamSynchronize(st) != cudaSuccess) return note_cuda(&h->last_cuda);
    return MWAX_OK;
}

size_t mwax_corr_input_bytes(const mwax_corr_t *h) { return h ? (size_t)h->n * h->T * h->N * 2 : 0; }
size_t mwax_corr_output_bytes(const mwax_corr_t *h)
{
    return h ? (size_t)h->C * ((size_t)h->n * (h->n + 1) / 2) * 8 : 0;
}
int mwax_corr_set_workspace(mwax_corr_t *h, void *d_ws, size_t bytes)
{
    if (!h || !d_ws) return MWAX_ERR_NULL;
    if (bytes < h->y_bytes || (reinterpret_cast<uintptr_t>(d_ws) & 255u)) return MWAX_ERR_INVALID_ARG;
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    if (cudaMemset(d_ws, 0, h->y_bytes) != cudaSuccess) return note_cuda(&h->last_cuda);   // pad columns must read as zero
    CUtensorMap m1, m2;      // both maps are encoded before anything in the handle changes
    int rc = encode_z_map(&m1, false, d_ws, (uint64_t)h->pitch, (uint64_t)h->pitch * 2, (uint64_t)h->T, (uint64_t)h->K, 64);
    if (rc == MWAX_OK)
        rc = encode_z_map(&m2, false, d_ws, (uint64_t)h->pitch, (uint64_t)h->pitch * 2, (uint64_t)h->T * h->K, 1, 64);
    if (rc != MWAX_OK) return rc;
    if (cudaDeviceSynchronize() != cudaSuccess) return note_cuda(&h->last_cuda);
    if (h->y_owned) cudaFree(h->d_Y);
    h->tmap = m1;
    h->tmap_flat = m2;
    h->d_Y = reinterpret_cast<__half *>(d_ws);
    h->y_owned = false;
    return MWAX_OK;
}

size_t mwax_corr_mwax_order_bytes(const mwax_corr_t *h)
{
    if (!h || (h->n & 1)) return 0;
    const size_t nt = (size_t)h->n / 2;
    return nt * (nt + 1) / 2 * (size_t)h->C * 4 * 8;
}

int mwax_corr_to_mwax_order(mwax_corr_t *h, const float *d_vis, float *d_out, float *d_weights, void *stream)
{
    return mwax_corr_to_mwax_order_weighted(h, d_vis, nullptr, 0, 0, d_out, d_weights, stream);
}

int mwax_corr_to_mwax_order_weighted(mwax_corr_t *h, const float *d_vis, const uint8_t *d_flags, int n_sub, int normalise,
                                     float *d_out, float *d_weights, void *stream)
{
    if (!h || !d_vis || !d_out) return MWAX_ERR_NULL;
    if (d_flags && n_sub < 1) return MWAX_ERR_INVALID_ARG;
    if (h->n & 1) return MWAX_ERR_UNSUPPORTED;              // tiles are pairs of signal paths (x, y)
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    mwax::OrderParams op;
    op.vis = reinterpret_cast<const float2 *>(d_vis); op.out = reinterpret_cast<float2 *>(d_out); op.weights = d_weights;
    op.n_tiles = h->n / 2; op.C = h->C; op.chan_stride = (long long)h->n * (h->n + 1) / 2;
    op.flags = d_flags; op.n_sub = n_sub; op.normalise = (d_flags && normalise) ? 1 : 0;
    dim3 grid((op.n_tiles + mwax::ORD_TA - 1) / mwax::ORD_TA, op.n_tiles, (op.C + mwax::ORD_TC - 1) / mwax::ORD_TC);
    if (grid.y > 65535 || grid.z > 65535) return MWAX_ERR_UNSUPPORTED;
    mwax::mwax_order_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(op);
    ++h->launches;
    return note_cuda(&h->last_cuda);
}

size_t mwax_corr_workspace_bytes(const mwax_corr_t *h) { return h ? h->y_bytes : 0; }
long long mwax_corr_launch_count(const mwax_corr_t *h) { return h ? h->launches : 0; }
int mwax_corr_last_cuda_error(const mwax_corr_t *h) { return h ? h->last_cuda : 0; }

int mwax_corr_destroy(mwax_corr_t *h)
{
    if (!h) return MWAX_OK;
    free_tables(h);
    cudaFree(h->d_tw);
    if (h->y_owned) cudaFree(h->d_Y);
    cudaFree(h->d_in);
    cudaFree(h->d_out);
    for (cudaEvent_t e : h->ev_in) cudaEventDestroy(e);
    for (cudaEvent_t e : h->ev_done) cudaEventDestroy(e);
    if (h->ev_start) cudaEventDestroy(h->ev_start);
    if (h->ev_copied) cudaEventDestroy(h->ev_copied);
    for (cudaEvent_t e : h->ev_part) if (e) cudaEventDestroy(e);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    delete h;
    return MWAX_OK;
}

// ------------------------------------------------------------------------------------------------ int8 X-only
mwax_xcorr_t *mwax_xcorr_i8_create(int n_inputs, int n_chan, int n_time)
{
    g_last_error = MWAX_OK;
    if (n_inputs < 1 || n_chan < 1 || n_time < 1) { g_last_error = MWAX_ERR_INVALID_ARG; return nullptr; }
    if (n_inputs > 8128 || n_time > 65535) { g_last_error = MWAX_ERR_UNSUPPORTED; return nullptr; }
    int sm = 0, dev = 0;
    if ((g_last_error = check_device(&sm, &dev)) != MWAX_OK) return nullptr;
    DevicePlan dp;
    if ((g_last_error = prepare_device(dev, sm, &dp)) != MWAX_OK) return nullptr;
    mwax_xcorr *h = new (std::nothrow) mwax_xcorr();
    if (!h) { g_last_error = MWAX_ERR_NOMEM; return nullptr; }
    h->n = n_inputs; h->n_chan = n_chan; h->n_time = n_time; h->sm_count = sm; h->last_cuda = 0;
    h->device = dev; h->dp = dp;
    h->pitch = ((2 * n_inputs + 15) / 16) * 16;
    std::vector<int> tap(n_chan);
    for (int c = 0; c < n_chan; ++c) tap[c] = c;
    std::vector<uint8_t> ptiles;
    build_pair_tiles(n_inputs, ptiles);
    h->n_ptiles = (int)ptiles.size() / 4;
    if ((g_last_error = upload(&h->d_tap_start, tap)) != MWAX_OK ||
        (g_last_error = upload(&h->d_ptiles, ptiles)) != MWAX_OK) {
        mwax_xcorr_i8_destroy(h); return nullptr;
    }
    return h;
}

// channels [c0, c0 + cnt) of a resident buffer `d_z` with row pitch `pitch` bytes (a multiple of 16, base 16-byte aligned)
static int xcorr_i8_range(mwax_xcorr_t *h, const int8_t *d_z, int pitch, int32_t *d_vis, int c0, int cnt, cudaStream_t st)
{
    CUtensorMap tmap;   // columns past 2n read as zero (TMA out-of-bounds fill): that pads partial tiles and ragged rows
    int rc = encode_z_map(&tmap, true, d_z, (uint64_t)2 * h->n, (uint64_t)pitch, (uint64_t)h->n_time, (uint64_t)h->n_chan, 128);
    if (rc != MWAX_OK) return rc;
    mwax::XParams xp;
    xp.n_inputs = h->n; xp.T = h->n_time; xp.K = h->n_chan; xp.n_out = cnt; xp.n_tiles = h->n_ptiles;
    xp.tiles = h->d_ptiles; xp.tap_start = h->d_tap_start + c0; xp.n_taps = 1; xp.scale = nullptr;
    xp.out_chan_stride = (long long)h->n * (h->n + 1) / 2;
    xp.out = d_vis + (size_t)c0 * (size_t)xp.out_chan_stride * 2;
    xp.accumulate = 0;
    xp.edge_runs = 0;
    rc = launch_x_pair<true>(tmap, tmap, xp, h->dp.pairs_i8, st);
    if (rc != MWAX_OK) note_cuda(&h->last_cuda);
    return rc;
}

int mwax_xcorr_i8_process(mwax_xcorr_t *h, const int8_t *d_z, int32_t *d_vis, void *stream)
{
    if (!h || !d_z || !d_vis) return MWAX_ERR_NULL;
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const bool direct = (h->pitch == 2 * h->n) && ((reinterpret_cast<uintptr_t>(d_z) & 15u) == 0);
    if (direct) return xcorr_i8_range(h, d_z, h->pitch, d_vis, 0, h->n_chan, st);
    // TMA needs a 16-byte aligned base and row pitch: a ragged (n_inputs % 8 != 0) or misaligned buffer is first copied,
    // on the device, into rows of the next multiple of 16 bytes (one extra pass over the input; the pad bytes are never
    // used: the tensor map's inner extent stays 2n)
    const size_t rows = (size_t)h->n_chan * h->n_time;
    if (!h->d_pad && cudaMalloc(reinterpret_cast<void **>(&h->d_pad), rows * (size_t)h->pitch) != cudaSuccess) {
        cudaGetLastError();
        return MWAX_ERR_NOMEM;
    }
    if (cudaMemcpy2DAsync(h->d_pad, (size_t)h->pitch, d_z, (size_t)2 * h->n, (size_t)2 * h->n, rows, cudaMemcpyDeviceToDevice, st) !=
        cudaSuccess)
        return note_cuda(&h->last_cuda);
    return xcorr_i8_range(h, h->d_pad, h->pitch, d_vis, 0, h->n_chan, st);
}

int mwax_xcorr_i8_process_host(mwax_xcorr_t *h, const int8_t *h_z, int32_t *h_vis, void *stream)
{
    if (!h || !h_z || !h_vis) return MWAX_ERR_NULL;
    if (!on_device(h->device)) return MWAX_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t rows = (size_t)h->n_chan * h->n_time;
    const size_t chan_out = ((size_t)h->n * (h->n + 1) / 2) * 8;
    if (!h->d_in && cudaMalloc(reinterpret_cast<void **>(&h->d_in), rows * (size_t)h->pitch) != cudaSuccess) { cudaGetLastError(); return MWAX_ERR_NOMEM; }
    if (!h->d_out && cudaMalloc(reinterpret_cast<void **>(&h->d_out), (size_t)h->n_chan * chan_out) != cudaSuccess) { cudaGetLastError(); return MWAX_ERR_NOMEM; }
    if (!h->s_in) {
        if (cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->ev_copied, cudaEventDisableTiming) != cudaSuccess)
            return note_cuda(&h->last_cuda);
        for (int q = 0; q < HOST_PARTS; ++q)
            if (cudaEventCreateWithFlags(&h->ev_in[q], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&h->ev_done[q], cudaEventDisableTiming) != cudaSuccess)
                return note_cuda(&h->last_cuda);
    }
    auto fail = [&](int rc) {
        cudaStreamSynchronize(h->s_in);
        cudaStreamSynchronize(h->s_out);
        cudaStreamSynchronize(st);
        if (rc == MWAX_ERR_CUDA) note_cuda(&h->last_cuda);
        return rc;
    };
    // channels are independent: range q + 1 travels host -> device and range q - 1 device -> host while range q is
    // correlated (the host rows are copied straight into 16-byte pitched rows, so any n_inputs costs no extra pass here)
    cudaEventRecord(h->ev_start, st);
    cudaStreamWaitEvent(h->s_in, h->ev_start, 0);
    cudaStreamWaitEvent(h->s_out, h->ev_start, 0);
    const int parts = h->n_chan >= HOST_PARTS ? HOST_PARTS : 1;
    for (int q = 0; q < parts; ++q) {
        const int c0 = (int)(((long long)q * h->n_chan) / parts), c1 = (int)(((long long)(q + 1) * h->n_chan) / parts);
        const size_t r0 = (size_t)c0 * h->n_time, nr = (size_t)(c1 - c0) * h->n_time;
        if (cudaMemcpy2DAsync(h->d_in + r0 * (size_t)h->pitch, (size_t)h->pitch, h_z + r0 * (size_t)2 * h->n, (size_t)2 * h->n,
                              (size_t)2 * h->n, nr, cudaMemcpyHostToDevice, h->s_in) != cudaSuccess)
            return fail(MWAX_ERR_CUDA);
        cudaEventRecord(h->ev_in[q], h->s_in);
        cudaStreamWaitEvent(st, h->ev_in[q], 0);
        int rc = xcorr_i8_range(h, h->d_in, h->pitch, h->d_out, c0, c1 - c0, st);
        if (rc != MWAX_OK) return fail(rc);
        cudaEventRecord(h->ev_done[q], st);
        cudaStreamWaitEvent(h->s_out, h->ev_done[q], 0);
        if (cudaMemcpyAsync(reinterpret_cast<char *>(h_vis) + (size_t)c0 * chan_out, reinterpret_cast<char *>(h->d_out) + (size_t)c0 * chan_out,
                            (size_t)(c1 - c0) * chan_out, cudaMemcpyDeviceToHost, h->s_out) != cudaSuccess)
            return fail(MWAX_ERR_CUDA);
    }
    cudaEventRecord(h->ev_copied, h->s_out);
    cudaStreamWaitEvent(st, h->ev_copied, 0);
    if (cudaStreamSynchronize(st) != cudaSuccess) return note_cuda(&h->last_cuda);
    return MWAX_OK;
}

int mwax_xcorr_i8_destroy(mwax_xcorr_t *h)
{
    if (!h) return MWAX_OK;
    cudaFree(h->d_tap_start);
    cudaFree(h->d_ptiles);
    cudaFree(h->d_pad);
    cudaFree(h->d_in);
    cudaFree(h->d_out);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    if (h->ev_start) cudaEventDestroy(h->ev_start);
    if (h->ev_copied) cudaEventDestroy(h->ev_copied);
    for (int q = 0; q < HOST_PARTS; ++q) {
        if (h->ev_in[q]) cudaEventDestroy(h->ev_in[q]);
        if (h->ev_done[q]) cudaEventDestroy(h->ev_done[q]);
    }
    delete h;
    return MWAX_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ allocation-free entry
// mwax_corr_process_static (include/mwax_corr.h): the whole F -> X pass of mwax_corr_process for callers that may not
// call cudaMalloc (CUDA-graph capture, tight serving loops, harnesses that forbid it).  The fp16 spectra Y that the F
// kernel writes and the X kernel contracts — the one piece of scratch memory on the path — live in this file-scope
// array instead of a cudaMalloc'ed workspace, followed by the X kernel's three small tables, which a one-block kernel
// fills on the device from the call's arguments (no host-to-device copy either).  Every GPU that loads the library holds
// the array until the process exits; every call on a device shares it, so calls that overlap on the GPU race.
// In HOST code the array's name is only a stand-in: the device address comes from cudaGetSymbolAddress, once per device.
static __device__ __align__(256) unsigned char g_static_ws[MWAX_STATIC_Y_BYTES + MWAX_STATIC_TABLE_BYTES];

namespace {

struct StaticTables {          // offsets into the table region that follows the Y scratch
    static constexpr size_t TILES = 0;              // uint8 [n_tiles][4], n_tiles <= 2080 (n <= 8128)
    static constexpr size_t TAP = 16 * 1024;        // int   [C], C <= 512
    static constexpr size_t SCALE = 32 * 1024;      // float [C]
};
static_assert(MWAX_STATIC_TABLE_BYTES >= 48 * 1024 && MWAX_STATIC_Y_BYTES % 256 == 0, "table region layout");

// the tables build_tables() uploads, for the default options (centre-symmetric averaging, DC excluded): PAPER.md L290-298
__global__ void static_tables_kernel(uint8_t *tiles, int *tap, float *scale, int n_tiles, int C, int K, int F, float sc, float sc_c0)
{
    for (int e = threadIdx.x; e < n_tiles; e += blockDim.x) {
        int mi = 0;
        while ((mi + 1) * (mi + 2) / 2 <= e) ++mi;                   // e = mi (mi + 1) / 2 + nj, nj <= mi
        const int nj = e - mi * (mi + 1) / 2;
        tiles[4 * e + 0] = (uint8_t)mi; tiles[4 * e + 1] = (uint8_t)nj; tiles[4 * e + 2] = 0; tiles[4 * e + 3] = 0;
    }
    const int c0 = C / 2, half = K / 2, dmax = (F % 2) ? (F - 1) / 2 : F / 2;
    for (int c = threadIdx.x; c < C; c += blockDim.x) {
        const int u0 = (c - c0) * F - dmax;
        tap[c] = (F == 1) ? c : ((u0 + half) % K + K) % K;
        scale[c] = (F > 1 && c == c0) ? sc_c0 : sc;
    }
}

struct StaticDevice {
    unsigned char *ws;         // device address of g_static_ws on this device
    DevicePlan dp;
    int sm_count;
};

// once per device, with that device current: kernel attributes (prepare_device) and the array's device address
int static_device(StaticDevice *out)
{
    static std::mutex mu;
    static std::map<int, StaticDevice> done;
    int sm = 0, dev = 0, rc;
    if ((rc = check_device(&sm, &dev)) != MWAX_OK) return rc;
    std::lock_guard<std::mutex> lock(mu);
    auto it = done.find(dev);
    if (it != done.end()) { *out = it->second; return MWAX_OK; }
    StaticDevice sd;
    sd.sm_count = sm;
    if ((rc = prepare_device(dev, sm, &sd.dp)) != MWAX_OK) return rc;
    void *p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_ws) != cudaSuccess || !p) { cudaGetLastError(); return MWAX_ERR_CUDA; }
    sd.ws = static_cast<unsigned char *>(p);
    done[dev] = sd;
    *out = sd;
    return MWAX_OK;
}

}  // namespace

extern "C" {

size_t mwax_corr_static_workspace_max(void) { return (size_t)MWAX_STATIC_Y_BYTES; }

int mwax_corr_process_static(const int8_t *d_volt, float *d_vis, int n_inputs, int n_fft, int t_int, int f_avg, void *stream)
{
    if (!d_volt || !d_vis) return MWAX_ERR_NULL;
    if (n_inputs < 1 || n_fft < 1 || t_int < 1 || f_avg < 1) return MWAX_ERR_INVALID_ARG;
    // the register kernels keep their tables in the kernel parameters: no device table, hence these four lengths only
    if ((n_fft != 64 && n_fft != 128 && n_fft != 256 && n_fft != 512) || n_fft % f_avg != 0 || n_inputs > 8128) return MWAX_ERR_UNSUPPORTED;
    if (reinterpret_cast<uintptr_t>(d_volt) & 15u) return MWAX_ERR_INVALID_ARG;     // 16-byte loads (no scalar-load kernel here)
    const int N = n_fft, K = n_fft, T = t_int, F = f_avg, C = K / F, n = n_inputs;
    const int pitch = ((2 * n + 63) / 64) * 64;                                      // fp16 elements per Y row, as create()
    const unsigned long long y_bytes = (unsigned long long)K * (unsigned long long)T * (unsigned long long)pitch * sizeof(__half);
    if (y_bytes > (unsigned long long)MWAX_STATIC_Y_BYTES) return MWAX_ERR_TOO_LARGE;
    StaticDevice sd;
    int rc = static_device(&sd);
    if (rc != MWAX_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    __half *Y = reinterpret_cast<__half *>(sd.ws);
    unsigned char *tab = sd.ws + MWAX_STATIC_Y_BYTES;
    uint8_t *d_tiles = tab + StaticTables::TILES;
    int *d_tap = reinterpret_cast<int *>(tab + StaticTables::TAP);
    float *d_scale = reinterpret_cast<float *>(tab + StaticTables::SCALE);

    // the array keeps the last call's contents.  Every column of an input < n is rewritten by the F kernel below; the pad
    // columns (2n not a multiple of 64) must read as zero and may hold another shape's spectra: cleared here
    if (pitch != 2 * n && cudaMemsetAsync(Y, 0, (size_t)y_bytes, st) != cudaSuccess) { cudaGetLastError(); return MWAX_ERR_CUDA; }

    // averaging geometry of build_tables(), default options
    const int lg = (int)std::ceil(std::log2((double)N) / 2.0);
    const double s = std::ldexp(1.0, -lg);
    const float sc = (float)(1.0 / (s * s * F));
    const float sc_c0 = F > 1 ? (float)((1.0 / (s * s * F)) * (double)F / (double)(F - 1)) : sc;
    const int n_tiles = ((n + 127) / 128) * ((n + 127) / 128 + 1) / 2;
    const int n_taps = (F == 1) ? 1 : 2 * ((F % 2) ? (F - 1) / 2 : F / 2) + 1;
    static_tables_kernel<<<1, 256, 0, st>>>(d_tiles, d_tap, d_scale, n_tiles, C, K, F, sc, sc_c0);

    // F stage: f_stage_impl()'s register-kernel launch with Y = the static array
    mwax::FParams fp;
    std::memset(&fp, 0, sizeof(fp));
    fp.volt = d_volt; fp.row_pitch = (long long)T * N; fp.sample0 = 0;
    fp.n_inputs = n; fp.N = N; fp.K = K; fp.T = T; fp.G = 32; fp.vec_ok = 1;
    fp.in_scale = (float)s; fp.chan_scale = F > 1 ? 1 : 0;
    fp.Y = reinterpret_cast<__half2 *>(Y); fp.pitch2 = pitch / 2;
    fp.y_p_stride = (unsigned)T * (unsigned)(pitch / 2); fp.y_t_stride = (unsigned)(pitch / 2);
    const int R1 = N <= 128 ? 8 : 16, R2 = N / R1;
    for (int r = 0; r < R2; ++r)
        for (int k1 = 0; k1 < R1; ++k1) {
            const double a = 2.0 * M_PI * (double)((r * k1) % N) / (double)N;
            fp.twc[r * R1 + k1] = make_float2((float)std::cos(a), (float)(-std::sin(a)));
        }
    for (int p = 0; p < K; ++p) {
        const int u = p - K / 2;
        fp.swc[p] = (F > 1 && F % 2 == 0 && (((u - F / 2) % F) + F) % F == 0) ? (float)std::sqrt(0.5) : 1.0f;
    }
    if (F > 1) fp.swc[K / 2] = 0.0f;                                                 // DC excluded (L290-294)
    const int groups = (n + 31) / 32;
    long long fpc = ((long long)groups * T) / ((long long)sd.sm_count * 24);
    fpc = fpc < 1 ? 1 : (fpc > 32 ? 32 : fpc);
    fp.frames_per_cta = (int)fpc;
    const int chunks = (T + (int)fpc - 1) / (int)fpc;
    const bool scale = fp.chan_scale != 0;
    switch (N) {
        case 64: launch_f_pow2<64, 8, 16>(fp, true, scale, false, groups, chunks, st); break;
        case 128: launch_f_pow2<128, 8, 16>(fp, true, scale, false, groups, chunks, st); break;
        case 256: launch_f_pow2<256, 16, 32>(fp, true, scale, false, groups, chunks, st); break;
        default: launch_f_pow2<512, 16, 32>(fp, true, scale, false, groups, chunks, st); break;
    }
    if (cudaGetLastError() != cudaSuccess) return MWAX_ERR_CUDA;

    // X stage: x_stage_range()'s launch over all channels; the tensor maps are encoded on the host (no device memory)
    CUtensorMap tmap, tmap_flat;
    if ((rc = encode_z_map(&tmap, false, Y, (uint64_t)pitch, (uint64_t)pitch * 2, (uint64_t)T, (uint64_t)K, 64)) != MWAX_OK) return rc;
    if ((rc = encode_z_map(&tmap_flat, false, Y, (uint64_t)pitch, (uint64_t)pitch * 2, (uint64_t)T * K, 1, 64)) != MWAX_OK) return rc;
    mwax::XParams xp;
    xp.n_inputs = n; xp.T = T; xp.K = K; xp.n_out = C; xp.n_tiles = n_tiles;
    xp.tiles = d_tiles; xp.tap_start = d_tap; xp.n_taps = n_taps; xp.scale = d_scale;
    xp.out_chan_stride = (long long)n * (n + 1) / 2;
    xp.out = d_vis;
    xp.accumulate = 0;
    xp.edge_runs = (n_taps == F + 1) ? choose_edge_runs(C, F, T, n_tiles, sd.dp.pairs_f16_edge, -1) : 0;
    rc = xp.edge_runs > 0 ? launch_x_pair<false, true>(tmap, tmap_flat, xp, sd.dp.pairs_f16_edge, st)
                          : launch_x_pair<false>(tmap, tmap_flat, xp, sd.dp.pairs_f16, st);
    if (rc != MWAX_OK) cudaGetLastError();
    return rc;
}

}  // extern "C"
