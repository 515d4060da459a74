// mwax_order.cuh — MWAX_ORDER emitter (§2.7, Figs 8-9): re-index the
// native packed lower triangle V[c][i(i+1)/2 + j] (signal paths i >= j) into the instrument's output order
//     M[baseline(antA <= antB, row by row)][channel][xx, xy, yx, yy]    complex fp32
// followed by the weights block W[baseline][4] (all 1.0, L328).  Signal path i = 2 tile + pol (reading Q20);
// element (antA, antB, ch, pq) = sum X_{antA,p} conj(X_{antB,q}) (reading Q21) = V[i][j] if i >= j else conj(V[j][i])
// with i = 2 antA + p, j = 2 antB + q.  The paper does this on the CPU in two passes after a device-to-host copy
// (0.6-1.8 s per 8 s subfile, Table 2); here it is one pass at HBM speed: a block takes antenna antB, 16
// antennas antA and 16 channels, reads the two native rows 2 antB, 2 antB + 1 as 256-byte runs, turns the tile in
// shared memory and writes 512-byte runs of each output row.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace mwax {

struct OrderParams {
    const float2 *vis;     // native [C][n(n+1)/2]
    float2 *out;           // [n_tiles(n_tiles+1)/2][C][4]
    float *weights;        // [n_tiles(n_tiles+1)/2][4] or nullptr
    int n_tiles, C;
    long long chan_stride; // n(n+1)/2
    // occupancy weights (§4.1): zeroing flags [2 n_tiles][n_sub] bytes, 1 = that sub-block of that
    // signal path was zeroed; nullptr = everything valid (weights 1.0).  normalise: divide each visibility by its weight.
    const uint8_t *flags;
    int n_sub, normalise;
};

constexpr int ORD_TA = 16, ORD_TC = 16;

__global__ void __launch_bounds__(256) mwax_order_kernel(const OrderParams P)
{
    __shared__ float2 tile[ORD_TC][2][2 * ORD_TA + 1];
    __shared__ float wt[ORD_TA][4];
    const int b = blockIdx.y;                                  // antB
    const int a0 = blockIdx.x * ORD_TA;                        // first antA of the tile
    const int c0 = blockIdx.z * ORD_TC;
    if (a0 > b) return;
    const int na = min(ORD_TA, b - a0 + 1);                    // antennas antA <= antB in this tile
    const int nc = min(ORD_TC, P.C - c0);

    // native rows i = 2b + q, columns j = 2 a0 .. 2 a0 + 2 na - 1 (row 2b stops at column 2b: its diagonal)
    for (int e = threadIdx.x; e < ORD_TC * 2 * 2 * ORD_TA; e += blockDim.x) {
        const int col = e % (2 * ORD_TA), q = (e / (2 * ORD_TA)) & 1, cl = e / (4 * ORD_TA);
        const long long i = 2ll * b + q, j = 2ll * a0 + col;
        float2 v = make_float2(0.f, 0.f);
        if (cl < nc && col < 2 * na && j <= i) v = P.vis[(long long)(c0 + cl) * P.chan_stride + i * (i + 1) / 2 + j];
        tile[cl][q][col] = v;
    }
    // weight(antA, antB, pq) = fraction of sub-blocks in which BOTH signal paths were fully populated
    for (int e = threadIdx.x; e < na * 4; e += blockDim.x) {
        float w = 1.0f;
        if (P.flags) {
            const uint8_t *fa = P.flags + (size_t)(2 * (a0 + (e >> 2)) + ((e >> 1) & 1)) * P.n_sub;
            const uint8_t *fb = P.flags + (size_t)(2 * b + (e & 1)) * P.n_sub;
            int both = 0;
            for (int sb = 0; sb < P.n_sub; ++sb) both += (!fa[sb] && !fb[sb]);
            w = (float)both / (float)P.n_sub;
        }
        wt[e >> 2][e & 3] = w;
    }
    __syncthreads();

    // output rows (antA = a0 + al, antB = b): [channel][p][q], 16 channels x 4 products = 512 contiguous bytes
    for (int e = threadIdx.x; e < na * ORD_TC * 4; e += blockDim.x) {
        const int pq = e & 3, cl = (e >> 2) % ORD_TC, al = e / (4 * ORD_TC);
        if (cl >= nc) continue;
        const int p = pq >> 1, q = pq & 1;
        const int a = a0 + al;
        float2 v;
        if (a < b || p <= q) {                                 // i = 2a + p <= j = 2b + q: conj(V[j][i])  (equal: a real auto)
            v = tile[cl][q][2 * al + p];
            v.y = -v.y;
            if (a == b && p == q) v.y = 0.0f;                  // -0.0 -> +0.0 for the autos
        } else {                                               // a == b, (p, q) = (1, 0): V[2a+1][2a] as stored
            v = tile[cl][1][2 * al];
        }
        if (P.normalise) {
            const float w = wt[al][pq];
            if (w > 0.0f) { v.x /= w; v.y /= w; }
        }
        const long long row = (long long)a * P.n_tiles - (long long)a * (a - 1) / 2 + (b - a);
        P.out[(row * P.C + c0 + cl) * 4 + pq] = v;
    }
    if (P.weights && blockIdx.z == 0) {
        for (int e = threadIdx.x; e < na * 4; e += blockDim.x) {
            const int a = a0 + (e >> 2);
            const long long row = (long long)a * P.n_tiles - (long long)a * (a - 1) / 2 + (b - a);
            P.weights[row * 4 + (e & 3)] = wt[e >> 2][e & 3];   // 1.0 without flags: "all values are set to 1.0" (L328)
        }
    }
}

}  // namespace mwax
