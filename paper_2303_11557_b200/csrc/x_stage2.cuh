// x_stage2.cuh — the X-stage kernel: persistent CTA PAIRS (tcgen05 cta_group::2), two SMs on one 256 x 256 tile of G.
// 6 warps per CTA: warp 0 = TMA producer (one lane), warp 1 = MMA issuer (+ TMEM owner; all lanes run the loops, one
// elected lane issues), warps 2..5 = epilogue (TMEM lanes 32*(warp%4)..+31).  A work item is (output channel c, G-tile);
// the 128 x 256 accumulator per CTA is double buffered in TMEM so the epilogue of one item overlaps the MMAs of the
// next.  Work items are ordered channel-major so concurrently running pairs share a channel's rows in L2.
//
// Why: ncu on the single-CTA kernel (128 x 256 tiles) shows ~12 TB/s of L2 -> SM operand traffic (253 M sectors in
// 0.68 ms at C3), i.e. the kernel sits on the L2 bandwidth limit, not on the tensor pipe (profiles/r1_ncu_full.md);
// narrower tiles made it slower.  A pair loads per contraction row 128 (A half) + 128 (B half) elements per CTA
// for 128 x 256 outputs per CTA, against 128 + 256 before: a third less L2 traffic per flop.
//
// CTA r of the pair (cluster rank r) holds G rows [256 mi + 128 r, +128) as its A operand and G columns
// [256 nj + 128 r, +128) as its half of B; its TMEM receives the accumulators of ITS 128 rows x all 256 columns, so
// the epilogue is the single-CTA one with mi -> 2 mi + r.  Protocol (cluster rank 0 = leader, issues every MMA):
//   full[s]    leader's barrier: 1 arrival (leader's producer, expect_tx = both CTAs' bytes) + TMA bytes of both CTAs
//   empty[s]   one per CTA: tcgen05.commit (cta_group::2, multicast to both CTAs) when the MMAs have read slot s
//   tfull[a]   one per CTA: commit multicast when an accumulator is complete
//   tempty[a]  leader's barrier: 8 arrivals (4 epilogue warps x 2 CTAs; the follower's arrive remotely)
#pragma once
#include "x_stage.cuh"

namespace mwax {

// kEdge: shared-edge schedule for even F (x_stage.cuh): 4 pipeline stages instead of 6 make room for the 64 KB of
// running sums (128 epilogue threads x 128 folded accumulator elements)
template <bool kInt8, bool kEdge = false>
struct XPairConfig {
    static constexpr int BM = 128;                        // G rows per CTA (256 per pair)
    static constexpr int BN = 256;                        // G columns per pair (128 staged per CTA)
    static constexpr int ESIZE = kInt8 ? 1 : 2;
    static constexpr int BK = kInt8 ? 128 : 64;           // rows (contraction) per pipeline stage
    static constexpr int KINST = kInt8 ? 32 : 16;         // rows per tcgen05.mma
    static constexpr int CHUNK_ELEMS = 128 / ESIZE;       // MN elements per 128-byte TMA box row
    static constexpr int CHUNKS = 128 / CHUNK_ELEMS;      // boxes per operand half (A: 128 rows of G, B: 128 columns)
    static constexpr int CHUNK_BYTES = 128 * BK;
    static constexpr int A_BYTES = CHUNKS * CHUNK_BYTES;  // 16 KB
    static constexpr int STAGE_BYTES = 2 * A_BYTES;       // 32 KB per CTA
    static constexpr int STAGES = kEdge ? 4 : 6;
    static constexpr int ACC_STAGES = 2;
    static constexpr int TMEM_COLS = 512;
    static constexpr int EPI_STAGE_WORDS = 16 * 34;
    static constexpr int EDGE_WORDS_PER_WARP = kEdge ? (BN / 32) * 16 * 32 : 0;   // [chunk][jj][lane] floats
    static constexpr int EDGE_OFF = STAGES * STAGE_BYTES + 4 * EPI_STAGE_WORDS * 4 + 256;
    static constexpr int SMEM_BYTES = 1024 + EDGE_OFF + 4 * EDGE_WORDS_PER_WARP * 4;
    static constexpr uint32_t IDESC = ptx::make_idesc(kInt8 ? 2u : 1u, kInt8 ? 1u : 0u, 256, BN);
    static constexpr int THREADS = 192;
};

// P.tiles: [n_tiles][4] = (mi, nj, 0, 0) in units of 128 inputs (256 rows / columns of G), nj <= mi
template <bool kInt8, bool kEdge = false>
__global__ void __launch_bounds__(192, 1) x_stage_pair_kernel(const __grid_constant__ CUtensorMap tmap,
                                                              const __grid_constant__ CUtensorMap tmap_flat, const XParams P)
{
    using C = XPairConfig<kInt8, kEdge>;
    static_assert(!(kInt8 && kEdge), "the shared-edge schedule belongs to the float path (averaging)");
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;   // SWIZZLE_128B atoms: 1024-byte alignment
    uint8_t *smem_gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t stage_base = smem_base;
    float *epi_stage = reinterpret_cast<float *>(smem_gen + C::STAGES * C::STAGE_BYTES);
    const uint32_t bar_base = smem_base + C::STAGES * C::STAGE_BYTES + 4 * C::EPI_STAGE_WORDS * 4;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (C::STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * C::STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * C::STAGES + 2 + s); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * C::STAGES + 4);
    volatile uint32_t *tmem_slot_gen =
        reinterpret_cast<volatile uint32_t *>(smem_gen + C::STAGES * C::STAGE_BYTES + 4 * C::EPI_STAGE_WORDS * 4 +
                                              8 * (2 * C::STAGES + 4));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();          // 0 = leader
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        ptx::prefetch_tensormap(&tmap_flat);
        for (int s = 0; s < C::STAGES; ++s) {
            ptx::mbar_init(full_bar(s), 1);
            ptx::mbar_init(empty_bar(s), 1);
        }
        for (int s = 0; s < C::ACC_STAGES; ++s) {
            ptx::mbar_init(tfull_bar(s), 1);
            ptx::mbar_init(tempty_bar(s), 8);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc_pair(tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish_pair();
    }
    ptx::tc_fence_before();
    __syncwarp();
    ptx::cluster_sync();                                   // both CTAs' barriers exist before anyone signals them
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    const int n_items = P.n_out * P.n_tiles;
    const int kb_per_tap = (P.T + C::BK - 1) / C::BK;
    // K-loop schedule of one work item (identical in the producer and the MMA issuer).  The taps of an output channel
    // are adjacent channel positions, i.e. ADJACENT ROWS of Y[p][t]: when T >= BK the contraction runs over the flattened
    // rows (p T + t) in whole BK-row blocks through `tmap_flat`, so only the END of a run is a partial block (C4: 51 taps
    // x 200 rows = 159 blocks + 24 rows instead of 51 x (3 blocks + 8 rows)).  The partial block is fetched through the
    // per-channel map, whose rows past T read as zero.  A tap window that wraps past K (cyclic taps, Q8) is
    // two runs.
    const bool flat = (P.n_taps > 1) && (P.T >= C::BK);

    // kEdge: the work of this pair, identical in the three roles.  Unit = (run r of adjacent output channels, tile);
    // fn(c, tile, first tap position, taps, mode) once per accumulator (x_stage.cuh, X_EDGE_*)
    auto for_each_edge_item = [&](auto &&fn) {
        const int n_units = P.edge_runs * P.n_tiles;
        for (int unit = pair; unit < n_units; unit += n_pairs) {
            const int r = unit / P.n_tiles, tile = unit - r * P.n_tiles;
            const int c_a = (int)(((long long)r * P.n_out) / P.edge_runs);
            const int c_b = (int)(((long long)(r + 1) * P.n_out) / P.edge_runs);
            fn(c_a, tile, P.tap_start[c_a], 1, (int)X_EDGE_INIT);
            for (int c = c_a; c < c_b; ++c) {
                int p = P.tap_start[c] + 1;
                if (p >= P.K) p -= P.K;
                fn(c, tile, p, P.n_taps - 2, (int)X_EDGE_ADD);
                p = P.tap_start[c] + P.n_taps - 1;
                if (p >= P.K) p -= P.K;
                fn(c, tile, p, 1, (int)X_EDGE_OUT);
            }
        }
    };
    // K-loop schedule of `nt` adjacent taps from position p0 (cyclic), T >= BK: whole BK-row blocks of the flattened rows,
    // the end of a run through the per-channel map; full(row), tail(row, chan, rows)
    auto k_schedule = [&](int p0, int nt, auto &&full, auto &&tail) {
        const int n1 = min(nt, P.K - p0);
        for (int run = 0; run < 2; ++run) {
            const int pf = run ? 0 : p0, ntr = run ? nt - n1 : n1;
            if (ntr <= 0) continue;
            const int rows = ntr * P.T, nfull = rows / C::BK, tl = rows - nfull * C::BK;
            for (int q = 0; q < nfull; ++q) full(pf * P.T + q * C::BK);
            if (tl) tail(P.T - tl, pf + ntr - 1, tl);
        }
    };

    if (warp == 0) {
        // ------------------------------------------------------------------ TMA producer (one thread in EACH CTA)
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            auto load_block = [&](const CUtensorMap *m, int mi, int nj, int row, int chan) {
                // diagonal tile: this CTA's half of B (columns 256 nj + 128 r ..) IS its A operand (rows 256 mi + 128 r ..):
                // loaded once, the MMA's B descriptor points at the A bytes (a fifth less L2 -> SM traffic at n = 512)
                const bool diag = (mi == nj);
                ptx::mbar_wait(empty_bar(s), ph ^ 1u);
                if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(s), diag ? 2u * C::A_BYTES : 2u * C::STAGE_BYTES);   // both CTAs' bytes
                const uint32_t lead_full = ptx::mapa(full_bar(s), 0);
                const uint32_t a_dst = stage_base + s * C::STAGE_BYTES;
                const uint32_t b_dst = a_dst + C::A_BYTES;
#pragma unroll
                for (int ch = 0; ch < C::CHUNKS; ++ch)
                    ptx::tma_load_3d_pair(a_dst + ch * C::CHUNK_BYTES, m, mi * 256 + (int)rank * 128 + ch * C::CHUNK_ELEMS, row,
                                          chan, lead_full);
                if (!diag) {
#pragma unroll
                    for (int ch = 0; ch < C::CHUNKS; ++ch)
                        ptx::tma_load_3d_pair(b_dst + ch * C::CHUNK_BYTES, m, nj * 256 + (int)rank * 128 + ch * C::CHUNK_ELEMS, row,
                                              chan, lead_full);
                }
                if (++s == C::STAGES) { s = 0; ph ^= 1u; }
            };
            if (kEdge) {
                for_each_edge_item([&](int, int tile, int p0, int nt, int) {
                    const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1];
                    k_schedule(p0, nt, [&](int row) { load_block(&tmap_flat, mi, nj, row, 0); },
                               [&](int row, int chan, int) { load_block(&tmap, mi, nj, row, chan); });
                });
            } else
            for (int item = pair; item < n_items; item += n_pairs) {
                const int c = item / P.n_tiles;
                const int tile = item - c * P.n_tiles;
                const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1];
                const int p0 = P.tap_start[c];
                if (flat) {
                    const int n1 = min(P.n_taps, P.K - p0);
                    for (int run = 0; run < 2; ++run) {
                        const int pf = run ? 0 : p0, nt = run ? P.n_taps - n1 : n1;
                        if (nt <= 0) continue;
                        const int rows = nt * P.T, nfull = rows / C::BK, tail = rows - nfull * C::BK;
                        for (int q = 0; q < nfull; ++q) load_block(&tmap_flat, mi, nj, pf * P.T + q * C::BK, 0);
                        if (tail) load_block(&tmap, mi, nj, P.T - tail, pf + nt - 1);
                    }
                } else {
                    for (int tap = 0; tap < P.n_taps; ++tap) {
                        int p = p0 + tap;
                        if (p >= P.K) p -= P.K;
                        for (int kb = 0; kb < kb_per_tap; ++kb) load_block(&tmap, mi, nj, kb * C::BK, p);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (leader CTA; the whole warp runs
        // the loops so that every operand is warp-uniform, one elected lane issues: see ptx::elect_one)
        if (rank == 0) {
            int s = 0;
            uint32_t ph = 0;
            int as = 0;
            uint32_t aph = 0;
            uint32_t d_tmem = 0, accumulate = 0, b_off = C::A_BYTES;
            auto mma_block = [&](int rows) {
                ptx::mbar_wait(full_bar(s), ph);
                ptx::tc_fence_after();
                const uint32_t a_src = stage_base + s * C::STAGE_BYTES;
                if (ptx::elect_one()) {
                    ptx::mma_block_issue<kInt8, true, C::BK, C::KINST>(a_src, a_src + b_off, C::CHUNK_BYTES, d_tmem, C::IDESC,
                                                                        rows, accumulate);
                    ptx::tc_commit_pair(empty_bar(s), 3);   // frees slot s in BOTH CTAs when these MMAs have read it
                }
                __syncwarp();
                accumulate = 1;
                if (++s == C::STAGES) { s = 0; ph ^= 1u; }
            };
            if (kEdge) {
                for_each_edge_item([&](int, int tile, int p0, int nt, int) {
                    b_off = (P.tiles[4 * tile] == P.tiles[4 * tile + 1]) ? 0u : (uint32_t)C::A_BYTES;   // diagonal tile: B = A
                    ptx::mbar_wait(tempty_bar(as), aph ^ 1u);
                    ptx::tc_fence_after();
                    d_tmem = tmem_base + (uint32_t)(as * C::BN);
                    accumulate = 0;
                    k_schedule(p0, nt, [&](int) { mma_block(C::BK); }, [&](int, int, int rows) { mma_block(rows); });
                    if (ptx::elect_one()) ptx::tc_commit_pair(tfull_bar(as), 3);
                    __syncwarp();
                    if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
                });
            } else
            for (int item = pair; item < n_items; item += n_pairs) {
                const int c = item / P.n_tiles;
                const int tile = item - c * P.n_tiles;
                b_off = (P.tiles[4 * tile] == P.tiles[4 * tile + 1]) ? 0u : (uint32_t)C::A_BYTES;   // diagonal tile: B = A
                ptx::mbar_wait(tempty_bar(as), aph ^ 1u);
                ptx::tc_fence_after();
                d_tmem = tmem_base + (uint32_t)(as * C::BN);
                accumulate = 0;
                if (flat) {
                    const int p0 = P.tap_start[c];
                    const int n1 = min(P.n_taps, P.K - p0);
                    for (int run = 0; run < 2; ++run) {
                        const int nt = run ? P.n_taps - n1 : n1;
                        if (nt <= 0) continue;
                        const int rows = nt * P.T, nfull = rows / C::BK, tail = rows - nfull * C::BK;
                        for (int q = 0; q < nfull; ++q) mma_block(C::BK);
                        if (tail) mma_block(tail);
                    }
                } else {
                    for (int tap = 0; tap < P.n_taps; ++tap)
                        for (int kb = 0; kb < kb_per_tap; ++kb) mma_block(min(C::BK, P.T - kb * C::BK));
                }
                if (ptx::elect_one()) ptx::tc_commit_pair(tfull_bar(as), 3);  // accumulator complete -> both CTAs' epilogues
                __syncwarp();
                if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue (4 warps per CTA, own 128 rows)
        const int q = warp & 3;                       // TMEM lane quadrant this warp may read
        float *stg = epi_stage + (warp - 2) * C::EPI_STAGE_WORDS;
        int as = 0;
        uint32_t aph = 0;
        if (kEdge) {
            float *S = reinterpret_cast<float *>(smem_gen + C::EDGE_OFF) + (warp - 2) * C::EDGE_WORDS_PER_WARP;
            for_each_edge_item([&](int c, int tile, int, int, int mode) {
                const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1];
                const int i_base = mi * 128 + (int)rank * 64 + q * 16;
                const float sc = P.scale[c];
                ptx::mbar_wait(tfull_bar(as), aph);
                ptx::tc_fence_after();
                const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * C::BN);
                x_epilogue_tile<kInt8, kEdge>(P, stg, t_row, c, i_base, nj * 128, C::BN / 32, sc, lane, mode, S);
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster_relaxed(ptx::mapa(tempty_bar(as), 0));
                if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
            });
        } else
        for (int item = pair; item < n_items; item += n_pairs) {
            const int c = item / P.n_tiles;
            const int tile = item - c * P.n_tiles;
            const int mi = P.tiles[4 * tile], nj = P.tiles[4 * tile + 1];
            const int i_base = mi * 128 + (int)rank * 64 + q * 16;      // first input of this warp's 16
            const float sc = kInt8 ? 1.0f : P.scale[c];
            ptx::mbar_wait(tfull_bar(as), aph);
            ptx::tc_fence_after();
            const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * C::BN);
            x_epilogue_tile<kInt8>(P, stg, t_row, c, i_base, nj * 128, C::BN / 32, sc, lane);
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster_relaxed(ptx::mapa(tempty_bar(as), 0));
            if (++as == C::ACC_STAGES) { as = 0; aph ^= 1u; }
        }
    }

    ptx::tc_fence_before();
    __syncwarp();
    ptx::cluster_sync();                                   // no CTA leaves while its pair can still signal or read it
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_pair(tmem_base, C::TMEM_COLS);
    }
}

}  // namespace mwax
