// ptx.cuh — thin inline-PTX wrappers for sm_100a: mbarrier, TMA (cp.async.bulk.tensor), tcgen05 (alloc, mma,
// commit, ld, fences).  Hand-written for this project; no CUTLASS/CuTe.
#pragma once
#include <cstdint>
#include <cuda.h>

namespace mwax {
namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok;
}
// Wait on an mbarrier phase.  try_wait suspends the thread in hardware for a bounded time, so the loop is not a busy
// spin.  The watchdog is WALL-CLOCK based (%globaltimer, checked every 4096 polls): a healthy wait of any length that a
// long integration, a profiler replay or time slicing can produce passes, while a protocol bug still ends in a trap
// (-> cudaErrorLaunchFailure) after 20 s instead of hanging the GPU for ever.  -DMWAX_NO_WATCHDOG removes it.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
#ifdef MWAX_NO_WATCHDOG
    while (!mbar_try_wait(bar, parity)) {}
#else
    uint32_t polls = 0;
    unsigned long long t0 = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++polls & 4095u) == 0) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (t0 == 0) t0 = now;
            else if (now - t0 > 20000000000ull) __trap();
        }
    }
#endif
}

// ---------------------------------------------------------------- TMA
__device__ __forceinline__ void prefetch_tensormap(const CUtensorMap *m)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(m)) : "memory");
}
// ---------------------------------------------------------------- tcgen05
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols)
                 : "memory");
}
__device__ __forceinline__ void tmem_relinquish()
{
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// TMEM -> registers: this warp's 32 lanes x 32 consecutive 32-bit columns (thread L gets lane base+L)
__device__ __forceinline__ void tmem_ld_32x32b_x32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------- CTA pairs (cluster of 2, tcgen05 cta_group::2)
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `saddr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// Arrive on an mbarrier anywhere in the cluster (address from mapa), WITHOUT release semantics: `.release.cluster` compiles to MEMBAR.ALL.GPU + ERRBAR in front of the arrive, i.e. it
// waits until every global store the thread has issued is acknowledged: for an epilogue warp handing its TMEM accumulator
// back that is its whole output tile (ncu, short integrations: 19 % of the epilogue's stall samples on that ERRBAR).  What
// the hand-over must order is the TMEM reads, and those are complete once tcgen05.wait::ld has returned.
__device__ __forceinline__ void mbar_arrive_cluster_relaxed(uint32_t cluster_bar)
{
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
// TMA load issued by either CTA of a pair: data lands in THIS CTA's shared memory, the transaction bytes are
// counted on `cluster_bar`, which may live in the other CTA of the pair (the leader's full barrier)
__device__ __forceinline__ void tma_load_3d_pair(uint32_t dst, const CUtensorMap *m, int c0, int c1, int c2, uint32_t cluster_bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(c0), "r"(c1), "r"(c2), "r"(cluster_bar)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc_pair(uint32_t dst_smem, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish_pair()
{
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// commit of the pair's MMAs: one arrival on the mbarrier at this offset in every CTA of `mask`
__device__ __forceinline__ void tc_commit_pair(uint32_t bar, uint16_t mask)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"(mask)
                 : "memory");
}

// ---------------------------------------------------------------- warp-uniform MMA issue
// One lane of a converged warp, chosen by the hardware.  The MMA warp runs its loops with ALL lanes (so that every
// operand is warp-uniform and lives in uniform registers) and only the tcgen05 instructions sit behind this
// predicate; issuing from inside an `if (lane == 0)` region costs ~20 instructions per MMA (R2UR broadcasts and a
// waterfall loop), which made the issuing thread, not the tensor pipe, the bottleneck.
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n .reg .pred p;\n elect.sync _|p, 0xffffffff;\n selp.u32 %0, 1, 0, p;\n}" : "=r"(pred));
    return pred != 0;
}
// low / high words of the MN-major SWIZZLE_128B descriptor (see make_smem_desc_mn_sw128): the high word is a
// constant, the low word moves by (bytes >> 4) along the contraction
__device__ __forceinline__ uint32_t desc_lo(uint32_t smem_addr, uint32_t lbo_bytes)
{
    return ((smem_addr & 0x3FFFFu) >> 4) | (((lbo_bytes >> 4) & 0x3FFFu) << 16);
}
__host__ __device__ constexpr uint32_t desc_hi(uint32_t sbo_bytes) { return ((sbo_bytes >> 4) & 0x3FFFu) | (1u << 14) | (2u << 29); }

// kind: 0 = f16, 1 = i8; pair: cta_group::2
template <bool kInt8, bool kPair>
__device__ __forceinline__ void mma_ss_lohi(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t hi, uint32_t idesc,
                                            uint32_t accumulate)
{
    if (kPair) {
        if (kInt8)
            asm volatile("{\n .reg .pred p;\n .reg .b64 da, db;\n setp.ne.b32 p, %5, 0;\n mov.b64 da, {%1, %3};\n mov.b64 db, {%2, %3};\n"
                         " tcgen05.mma.cta_group::2.kind::i8 [%0], da, db, %4, p;\n}" ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(hi),
                         "r"(idesc), "r"(accumulate) : "memory");
        else
            asm volatile("{\n .reg .pred p;\n .reg .b64 da, db;\n setp.ne.b32 p, %5, 0;\n mov.b64 da, {%1, %3};\n mov.b64 db, {%2, %3};\n"
                         " tcgen05.mma.cta_group::2.kind::f16 [%0], da, db, %4, p;\n}" ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(hi),
                         "r"(idesc), "r"(accumulate) : "memory");
    } else {
        if (kInt8)
            asm volatile("{\n .reg .pred p;\n .reg .b64 da, db;\n setp.ne.b32 p, %5, 0;\n mov.b64 da, {%1, %3};\n mov.b64 db, {%2, %3};\n"
                         " tcgen05.mma.cta_group::1.kind::i8 [%0], da, db, %4, p;\n}" ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(hi),
                         "r"(idesc), "r"(accumulate) : "memory");
        else
            asm volatile("{\n .reg .pred p;\n .reg .b64 da, db;\n setp.ne.b32 p, %5, 0;\n mov.b64 da, {%1, %3};\n mov.b64 db, {%2, %3};\n"
                         " tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n}" ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(hi),
                         "r"(idesc), "r"(accumulate) : "memory");
    }
}

// All the MMAs of one pipeline block (`rows` contraction rows staged at a_src / b_src), issued by the elected lane.
// KINST rows per instruction = KINST/8 swizzle atoms of 1024 B further along the contraction.
template <bool kInt8, bool kPair, int BK, int KINST>
__device__ __forceinline__ void mma_block_issue(uint32_t a_src, uint32_t b_src, uint32_t chunk_bytes, uint32_t d_tmem,
                                                uint32_t idesc, int rows, uint32_t accumulate)
{
    constexpr uint32_t STEP = (KINST / 8) * 1024u / 16u;
    constexpr uint32_t HI = desc_hi(1024);
    const uint32_t a_lo = desc_lo(a_src, chunk_bytes), b_lo = desc_lo(b_src, chunk_bytes);
    if (rows == BK) {
#pragma unroll
        for (int ks = 0; ks < BK / KINST; ++ks)
            mma_ss_lohi<kInt8, kPair>(d_tmem, a_lo + ks * STEP, b_lo + ks * STEP, HI, idesc, ks == 0 ? accumulate : 1u);
    } else {
        const int ksteps = (rows + KINST - 1) / KINST;     // rows past the end are TMA zero fill
        for (int ks = 0; ks < ksteps; ++ks)
            mma_ss_lohi<kInt8, kPair>(d_tmem, a_lo + ks * STEP, b_lo + ks * STEP, HI, idesc, ks == 0 ? accumulate : 1u);
    }
}

// ---------------------------------------------------------------- descriptors
// Shared-memory matrix descriptor for an MN-major operand stored as TMA writes it with SWIZZLE_128B:
//   rows of 128 bytes (one K index each, 128 B = 64 fp16 / 128 int8 consecutive MN elements),
//   8 rows = one 1024-byte swizzle atom, atoms of one MN-chunk stacked along K (SBO = 1024 B),
//   next MN-chunk LBO bytes away.
// bits [0,14) start>>4 | [16,30) LBO>>4 | [32,46) SBO>>4 | [46,48) version=1 | [61,64) layout: 2 = SWIZZLE_128B
// (built as two 32-bit words by desc_lo / desc_hi above)

// Instruction descriptor (32 bit): [4,6) D format (1 = F32, 2 = S32) | [7,10) A format | [10,13) B format
// (kind::f16: 0 = F16; kind::i8: 1 = signed int8) | bit 15 A major (1 = MN) | bit 16 B major (1 = MN) |
// [17,23) N>>3 | [24,29) M>>4
__host__ __device__ constexpr uint32_t make_idesc(uint32_t d_fmt, uint32_t ab_fmt, uint32_t M, uint32_t N)
{
    return (d_fmt << 4) | (ab_fmt << 7) | (ab_fmt << 10) | (1u << 15) | (1u << 16) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

}  // namespace ptx
}  // namespace mwax
