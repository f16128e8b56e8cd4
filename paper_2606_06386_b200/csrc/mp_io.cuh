// Batch I/O of a block: rows of u, v, q, r between HBM and shared memory (SURVEY 8(a) a1 / a12; PAPER.md:184, :202,
// Listing 1.1 PAPER.md:206-259 stages rows through shared memory with coalesced per-thread copies).
//
// On sm_100a a row is ONE 1-D bulk asynchronous copy (`cp.async.bulk`, the TMA unit's linear form): an elected thread
// posts the expected byte count on an mbarrier and issues the copies, the copy engine moves the row without a register
// or an issue slot of the block, and every thread waits on the barrier's phase.  Stores go the other way as a bulk
// group.  Rows are 16-byte aligned and a multiple of 16 bytes long (include/mpdiv.h), which is all a bulk copy asks.
// The per-thread forms (load_number / store_number) remain for the unaligned and partial cases (a one-limb divisor
// re-bases its operands by a limb; special cases store a prefix).
#pragma once
#include "mp_block.cuh"
#include "mp_mma.cuh"

namespace mpd {

// dst[0..n) = src[0..n) with 128-bit coalesced loads (n multiple of 4), dst[n..pad) = 0.
template <int T>
__device__ __forceinline__ void load_number(limb *dst, const limb *__restrict__ src, int n, int pad)
{
    const uint4 *s4 = reinterpret_cast<const uint4 *>(src);
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    for (int i = threadIdx.x; i < n / 4; i += T) d4[i] = __ldg(s4 + i);
    for (int i = n + (int)threadIdx.x; i < pad; i += T) dst[i] = 0u;
}

// dst[0..n) = (i < valid) ? src[i] : 0, 128-bit coalesced stores; valid multiple of 4 not required.
template <int T>
__device__ __forceinline__ void store_number(limb *__restrict__ dst, const limb *src, int n, int valid)
{
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    for (int i = threadIdx.x; i < n / 4; i += T) {
        const int b = 4 * i;
        uint4 x;
        x.x = (b + 0 < valid) ? src[b + 0] : 0u;
        x.y = (b + 1 < valid) ? src[b + 1] : 0u;
        x.z = (b + 2 < valid) ? src[b + 2] : 0u;
        x.w = (b + 3 < valid) ? src[b + 3] : 0u;
        d4[i] = x;
    }
}

// The block's I/O barrier: one mbarrier word pair in BlkScratch, the number of phases completed kept in a register.
struct IoBar {
    uint32_t bar;      // shared address of the mbarrier
    uint32_t phase;    // phases completed so far (block-uniform)
};

// All threads call it once per kernel, before the first load; ends with a block barrier.
template <int T>
__device__ __forceinline__ void io_init(IoBar &io, BlkScratch *sc)
{
    io.bar = smem_u32(&sc->io_bar);
    io.phase = 0;
    if (threadIdx.x == 0) {
        mbar_init(io.bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    grp_sync<T>();
}

__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// global -> shared, completion counted in bytes on the mbarrier (a CTA-local shared address is a valid shared::cluster
// address of the executing CTA), with an L2 eviction priority for the row: a row that is fetched again later in the
// kernel (u, whose shared-memory words serve Refine as an iterate buffer in between) is kept in L2, a row read for the
// last time is not
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst_smem, const void *src, uint32_t bytes, uint32_t bar, bool keep)
{
    uint64_t pol;
    if (keep) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    else asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
// shared -> global, tracked by the issuing thread's bulk groups
__device__ __forceinline__ void bulk_s2g(void *dst, uint32_t src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// Up to two rows HBM -> shared memory by bulk copy: d_i[0..n_i) = s_i[0..n_i), d_i[n_i..pad_i) = 0 (n_i a multiple of 4,
// n_1 = 0 for a single row).  The destinations must not be in use by any thread (the caller's last block barrier is
// behind every earlier access); on return both rows and their padding are visible to the whole block.
// keep1: row 1 will be fetched again by this block (L2 evict_last); every other row is read for the last time.
template <int T>
__device__ __forceinline__ void load_rows(IoBar &io, limb *d0, const limb *__restrict__ s0, int n0, int pad0,
                                          limb *d1, const limb *__restrict__ s1, int n1, int pad1, bool keep1 = false)
{
    if (threadIdx.x == 0) {
        fence_async_smem();                                  // earlier generic-proxy accesses of the destinations
        mbar_expect_tx(io.bar, 4u * (uint32_t)(n0 + n1));
        bulk_g2s_hint(smem_u32(d0), s0, 4u * (uint32_t)n0, io.bar, false);
        if (n1 > 0) bulk_g2s_hint(smem_u32(d1), s1, 4u * (uint32_t)n1, io.bar, keep1);
    }
    for (int i = n0 + (int)threadIdx.x; i < pad0; i += T) d0[i] = 0u;
    for (int i = n1 + (int)threadIdx.x; i < pad1; i += T) d1[i] = 0u;
    if (!mbar_wait(io.bar, io.phase & 1u)) raise_status(ST_IO_WAIT);
    io.phase++;
    grp_sync<T>();
}

// One row shared memory -> HBM: dst[0..bulk) = src[0..bulk) by bulk copy, dst[bulk..n) = 0 by vector stores
// (bulk, n multiples of 4; src visible to the block, i.e. a block barrier lies behind its last write).  The caller's
// next block barrier orders the reuse of src behind the copy (the issuing thread waits for its bulk group).
template <int T>
__device__ __forceinline__ void store_row(limb *__restrict__ dst, const limb *src, int n, int bulk)
{
    if (threadIdx.x == 0 && bulk > 0) {
        fence_async_smem();
        bulk_s2g(dst, smem_u32(src), 4u * (uint32_t)bulk);
    }
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    for (int i = bulk / 4 + (int)threadIdx.x; i < n / 4; i += T) d4[i] = make_uint4(0u, 0u, 0u, 0u);
    if (threadIdx.x == 0 && bulk > 0) bulk_commit_wait();
}

}  // namespace mpd
