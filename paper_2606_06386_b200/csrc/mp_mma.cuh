// Tensor-core multiplier for the large products: a big-integer product as an int8 tcgen05 GEMM (sm_100a).
//
// The product of two numbers is the convolution of their BYTE strings, c[t] = sum_x a[x] * b[t - x],
// followed by carry propagation.  Write t = 128 d + i (i < 128) and cut b into 128-byte chunks e; then
//
//     c[128 d + i] = sum_p  sum_{j < 128}  a[128 p + i - j] * b[128 (d - p) + j]
//                  = sum_p  ( A_p  x  B_p )[i][d],      A_p[i][j] = a[128 p + i - j]   (128 x 128 Toeplitz tile)
//                                                        B_p[j][d] = b[128 (d - p) + j] (chunk d - p of b)
//
// i.e. one GEMM with M = 128 (byte position inside an output block), N = number of output blocks,
// K = 128 x (number of chunks of a + 1), u8 x u8 -> s32 (`tcgen05.mma.kind::i8`, accumulators in TMEM;
// a column sum is below 255^2 * 32768 < 2^31 for operands up to 8192 limbs).
//   * B_p needs no work per step: b is stored ONCE as 128-byte rows in the K-major SWIZZLE_128B layout
//     (16-byte units XOR-ed with the row number, on absolute shared-memory addresses), and a step simply
//     starts its descriptor one row further.
//   * A_p is never materialised.  A Toeplitz tile holds 255 distinct bytes; what the tensor core needs is a
//     shared-memory matrix descriptor under which those bytes LOOK like the 128 x 128 tile.  The K-major
//     no-swizzle layout reads an 8-row x 16-byte core matrix as 8 consecutive 16-byte units, the next core matrix
//     along K at +LBO and the next 8 rows at +SBO.  Take the rows in the order i = g + 16 (7 - r) (g = 8-row
//     group, r = row inside it): rows of a group differ by 16 bytes of the Toeplitz window, i.e. by exactly one
//     unit, so with LBO = 16 bytes (core matrices that OVERLAP) the whole group is one reversed string
//     C_g[y] = a[128 p + g + 112 - y], y < 240, read at unit r + c for K-chunk c; the 16 groups are the same
//     string shifted by one byte each, 16 copies SBO bytes apart.  Consecutive steps slide the window by 128
//     bytes, so a step costs 16 x 128 new bytes (one 16-byte store per producer thread) in a ring of four or six
//     128-byte segments per copy (plus a mirror of segment 0 that keeps every window contiguous) -- against
//     16 KB per step when the tile was generated row by row into tensor memory (33 LDS + 32 PRMT + a 32-register
//     tcgen05.st per thread and step: ~330 cycles per step whatever N was, the limit of round 1).
//     The MMA then reads A from shared memory (SS form): 128 rows x 32 bytes per instruction = 32 cycles of
//     shared-memory bandwidth, so an instruction takes max(32 + N/4, N/2) cycles (measured: 40.1 at N = 32)
//     and the loop is tensor-core bound from N = 128 on.  The accumulator row of byte position i is
//     lane 8 (i mod 16) + 7 - (i div 16); the epilogue undoes the permutation.
//   * Warp roles: the first two (128-thread blocks) or four warps produce the ring segments, several steps ahead;
//     the last two warps issue alternate steps into an accumulator set each (an issuer's own instruction stream --
//     barrier poll, operand words, election, four MMAs, commit -- takes ~500 cycles per step whatever N is, which
//     was the step time with one issuer).  The whole issuer warp walks its steps, the operand words are prepared in ordinary registers and one
//     lane elected by elect.sync directly around straight-line code issues the four MMAs and the commit of a step
//     (under `if (tid == X)` ptxas wraps every tcgen05 instruction in an ELECT / BRA.U.ANY loop).
//   * Epilogue: `tcgen05.ld` (lane = permuted byte position, column = block) by ALL warps (a warp reaches the
//     lane quarter warp % 4), four lanes 8 apart give one limb's 64-bit column sum, low words go to P, high
//     words to HI one limb up, and one block-wide carry-propagating add (mp_block.cuh) finishes.
// A range of output blocks dlo <= d < dhi can be asked for (clipped products); what is omitted below
// block dlo is less than B^(32 dlo + 1).  Only steps p whose chunk d - p can be non-zero are issued.
#pragma once
#include "mp_block.cuh"

namespace mpd {

#ifndef MMA_SPIN_LIMIT_LOG2
#define MMA_SPIN_LIMIT_LOG2 26
#endif
constexpr uint32_t MMA_SPIN_LIMIT = 1u << MMA_SPIN_LIMIT_LOG2;

// shared-memory scratch of the engine: rows of the row operand | ring of the Toeplitz operand | mbarriers
// The ring is recycled in pairs of segments (see the issuers): three pairs, two in 128-thread blocks (four of them
// share an SM's shared memory).
__host__ __device__ constexpr int ring_pairs(int T) { return T <= 128 ? 2 : 3; }
__host__ __device__ constexpr int ring_segs(int T) { return 2 * ring_pairs(T); }              // 128-byte segments per copy
__host__ __device__ constexpr int ring_copy_bytes(int T) { return (ring_segs(T) + 1) * 128; }   // + 1 mirror of segment 0; = SBO
__host__ __device__ constexpr int ring_bytes(int T) { return 16 * ring_copy_bytes(T); }
constexpr int MMA_ISSUERS = 2;                             // issuing warps, one accumulator set each
constexpr int MMA_BAR_BYTES = 256;                         // full[s] +8s, empty[pair] +64+8 pair, done +128, TMEM slot +160
// rows of the row operand | ring of the Toeplitz operand (the mbarriers live elsewhere: MMA_BAR_BYTES of their own)
__host__ __device__ constexpr int mma_scratch_bytes(int rows, int T) { return rows * 128 + ring_bytes(T); }

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// bounded wait: a protocol error must not hang the GPU; false = gave up
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity)
{
    for (uint32_t it = 0; it < MMA_SPIN_LIMIT; ++it) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return true;
    }
    return false;
}
// one lane of a converged warp (elect.sync): the branch it guards is uniform for ptxas, so the tcgen05
// instructions inside are issued straight from uniform registers
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// Shared-memory matrix descriptors, given by their low words; the high words are constants.
//   row operand  : K-major SWIZZLE_128B, rows of 128 bytes, 8-row groups 1024 bytes apart
//   Toeplitz     : K-major no swizzle, LBO = 16 bytes (overlapping core matrices), SBO = ring_copy_bytes(T)
constexpr uint32_t DESC_HI_ROWS = (1024u >> 4) | (1u << 14) | (2u << 29);
__host__ __device__ constexpr uint32_t desc_hi_ring(int T) { return ((uint32_t)ring_copy_bytes(T) >> 4) | (1u << 14); }
__device__ __forceinline__ uint32_t mma_desc_lo(uint32_t saddr) { return ((saddr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint32_t mma_idesc(int n_cols)      // u8 x u8 -> s32, both K-major, M = 128
{
    return (2u << 4) | ((uint32_t)(n_cols >> 3) << 17) | ((128u >> 4) << 24);
}
// D[tmem] (+)= A[smem, Toeplitz descriptor] x B[smem, row descriptor], u8 x u8 -> s32, M = 128, K = 32.
// The issuer prepares the words in ordinary registers BEFORE it elects its lane, so that the elected path is
// R2UR + tcgen05.mma only (arithmetic on the uniform datapath sits on the issue path).
template <int T>
__device__ __forceinline__ void tc_mma_i8_ss(uint32_t tmem_d, uint32_t adesc_lo, uint32_t bdesc_lo, uint32_t idesc,
                                             uint32_t accumulate)
{
    constexpr uint32_t DESC_HI_RING = desc_hi_ring(T);
    const uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b64 ad, bd;\n\tsetp.ne.b32 p, %4, 0;\n\tmov.b64 ad, {%1, %6};\n\tmov.b64 bd, {%2, %7};\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], ad, bd, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "r"(adesc_lo), "r"(bdesc_lo), "r"(idesc), "r"(accumulate), "r"(z), "r"(DESC_HI_RING),
                   "r"(DESC_HI_ROWS) : "memory");
}
// same with A in tensor memory (128 lanes x 8 columns): the pure rate of the pipe, used by the roofline probe
__device__ __forceinline__ void tc_mma_i8_ts(uint32_t tmem_d, uint32_t tmem_a, uint32_t bdesc_lo, uint32_t idesc,
                                             uint32_t accumulate)
{
    const uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b64 bd;\n\tsetp.ne.b32 p, %4, 0;\n\tmov.b64 bd, {%2, %6};\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], bd, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "r"(tmem_a), "r"(bdesc_lo), "r"(idesc), "r"(accumulate), "r"(z), "r"(DESC_HI_ROWS) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                 "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Per-block state of the tensor-core multiplier (block-uniform values, kept in registers).
struct MmaCtx {
    uint32_t tmem_base;   // first allocated TMEM column
    int tmem_cols;        // allocated columns (power of two >= 32) = accumulator columns: output blocks per call
    uint8_t *brows;       // the row operand in swizzled 128-byte rows, 1024-byte aligned
    int brows_cap;        // rows available at brows
    uint8_t *ring;        // 16 copies x (RING_SEGS + 1) segments of the reversed Toeplitz operand
    uint32_t bar;         // shared address of the mbarriers
    uint32_t full_par, empty_par;   // bit s = parity of the phases completed so far on full[s] / empty[pair slot s]
    uint32_t ndone;       // products finished so far (parity of the done barrier)
    uint32_t fail;        // set when a bounded wait gave up: the engine is retired for this block
};

__device__ unsigned int g_mma_fail;   // bounded waits that gave up (expected 0); reported with the debug counters

// Warp roles: the last MMA_ISSUERS warps issue and do nothing else (their instruction streams are the critical path
// of the loop: ~500 cycles per step for one warp, whatever N is); the first PRODUCERS warps write the ring segments.
template <int T>
struct MmaRoles {
    static constexpr int WARPS = T / 32;
    static constexpr int FIRST_ISSUER = WARPS - MMA_ISSUERS;
    static constexpr int PRODUCERS = WARPS == 4 ? 2 : 4;
    static constexpr int RING_PAIRS = ring_pairs(T), RING_SEGS = ring_segs(T), RING_COPY_BYTES = ring_copy_bytes(T);
    static_assert(WARPS >= 4 && RING_SEGS <= 8 && RING_PAIRS <= 4 && MMA_ISSUERS == 2, "128 threads or more, two issuers");
};

// One-time setup per block: mbarriers, TMEM allocation (warp 0 owns it).  All threads call it.
// scratch: mma_scratch_bytes(rows, T) bytes, 1024-byte aligned (rewritten by every product: it may overlap buffers
// that are dead while a product runs); bars: MMA_BAR_BYTES that nothing else ever touches.
template <int T>
__device__ __forceinline__ void mma_init(MmaCtx &cx, uint8_t *scratch, int rows, uint8_t *bars, int tmem_cols)
{
    cx.brows = scratch;
    cx.brows_cap = rows;
    cx.ring = scratch + rows * 128;
    cx.bar = smem_u32(bars);
    cx.tmem_cols = tmem_cols;
    cx.ndone = 0;
    cx.fail = 0;
    cx.full_par = 0;
    cx.empty_par = 0;
    uint32_t *slot = reinterpret_cast<uint32_t *>(bars + 160);
    if (threadIdx.x == 0) {
        for (int s = 0; s < ring_segs(T); s++) mbar_init(cx.bar + 8 * s, 1);                 // the segment's producer warp
        for (int s = 0; s < ring_pairs(T); s++) mbar_init(cx.bar + 64 + 8 * s, 2);           // the commits of the pair's two steps
        mbar_init(cx.bar + 128, MMA_ISSUERS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (threadIdx.x < 32) {
        __syncwarp();                                // thread 0 rejoins its warp before the aligned instructions
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    cx.tmem_base = *slot;
}

// A kernel that CONTAINS tcgen05.alloc holds the SM's allocation permit from launch until it relinquishes it,
// and no other block is co-scheduled on the SM meanwhile: a block that will not allocate must say so at
// once (measured: without this, blocks that skipped mma_init ran one per SM instead of four).
__device__ __forceinline__ void mma_decline()
{
    if (threadIdx.x < 32) asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
}

template <int T>
__device__ __forceinline__ void mma_fini(MmaCtx &cx)
{
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(cx.tmem_base), "r"(cx.tmem_cols));
}

// Four 16-byte units of reversed strings that start one word apart: unit j (j < 4), byte e (e < 16) = a[x + 4 j - e],
// a = the bytes of the limbs W (nw words, zero outside).  Word m of unit j holds a[x + 4j - 4m - k], k = 0..3 from the
// low byte up: one PRMT from two neighbouring words of a; the four units share 8 words.  (The four units a producer
// lane writes per segment belong to copies g, g + 4, g + 8, g + 12: same unit, byte shifts 4 apart.)
__device__ __forceinline__ void reversed16x4(const limb *W, int nw, int x, uint4 (&o)[4])
{
    const int z0 = x - 3;                                    // lowest byte of word 0 of unit 0
    const int s = z0 & 3;
    const uint32_t sel = (uint32_t)(s + 3) | ((uint32_t)(s + 2) << 4) | ((uint32_t)(s + 1) << 8) | ((uint32_t)s << 12);
    const int wi = z0 >> 2;                                  // floor(z0 / 4), also for negative z0
    uint32_t w[9];                                           // w[i] = word wi + 4 - i, i.e. words wi + 4 down to wi - 4
    if (wi - 4 >= 0 && wi + 4 < nw) {
#pragma unroll
        for (int i = 0; i < 9; ++i) w[i] = W[wi + 4 - i];
    } else {
#pragma unroll
        for (int i = 0; i < 9; ++i) { const int k = wi + 4 - i; w[i] = (k >= 0 && k < nw) ? W[k] : 0u; }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {                            // unit j, word m = PRMT(lo = word wi + j - m, hi = word wi + j + 1 - m)
        o[j].x = __byte_perm(w[4 - j], w[3 - j], sel);
        o[j].y = __byte_perm(w[5 - j], w[4 - j], sel);
        o[j].z = __byte_perm(w[6 - j], w[5 - j], sel);
        o[j].w = __byte_perm(w[7 - j], w[6 - j], sel);
    }
}

// Steps (Toeplitz windows) a range product needs when `na` is the Toeplitz operand.
__device__ __forceinline__ int mma_steps(int na, int nb, int dlo, int dhi)
{
    const int Ea = (na + 31) / 32, Eb = (nb + 31) / 32;
    return min(Ea, dhi - 1) - max(0, dlo - Eb + 1) + 1;
}

// Should this range product run on the tensor core?  Cost model in cycles of the SM: a step costs
// 4 x max(32 + N/4, N/2) cycles (shared-memory read of the Toeplitz tile, then the tensor core) and at least the
// issuing warp's ~40 cycles per instruction; a call costs the row operand, the epilogue and the final add; against
// about 1/26 cycle per limb product on the IMAD path, of which a block of T threads gets T/512.  MMA_PLAN_PCT
// scales the tensor side to what is measured.  swap = take b as the Toeplitz operand (fewer steps).  Block-uniform.
#ifndef MMA_PLAN_PCT
#define MMA_PLAN_PCT 100
#endif
// What a caller needs to decide about the engine, by value: the context lives in memory (mma_mul_range is not inlined and
// takes it by reference), and three dependent loads from it before every product were 3 % of a config-2 division.
struct MmaRef {
    MmaCtx *cx;      // nullptr: no engine for this instance
    int cols;        // allocated TMEM columns
    int cap;         // rows available for the row operand
};

template <int T>
__device__ __forceinline__ bool mma_plan(const MmaRef &m, int na, int nb, int dlo, int dhi, bool &swap)
{
    if (m.cx == nullptr || na <= 0 || nb <= 0 || dlo < 0) return false;
    dhi = min(dhi, (na + nb + 31) / 32);
    const int N = dhi - dlo, Nn = (N + 15) & ~15;
    if (N <= 0) return false;
    const int sa = mma_steps(na, nb, dlo, dhi), sb = mma_steps(nb, na, dlo, dhi);
    swap = sb < sa;
    const int steps = swap ? sb : sa;
    if (steps <= 0 || Nn > m.cols || Nn + steps - 1 > m.cap) return false;
    const long long est = (long long)(32 * N) * (long long)min(na, nb);      // limb products, upper bound
    const long long step_cycles = 4ll * max(max(32 + Nn / 4, Nn / 2), 40);
    const long long call_cycles = 2500ll + 20ll * Nn * (512 / T) + 6ll * (Nn + steps);
    // the blocks of an SM run in lock step and enter their MMA loops together: the unit is shared by 512 / T of them,
    // just as the IMAD pipe is (config 2: a 33-step band product took 21 000 cycles on the shared unit, ~11 000 on IMAD)
    const long long mma_cycles = steps * step_cycles * (512 / T) + call_cycles;
    const long long imad_cycles = est * 512ll / (26ll * T);
    if (100ll * imad_cycles < (long long)MMA_PLAN_PCT * mma_cycles) return false;
    return m.cx->fail == 0;                                      // a context whose pipeline gave up once is retired
}

// P[i] = limb 32*dlo + i of ((A * B) - E) mod B^(32 dhi), 0 <= E < B^(32 dlo + 1); i < 32 (dhi - dlo).
// A (na limbs) is the Toeplitz operand, B (nb limbs) the row operand; both plain little-endian limbs in
// shared memory, read as zero beyond na / nb.  HI is scratch of the same size as P (+8).  dhi is clamped
// to the size of the full product.  All T threads call it; ends with the result visible to the block.
// Returns the number of limbs stored, -1 when the request does not fit (TMEM columns or row buffer), -2 when a
// bounded pipeline wait gave up (status bit set, engine retired; P holds nothing: redo the product elsewhere).
template <int T>
__device__ __noinline__ int mma_mul_range(MmaCtx &cx_mem, const limb *A, int na, const limb *B, int nb, int dlo, int dhi,
                                          limb *P, limb *HI, Blk &blk)
{
    using Roles = MmaRoles<T>;
    constexpr int RING_PAIRS = Roles::RING_PAIRS, RING_SEGS = Roles::RING_SEGS, RING_COPY_BYTES = Roles::RING_COPY_BYTES;
    MmaCtx cx = cx_mem;        // work on a register copy: the asm memory clobbers would reload every field
    const int tid = threadIdx.x, warp = tid >> 5;
    const int Ea = (na + 31) / 32, Eb = (nb + 31) / 32;
    dhi = min(dhi, (na + nb + 31) / 32);
    const int N = dhi - dlo;
    const int Nn = (N + 15) & ~15;
    const int pmin = max(0, dlo - Eb + 1), pmax = min(Ea, dhi - 1);
    const int e0 = dlo - pmax;                                // chunk of b held by row 0
    const int nsteps = pmax - pmin + 1;
    const int R = Nn + nsteps - 1;                            // rows: chunks e0 .. dlo + Nn - 1 - pmin
    if (N <= 0 || pmax < pmin || Nn > cx.tmem_cols || R > cx.brows_cap) return -1;

    // ---- the row operand: chunk e of b -> row e - e0, 16-byte units swizzled by the row number ----
    for (int q = tid; q < R * 8; q += T) {
        const int r = q >> 3, c = q & 7;
        const int w0 = (r + e0) * 32 + c * 4;
        uint4 val;
        val.x = (w0 + 0 >= 0 && w0 + 0 < nb) ? B[w0 + 0] : 0u;
        val.y = (w0 + 1 >= 0 && w0 + 1 < nb) ? B[w0 + 1] : 0u;
        val.z = (w0 + 2 >= 0 && w0 + 2 < nb) ? B[w0 + 2] : 0u;
        val.w = (w0 + 3 >= 0 && w0 + 3 < nb) ? B[w0 + 3] : 0u;
        *reinterpret_cast<uint4 *>(cx.brows + r * 128 + ((c ^ (r & 7)) << 4)) = val;
    }
    fence_async_smem();
    __syncthreads();

    // Steps run from p = pmax down to pmin (step t <-> p = pmax - t): the reversed string of copy g is
    // S_g[z] = a[128 pmax + 112 + g - z], step t reads z in [128 t, 128 t + 240) = segments t and t + 1, and the
    // row-operand descriptor starts one row further every step.
    const uint32_t ring_u32 = smem_u32(cx.ring);
    const uint32_t b_lo0 = mma_desc_lo(smem_u32(cx.brows));
    // Two issuers: issuer i takes the steps t = i, i + 2, .. and accumulates them in its own set of Nn columns (the sets
    // are added in the epilogue); when two sets do not fit the allocated columns issuer 0 takes every step.  The ring
    // is recycled in PAIRS of segments: step t reads segments t and t + 1, so pair P = (2P, 2P + 1) is free once the
    // steps 2P and 2P + 1 are done (each issuer's earlier steps finish before its later ones): every step commits
    // once, to empty[pair t / 2], a barrier of two arrivals.
    const int ni = (2 * Nn <= cx.tmem_cols && nsteps >= 2) ? 2 : 1;
    const int last_pair = nsteps / 2;                         // pair of segment nsteps, the last one produced
    if (warp < Roles::PRODUCERS) {
        // ---- producers: warp w writes the segments sg = w, w + PRODUCERS, .. on its own (the latency of a segment
        // -- barrier poll, dependent loads, store, proxy fence, arrive -- is a few hundred cycles, so the warps work on
        // different segments); lane l writes unit u = l % 8 of the copies g = l / 8 + 4 j, j < 4 ----
        const int lane = tid & 31;
        const int u = lane & 7, g0 = lane >> 3;
        uint8_t *dst0 = cx.ring + g0 * RING_COPY_BYTES + 16 * u;
        for (int sg = warp; sg <= nsteps; sg += Roles::PRODUCERS) {
            const int s = sg % RING_SEGS, pr = sg >> 1, ps = pr % RING_PAIRS;
            // the pair's slot was last used by pair pr - RING_PAIRS: phase number pr / RING_PAIRS - 1 of empty[ps] in
            // this product
            if (pr >= RING_PAIRS &&
                !mbar_wait(cx.bar + 64 + 8 * ps, ((cx.empty_par >> ps) + (uint32_t)(pr / RING_PAIRS) - 1u) & 1)) { cx.fail = 1; break; }
            uint4 val[4];
            reversed16x4(A, na, 128 * (pmax - sg) + 112 + g0 - 16 * u, val);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint8_t *dst = dst0 + 4 * j * RING_COPY_BYTES + 128 * s;
                *reinterpret_cast<uint4 *>(dst) = val[j];
                if (s == 0) *reinterpret_cast<uint4 *>(dst + 128 * RING_SEGS) = val[j];   // the mirror keeps windows contiguous
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(cx.bar + 8 * s);
        }
    } else if (warp >= Roles::FIRST_ISSUER) {
        // ---- the issuers: a whole warp walks its steps; a step is one poll per segment it has not seen yet, the
        // operand words advanced incrementally in ordinary registers, one lane elected directly around straight-line
        // tcgen05 code (four MMAs and the commit).  The tcgen05 fence is needed once per product (the accumulators
        // were last read by the epilogue of the previous one); the ring data comes through the generic proxy and
        // fence.proxy.async. ----
        const int me = warp - Roles::FIRST_ISSUER;
        const int stride = ni;                                               // steps me, me + ni, ..
        tc_fence_after();
        bool ok = true;
        if (me < ni) {
            const uint32_t a_lo0 = mma_desc_lo(ring_u32);
            const uint32_t d_base = cx.tmem_base + (uint32_t)(me * Nn);
            uint32_t acc0 = 0u;
            for (int t = me; ok && t < nsteps; t += stride) {
                const int s0 = t % RING_SEGS, s1 = (t + 1) % RING_SEGS;
                // segments t and t + 1 (with one issuer segment t was already awaited a step earlier)
                if (ni == 2 || t == 0) ok = mbar_wait(cx.bar + 8 * s0, ((cx.full_par >> s0) + (uint32_t)(t / RING_SEGS)) & 1);
                ok = ok && mbar_wait(cx.bar + 8 * s1, ((cx.full_par >> s1) + (uint32_t)((t + 1) / RING_SEGS)) & 1);
                if (!ok) break;
                uint32_t a_lo = a_lo0 + 8u * (uint32_t)s0, b_lo = b_lo0 + 8u * (uint32_t)t;
                uint32_t ebar = cx.bar + 64 + 8 * ((t >> 1) % RING_PAIRS);
                if (Nn <= 256) {
                    uint32_t d_tmem = d_base, idesc = mma_idesc(Nn), ac = acc0;
                    asm volatile("" : "+r"(d_tmem), "+r"(a_lo), "+r"(b_lo), "+r"(idesc), "+r"(ac), "+r"(ebar));
                    if (elect_one()) {
                        tc_mma_i8_ss<T>(d_tmem, a_lo, b_lo, idesc, ac);
                        tc_mma_i8_ss<T>(d_tmem, a_lo + 2, b_lo + 2, idesc, 1u);
                        tc_mma_i8_ss<T>(d_tmem, a_lo + 4, b_lo + 4, idesc, 1u);
                        tc_mma_i8_ss<T>(d_tmem, a_lo + 6, b_lo + 6, idesc, 1u);
                        tc_commit(ebar);
                    }
                } else {
                    // more than 256 output blocks: the accumulator columns in chunks of 256 (the election sits directly
                    // around straight-line tcgen05 code: a loop inside it brings ptxas' ELECT loops back)
                    for (int nc = 0; nc < Nn; nc += 256) {
                        uint32_t d_tmem = d_base + (uint32_t)nc, idesc = mma_idesc(min(256, Nn - nc));
                        uint32_t bl = b_lo + 8u * (uint32_t)nc, al = a_lo, ac = acc0;
                        asm volatile("" : "+r"(d_tmem), "+r"(al), "+r"(bl), "+r"(idesc), "+r"(ac));
                        if (elect_one()) {
                            tc_mma_i8_ss<T>(d_tmem, al, bl, idesc, ac);
                            tc_mma_i8_ss<T>(d_tmem, al + 2, bl + 2, idesc, 1u);
                            tc_mma_i8_ss<T>(d_tmem, al + 4, bl + 4, idesc, 1u);
                            tc_mma_i8_ss<T>(d_tmem, al + 6, bl + 6, idesc, 1u);
                        }
                    }
                    if (elect_one()) tc_commit(ebar);
                }
                acc0 = 1u;
            }
        }
        if (!ok) cx.fail = 2;
        if (elect_one()) tc_commit(cx.bar + 128);            // arrives when this warp's MMAs are done
        __syncwarp();
        // one issuer alone polls for the end of the MMAs; everybody else sleeps at the block barrier below (a dozen
        // warps polling an mbarrier take the issue slots and the shared-memory port the loop needs)
        if (me == 0) {
            if (!mbar_wait(cx.bar + 128, cx.ndone & 1)) cx.fail = 3;
            // The last pair holds segment nsteps (and segment nsteps - 1 when nsteps is odd): the steps 2 last_pair and
            // 2 last_pair + 1 that would commit to it do not all exist; plain arrivals complete its phase.  They come
            // AFTER every commit has arrived (an earlier pair of the same slot may still be in its phase before that).
            if ((tid & 31) == 0) {
                const int have = (2 * last_pair <= nsteps - 1) + (2 * last_pair + 1 <= nsteps - 1);
                for (int k = have; k < 2; ++k) mbar_arrive(cx.bar + 64 + 8 * (last_pair % RING_PAIRS));
            }
            __syncwarp();
        }
    }
    // phases completed on each barrier when this product is over: segments sg = s, s + RING_SEGS, .. <= nsteps on
    // full[s], pairs P = s, s + RING_PAIRS, .. <= last_pair on empty[s]; only their parities are kept
#pragma unroll
    for (int s = 0; s < RING_SEGS; s++)
        if (s <= nsteps) cx.full_par ^= ((uint32_t)((nsteps - s) / RING_SEGS + 1) & 1u) << s;
#pragma unroll
    for (int s = 0; s < RING_PAIRS; s++)
        if (s <= last_pair) cx.empty_par ^= ((uint32_t)((last_pair - s) / RING_PAIRS + 1) & 1u) << s;
    __syncwarp();

    // ---- epilogue: TMEM lane 8 (i mod 16) + 7 - (i div 16), column d  ->  byte-column sum of output byte
    // 128 (dlo + d) + i.  A warp reaches lane quarter warp % 4; the warps of a quarter share the columns. ----
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    {
        // The four byte-column sums of a limb sit in lanes 8 apart of one lane quarter, i.e. of one warp.  They are
        // brought together through the warp's own 2 KB of the engine's scratch (dead once the MMAs are done) instead of
        // by shuffles: lane (b, j) stores the 16 columns it holds at [column][j][b], conflict free, and reads back the
        // four words of (column, limb) pairs as one 16-byte load -- 64 shuffles per 16 columns made the epilogue
        // shuffle-bound (a third of an SM's shuffle rate with four resident blocks).
        const int lane = tid & 31, quarter = warp & 3;
        const int groups = min(T / 128, mma_scratch_bytes(cx.brows_cap, T) / 8192);     // 4 warps x 2 KB each
        uint32_t *S = reinterpret_cast<uint32_t *>(cx.brows) + 512 * warp;
        if ((warp >> 2) < groups) {
            for (int d0 = 16 * (warp >> 2); d0 < Nn; d0 += 16 * groups) {
                uint32_t v[16];
                tmem_ld16(cx.tmem_base + ((uint32_t)(32 * quarter) << 16) + d0, v);
                if (ni == 2) {                                            // the second issuer's accumulator set
                    uint32_t v2[16];
                    tmem_ld16(cx.tmem_base + ((uint32_t)(32 * quarter) << 16) + (uint32_t)(Nn + d0), v2);
#pragma unroll
                    for (int k = 0; k < 16; ++k) v[k] += v2[k];
                }
                uint32_t *Sw = S + (lane & 7) * 4 + (lane >> 3);          // [k][j = lane % 8][b = lane / 8]
#pragma unroll
                for (int k = 0; k < 16; ++k) Sw[32 * k] = v[k];
                __syncwarp();
#pragma unroll
                for (int s4 = 0; s4 < 4; ++s4) {
                    const int k = (lane >> 3) + 4 * s4, jj = lane & 7;    // item lane + 32 s4: words [k][jj][0..3]
                    const uint4 w = *reinterpret_cast<const uint4 *>(S + 4 * lane + 128 * s4);
                    const unsigned long long sv = (unsigned long long)w.x + ((unsigned long long)w.y << 8) +
                                                  ((unsigned long long)w.z << 16) + ((unsigned long long)w.w << 24);
                    if (d0 + k < N) {
                        const int L = 32 * (d0 + k) + quarter + 4 * (7 - jj);   // (i div 4) for i = g + 16 (7 - r)
                        P[L] = (uint32_t)sv;
                        HI[L + 1] = (uint32_t)(sv >> 32);
                    }
                }
                __syncwarp();
            }
        }
        if (tid == 0) HI[0] = 0u;
        tc_fence_before();
    }
    cx.ndone += 1;
    if (cx.fail) atomicOr(&g_mma_fail, 1u << (cx.fail - 1));
    if (__syncthreads_or(cx.fail != 0)) {
        // a bounded wait gave up somewhere in the block: the accumulators cannot be trusted and the barrier
        // phases are out of step.  Say so (sticky status bit), retire the engine for the rest of this block
        // (mma_plan refuses a failed context) and let the caller redo this product on the IMAD path.
        raise_status(ST_MMA_WAIT);
        cx_mem.fail = 1;
        return -2;
    }
    // ---- P += HI with block-wide carry propagation (the carry out of the top block is dropped: mod B^(32 dhi)) ----
    lin_addsub<T, false>(P, 32 * N, LimbView{P, 32 * N, 0}, LimbView{HI, 32 * N, 0}, 0u, blk);
    cx_mem.full_par = cx.full_par;
    cx_mem.empty_par = cx.empty_par;
    cx_mem.ndone = cx.ndone;
    count(CNT_MMA_COLSTEPS, (unsigned long long)nsteps * (unsigned long long)Nn);   // x 16384 = u8 MACs executed
    {   // cycles the tensor unit is occupied by this product's instructions: 4 per step and 256-column chunk, each
        // max(32 + n/4, n/2) -- the Toeplitz tile comes from shared memory (128 rows x 32 bytes = 32 cycles), see the header
        unsigned long long cyc = 0;
        for (int nc = 0; nc < Nn; nc += 256) {
            const int n = min(256, Nn - nc);
            cyc += 4ull * (unsigned long long)max(32 + n / 4, n / 2);
        }
        count(CNT_MMA_UNIT_CYCLES, cyc * (unsigned long long)nsteps);
    }
    return 32 * N;
}

}  // namespace mpd
