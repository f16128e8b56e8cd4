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
//     (16-byte units XOR-ed with the row number, on absolute shared-memory addresses), and step p simply
//     starts its descriptor p rows lower.
//   * A_p is generated on the fly by the CUDA cores: row i is the byte-reversed 128-byte window of a
//     ending at byte 128 p + i -- one PRMT per word from two neighbouring words.  The row goes straight
//     from registers into TENSOR MEMORY (`tcgen05.st`, lane = row, 32 columns = 128 bytes of K) and the
//     MMA takes its A operand from there (`tcgen05.mma [d], [a_tmem], b_desc`): the tile never touches
//     shared memory, whose bandwidth was the limit of a first version that staged A tiles in a 16 KB ring
//     (about 840 cycles per step).  Stages of 32 TMEM columns are handed to the MMA-issuing warp through
//     mbarriers and freed by `tcgen05.commit`.
//   * The issuing warp's own instruction stream is the critical path of the loop.  One `tcgen05.mma` (M = 128,
//     K = 32, u8) occupies the tensor core for max(~48, N / 2) cycles (measured: two warps issuing to disjoint
//     accumulators reach N / 2 per instruction together; one lean warp 48 cycles at N <= 64, 64 at N = 128),
//     but a first version issued from `if (tid == ISSUER)`, where ptxas wraps every tcgen05 instruction in an
//     ELECT / BRA.U.ANY loop and builds each descriptor on the uniform datapath after the R2UR: 170 cycles per
//     instruction whatever N was (690 per step).  Now the whole issuer warp walks the steps, the operand words
//     are prepared in ordinary registers and one elected lane issues the four MMAs and the commit of a step:
//     ~330 cycles per step at N = 128 (tensor-core time 256), ~500 at N = 256 (tensor-core time 512).
//   * Epilogue: `tcgen05.ld` (lane = i, column = d), four adjacent lanes form one limb's 64-bit column
//     sum, low words go to P, high words to HI one limb up, and one block-wide carry-propagating add
//     (mp_block.cuh) finishes.
// A range of output blocks dlo <= d < dhi can be asked for (clipped products); what is omitted below
// block dlo is less than B^(32 dlo + 1).  Only steps p whose chunk d - p can be non-zero are issued.
//
// Measured on B200 (mpmul_batch_ex, whole batches): 592 full 4096 x 4096-limb products in 0.245 ms = 4.1e13
// limb products/s against 9.15e12 for the IMAD.WIDE roofline probe; 1184 x (2048 x 2048) in 0.226 ms.
#pragma once
#include "mp_block.cuh"

namespace mpd {

constexpr int MMA_STAGE_COLS = 32;    // one Toeplitz tile = 128 lanes x 32 columns of tensor memory
#ifndef MMA_SPIN_LIMIT_LOG2
#define MMA_SPIN_LIMIT_LOG2 26
#endif
constexpr uint32_t MMA_SPIN_LIMIT = 1u << MMA_SPIN_LIMIT_LOG2;

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
// instructions inside are issued straight from uniform registers -- under `if (tid == X)` every
// tcgen05.mma / tcgen05.commit is wrapped in an ELECT / BRA.U.ANY loop over the "possibly several" active lanes
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
// D[tmem] (+)= A[smem desc] x B[smem desc], u8 x u8 -> s32, M = 128, K = 32
__device__ __forceinline__ void tc_mma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate)
{
    const uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(z) : "memory");
}
// D[tmem] (+)= A[tmem] x B[smem desc]: A is 128 lanes x 8 columns (row m in lane m, 4 bytes of K per column)
__device__ __forceinline__ void tc_mma_i8_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc,
                                             uint32_t accumulate)
{
    const uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(z) : "memory");
}
// same with the shared-memory descriptor given by its low word (mma_desc_lo); the high word is the constant
// part of mma_smem_desc.  The issuer prepares the words in ordinary registers BEFORE it elects its lane, so
// that the elected path is R2UR + tcgen05.mma only (arithmetic on the uniform datapath sits on the issue path:
// a chain R2UR - UIADD3 - USHF - ULOP3 - ULOP3 in front of every instruction cost ~120 cycles per MMA against
// a tensor-core time of N / 2 cycles)
constexpr uint32_t MMA_DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
__device__ __forceinline__ uint32_t mma_desc_lo(uint32_t saddr) { return ((saddr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ void tc_mma_i8_ts_lo(uint32_t tmem_d, uint32_t tmem_a, uint32_t bdesc_lo, uint32_t idesc,
                                                uint32_t accumulate)
{
    const uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b64 bd;\n\tsetp.ne.b32 p, %4, 0;\n\tmov.b64 bd, {%2, %6};\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], bd, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "r"(tmem_a), "r"(bdesc_lo), "r"(idesc), "r"(accumulate), "r"(z), "r"(MMA_DESC_HI) : "memory");
}
// 32 lanes x 32 columns: each thread of the warp stores its 32 registers into its own lane
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
                 "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,"
                 "%29,%30,%31,%32};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                   "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
                   "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
                   "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
                 : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
// K-major SWIZZLE_128B shared-memory matrix descriptor: rows of 128 bytes, 8-row groups 1024 bytes apart
__device__ __forceinline__ uint64_t mma_smem_desc(uint32_t saddr)
{
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ uint32_t mma_idesc(int n_cols)      // u8 x u8 -> s32, both K-major, M = 128
{
    return (2u << 4) | ((uint32_t)(n_cols >> 3) << 17) | ((128u >> 4) << 24);
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
    int tmem_cols;        // allocated columns (power of two >= 32)
    int acc_cols;         // columns [0, acc_cols) hold the accumulators: at most this many output blocks per call;
                          // the Toeplitz stages follow
    uint8_t *brows;       // the row operand in swizzled 128-byte rows, 1024-byte aligned
    int brows_cap;        // rows available at brows
    uint32_t bar;         // shared address of the mbarriers: full[s] at +8 s, empty[s] at +64 + 8 s, done at +128
    uint32_t it;          // tiles produced so far (stage index and barrier parities follow from it)
    uint32_t ndone;       // products finished so far (parity of the done barrier)
    uint32_t fail;        // set when a bounded wait gave up: the engine is retired for this block
};

__device__ unsigned int g_mma_fail;   // bounded waits that gave up (expected 0); reported with the debug counters

constexpr int MMA_BAR_BYTES = 256;    // full[s] (up to 8), empty[s] (up to 8), done, TMEM slot

// Warp roles for a block of T threads: the last warp issues the MMAs; of the others, groups of four warps
// (one per 32-lane quarter of tensor memory) generate Toeplitz tiles.  Group g owns the tiles t = g mod G and
// cycles through its own PER_GROUP stages, so that every producer warp sees every phase of the stage
// barriers it waits on (a warp that skipped a phase would misread the parity).
template <int T>
struct MmaRoles {
    static constexpr int WARPS = T / 32;
    // 128 threads: the four warps all produce and thread 0 issues the MMAs of a step right after its own row
    // (COMBINED); four such blocks share an SM, so each gets 128 TMEM columns: 64 accumulators + 2 stages.
    static constexpr bool COMBINED = (WARPS == 4);
    static constexpr int GROUPS = COMBINED ? 1 : (WARPS - 1) / 4;
    static constexpr int PER_GROUP = COMBINED ? 2 : (GROUPS == 1 ? 4 : 2);
    static constexpr int STAGES = GROUPS * PER_GROUP;
    static constexpr int ISSUER = COMBINED ? 0 : T - 32;
    static_assert(GROUPS >= 1 && STAGES <= 6, "128, 256 or 512 threads");
    // stage and use count of global tile number t
    __device__ static __forceinline__ int stage(uint32_t t) { return (int)(t % GROUPS) * PER_GROUP + (int)((t / GROUPS) % PER_GROUP); }
    __device__ static __forceinline__ uint32_t use(uint32_t t) { return (t / GROUPS) / PER_GROUP; }
};

// One-time setup per block: mbarriers, TMEM allocation (warp 0 owns it).  All threads call it.
template <int T>
__device__ __forceinline__ void mma_init(MmaCtx &cx, uint8_t *brows, int brows_cap, uint8_t *bars, int tmem_cols)
{
    cx.brows = brows;
    cx.brows_cap = brows_cap;
    cx.bar = smem_u32(bars);
    cx.tmem_cols = tmem_cols;
    cx.acc_cols = tmem_cols - MmaRoles<T>::STAGES * MMA_STAGE_COLS;
    cx.it = 0;
    cx.ndone = 0;
    cx.fail = 0;
    uint32_t *slot = reinterpret_cast<uint32_t *>(bars + 144);
    if (threadIdx.x == 0) {
        for (int s = 0; s < MmaRoles<T>::STAGES; s++) {
            mbar_init(cx.bar + 8 * s, 4);             // one arrival per producer warp of the group
            mbar_init(cx.bar + 64 + 8 * s, 1);        // tcgen05.commit
        }
        mbar_init(cx.bar + 128, 1);
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

// One row of a Toeplitz tile in registers: word m holds bytes j = 4m .. 4m+3 of out[j] = a[x0 - j], x0 = 128 p + row.
// W = the operand's limbs, nw = valid words (zero outside [0, nw)); CHECK = false skips the bounds tests.
template <bool CHECK>
__device__ __forceinline__ void toeplitz_row(const limb *W, int nw, int x0, uint32_t (&o)[32])
{
    const int z0 = x0 - 3;                                   // lowest byte of the first output word
    const int s = z0 & 3;
    const uint32_t sel = (uint32_t)(s + 3) | ((uint32_t)(s + 2) << 4) | ((uint32_t)(s + 1) << 8) | ((uint32_t)s << 12);
    const int wi = z0 >> 2;                                  // floor(z0 / 4), also for negative z0
    auto ld = [&](int i) -> uint32_t { return CHECK ? ((i >= 0 && i < nw) ? W[i] : 0u) : W[i]; };
    uint32_t hi = ld(wi + 1);
#pragma unroll
    for (int m = 0; m < 32; ++m) {
        const uint32_t lo = ld(wi - m);
        o[m] = __byte_perm(lo, hi, sel);                     // bytes a[z+3], a[z+2], a[z+1], a[z]
        hi = lo;
    }
}

// Steps (Toeplitz tiles) a range product needs when `na` is the Toeplitz operand.
__device__ __forceinline__ int mma_steps(int na, int nb, int dlo, int dhi)
{
    const int Ea = (na + 31) / 32, Eb = (nb + 31) / 32;
    return min(Ea, dhi - 1) - max(0, dlo - Eb + 1) + 1;
}

// Should this range product run on the tensor core?  Cost model in cycles of a block alone on its SM: a step
// (four MMA instructions) is entered as 700 cycles and a call as 12 000 cycles of fixed work (row operand,
// epilogue, final add), against about 1/26 cycle per limb product on the IMAD path; MMA_PLAN_PCT scales the
// tensor side to what is measured (a step of the warp-issued loop takes ~330 cycles at N <= 144).  swap = take
// b as the Toeplitz operand (fewer steps).  Block-uniform.
template <int T>
__device__ __forceinline__ bool mma_plan(const MmaCtx *cx, int na, int nb, int dlo, int dhi, bool &swap)
{
    if (cx == nullptr || cx->fail || na <= 0 || nb <= 0 || dlo < 0) return false;
    dhi = min(dhi, (na + nb + 31) / 32);
    const int N = dhi - dlo, Nn = (N + 15) & ~15;
    if (N <= 0) return false;
    const int sa = mma_steps(na, nb, dlo, dhi), sb = mma_steps(nb, na, dlo, dhi);
    swap = sb < sa;
    const int steps = swap ? sb : sa;
    if (steps <= 0 || Nn > cx->acc_cols || Nn + steps - 1 > cx->brows_cap) return false;
    const long long est = (long long)(32 * N) * (long long)min(na, nb);      // limb products, upper bound
    // the IMAD path of a block of T threads gets T/512 of the SM's 26 limb products per cycle
#ifndef MMA_PLAN_PCT
#define MMA_PLAN_PCT 10     // measured (sweep 3..35 with the warp-issued MMA loop, ~330 cycles per step): 10 % is best at 2^17
                            // bits and within 1 % of the best (6 %) at 2^18 bits; 35 % was the optimum of the thread-issued loop
#endif
    // 128-thread blocks share their SM with three others and their warp 0 both produces and issues: the sweep
    // there gives 20-30 % (config 2: 3.57 M div/s against 3.28 M at 10 % and 3.50 M at 45-70 %)
    constexpr int pct = (T <= 128) ? 25 : MMA_PLAN_PCT;
    return 100 * est >= (long long)(pct * 52 * T / 512) * (700ll * steps + 12000ll);
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
    static_assert(T >= 128 && T % 32 == 0, "a producer group of four warps");
    MmaCtx cx = cx_mem;        // work on a register copy: the asm memory clobbers would reload every field
    const int tid = threadIdx.x, warp = tid >> 5;
    const int Ea = (na + 31) / 32, Eb = (nb + 31) / 32;
    dhi = min(dhi, (na + nb + 31) / 32);
    const int N = dhi - dlo;
    const int Nn = (N + 15) & ~15;
    const int pmin = max(0, dlo - Eb + 1), pmax = min(Ea, dhi - 1);
    const int e0 = dlo - pmax;                                // chunk of b held by row 0
    const int R = (dlo + Nn - 1 - pmin) - e0 + 1;
    if (N <= 0 || pmax < pmin || Nn > cx.acc_cols || R > cx.brows_cap) return -1;

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
    const int nsteps = pmax - pmin + 1;
    using Roles = MmaRoles<T>;
    constexpr int G = Roles::GROUPS;
    const uint32_t a_tmem0 = cx.tmem_base + (uint32_t)cx.acc_cols;
    // The four MMAs of one step for the accumulator columns nc .. nc+255 (products wider than 256 output blocks
    // only; the common case is inlined in warp_issue): D[:, nc..] += A_p x B_p, K = 128 as four instructions of
    // K = 32.  Called by a whole converged warp; one elected lane issues.  The election sits directly around the
    // straight-line tcgen05 code: with a loop inside the elected region ptxas falls back to an ELECT / BRA.U.ANY
    // loop around every instruction.
    auto issue_mmas = [&](int step, int s, int nc) {
        const int p = pmin + step;
        uint32_t d_tmem = cx.tmem_base + (uint32_t)nc;
        uint32_t a_tmem = a_tmem0 + (uint32_t)(MMA_STAGE_COLS * s);
        uint32_t b_lo = mma_desc_lo(smem_u32(cx.brows + (dlo + nc - p - e0) * 128));   // + 2 per K slice of 32 bytes
        uint32_t idesc = mma_idesc(min(256, Nn - nc));
        uint32_t acc0 = step > 0 ? 1u : 0u;
        // every lane computes the operand words; the empty asm keeps the arithmetic out of the elected branch
        asm volatile("" : "+r"(d_tmem), "+r"(a_tmem), "+r"(b_lo), "+r"(idesc), "+r"(acc0));
        if (elect_one()) {
            tc_mma_i8_ts_lo(d_tmem, a_tmem, b_lo, idesc, acc0);
            tc_mma_i8_ts_lo(d_tmem, a_tmem + 8, b_lo + 2, idesc, 1u);
            tc_mma_i8_ts_lo(d_tmem, a_tmem + 16, b_lo + 4, idesc, 1u);
            tc_mma_i8_ts_lo(d_tmem, a_tmem + 24, b_lo + 6, idesc, 1u);
        }
    };
    // One step issued by a whole converged warp: poll the tile's `full` barrier (stage s, parity par), then one
    // elected lane issues the MMAs and the commit.  b_lo = descriptor word of the row that column 0 reads at this
    // step.  The warp's own instructions are the critical path of the MMA loop (a tensor-core step takes 2 N
    // cycles, 256 for N = 128), so the operand words are prepared by every lane in ordinary registers (the empty
    // asm keeps the arithmetic out of the elected branch) and the elected region is straight-line code.
    auto warp_issue = [&](int step, int s, uint32_t par, uint32_t b_lo) -> bool {
        if (!mbar_wait(cx.bar + 8 * s, par)) return false;
        tc_fence_after();
        if (Nn <= 256) {
            uint32_t d_tmem = cx.tmem_base, a_tmem = a_tmem0 + (uint32_t)(MMA_STAGE_COLS * s);
            uint32_t idesc = mma_idesc(Nn), acc0 = step > 0 ? 1u : 0u, ebar = cx.bar + 64 + 8 * s;
            asm volatile("" : "+r"(d_tmem), "+r"(a_tmem), "+r"(b_lo), "+r"(idesc), "+r"(acc0), "+r"(ebar));
            if (elect_one()) {
                tc_mma_i8_ts_lo(d_tmem, a_tmem, b_lo, idesc, acc0);
                tc_mma_i8_ts_lo(d_tmem, a_tmem + 8, b_lo + 2, idesc, 1u);
                tc_mma_i8_ts_lo(d_tmem, a_tmem + 16, b_lo + 4, idesc, 1u);
                tc_mma_i8_ts_lo(d_tmem, a_tmem + 24, b_lo + 6, idesc, 1u);
                tc_commit(ebar);
            }
        } else {
            for (int nc = 0; nc < Nn; nc += 256) issue_mmas(step, s, nc);
            if (elect_one()) tc_commit(cx.bar + 64 + 8 * s);      // frees the step's Toeplitz stage
        }
        return true;
    };
    const uint32_t b_lo_first = mma_desc_lo(smem_u32(cx.brows + (dlo - pmin - e0) * 128));   // step 0, column 0
    if (warp < 4 * G) {
        // ---- Toeplitz producers: warp j fills lanes 32 (j % 4) .. +31 of the tiles of group j / 4 ----
        const int grp = warp >> 2, row = tid & 127;
        for (int step = 0; step < nsteps; ++step) {
            const uint32_t t = cx.it + (uint32_t)step;
            if ((int)(t % G) != grp) continue;
            const int p = pmin + step;
            const int s = Roles::stage(t);
            const uint32_t use = Roles::use(t);
            if (use >= 1 && !mbar_wait(cx.bar + 64 + 8 * s, (use - 1) & 1)) { cx.fail = 1; break; }
            tc_fence_after();
            uint32_t o[32];
            if (p >= 1 && 32 * p + 33 <= na) toeplitz_row<false>(A, na, 128 * p + row, o);
            else toeplitz_row<true>(A, na, 128 * p + row, o);
            tmem_st32(a_tmem0 + ((uint32_t)(row & ~31) << 16) + (uint32_t)(MMA_STAGE_COLS * s), o);
            tc_fence_before();
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(cx.bar + 8 * s);
            if (Roles::COMBINED && warp == 0 &&            // 128-thread blocks: warp 0 also issues the step
                !warp_issue(step, s, use & 1, b_lo_first - 8u * (uint32_t)step)) { cx.fail = 2; break; }
        }
        if (Roles::COMBINED && warp == 0) {
            if (elect_one()) tc_commit(cx.bar + 128);
            __syncwarp();
        }
    } else if (!Roles::COMBINED && warp == Roles::ISSUER / 32) {
        // ---- the MMA issuer: the whole warp walks the steps (uniform control flow); stage index, barrier parity
        // and descriptor word are carried incrementally (no division by GROUPS per step)
        uint32_t tg = cx.it % (uint32_t)G, tq = cx.it / (uint32_t)G;              // tile t = tq * G + tg
        uint32_t b_lo = b_lo_first;
        for (int step = 0; step < nsteps; ++step) {
            const int s = (int)tg * Roles::PER_GROUP + (int)(tq % Roles::PER_GROUP);
            if (!warp_issue(step, s, (tq / Roles::PER_GROUP) & 1, b_lo)) { cx.fail = 2; break; }
            b_lo -= 8u;                                          // the next step starts one 128-byte row lower
            if (++tg == (uint32_t)G) { tg = 0; ++tq; }
        }
        if (elect_one()) tc_commit(cx.bar + 128);
        __syncwarp();
    }
    cx.it += (uint32_t)nsteps;
    __syncwarp();

    // ---- epilogue: TMEM lane i, column d  ->  byte-column sum of output byte 128 (dlo + d) + i ----
    if (warp < 4) {
        if (!mbar_wait(cx.bar + 128, cx.ndone & 1)) cx.fail = 3;
        tc_fence_after();
        for (int d0 = 0; d0 < Nn; d0 += 16) {
            uint32_t v[16];
            tmem_ld16(cx.tmem_base + ((uint32_t)(32 * warp) << 16) + d0, v);
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                unsigned long long sv = (unsigned long long)v[k] << (8 * (tid & 3));
                sv += __shfl_xor_sync(0xffffffffu, sv, 1);
                sv += __shfl_xor_sync(0xffffffffu, sv, 2);
                if ((tid & 3) == 0 && d0 + k < N) {
                    const int L = 32 * (d0 + k) + (tid >> 2);
                    P[L] = (uint32_t)sv;
                    HI[L + 1] = (uint32_t)(sv >> 32);
                }
            }
        }
        if (tid == 0) HI[0] = 0u;
        tc_fence_before();
    }
    cx.ndone += 1;
    if (cx.fail) atomicOr(&g_mma_fail, 1u << (cx.fail - 1));
    if (__syncthreads_or(cx.fail != 0)) {
        // a bounded wait gave up somewhere in the block: the accumulators cannot be trusted and the barrier
        // parities are out of step.  Say so (sticky status bit), retire the engine for the rest of this block
        // (mma_plan refuses a failed context) and let the caller redo this product on the IMAD path.
        raise_status(ST_MMA_WAIT);
        cx_mem.fail = 1;
        return -2;
    }
    // ---- P += HI with block-wide carry propagation (the carry out of the top block is dropped: mod B^(32 dhi)) ----
    lin_addsub<T, false>(P, 32 * N, LimbView{P, 32 * N, 0}, LimbView{HI, 32 * N, 0}, 0u, blk);
    cx_mem.it = cx.it;
    cx_mem.ndone = cx.ndone;
    count(CNT_MMA_COLSTEPS, (unsigned long long)nsteps * (unsigned long long)Nn);   // x 16384 = u8 MACs executed
    return 32 * N;
}

}  // namespace mpd
