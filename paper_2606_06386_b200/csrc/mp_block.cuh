// Block-level multi-precision primitives for sm_100a (one big integer per thread block).
//
// Numbers are little-endian arrays of 32-bit limbs held in shared memory for the whole
// division ("the remaining computation uses fast memory").  Every buffer is zero
// padded to a multiple of TILE limbs so that the multiplier can always read whole tiles.
//
// Linear-cost operations (PAPER.md 3.2-3.3): each thread owns 8 consecutive limbs, resolves
// carries sequentially inside them with add.cc/addc.cc chains and publishes a 2-bit
// (generate, propagate) code -- the CarryOP code of PAPER.md:343-358, :440.  Unlike the
// paper's shuffle scan (Listing 1.6) the codes of a warp are gathered with
// two ballots and the prefix is computed by ONE integer addition: adding the words G|P and G
// ripples a carry through exactly the propagate bits, so (sum ^ (G|P) ^ G) holds the carry
// into every lane.  The same trick over the per-warp codes finishes the block, with a single
// __syncthreads per operation.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mpd {

typedef uint32_t limb;
constexpr int TILE = 8;        // limbs per multiplier tile edge
constexpr int CHUNK = 8;       // limbs per thread in linear operations

__host__ __device__ constexpr int round_up(int x, int m) { return (x + m - 1) / m * m; }

// Sticky status word (include/mpdiv.h: mpdiv_status): conditions only a running kernel can find.
enum : uint32_t { ST_MMA_WAIT = 1u, ST_CORR_BOUND = 2u, ST_REM_RANGE = 4u, ST_V_ZERO = 8u, ST_IO_WAIT = 16u };
__device__ unsigned int g_status;
__device__ __forceinline__ void raise_status(uint32_t bits)
{
    if (threadIdx.x == 0) atomicOr(&g_status, bits);
}

// debug counters (include/mpdiv.h: mpdiv_debug_counters): a few atomics per division
constexpr int NUM_COUNTERS = 24;
__device__ unsigned long long g_counters[NUM_COUNTERS];
enum { CNT_DELTA_NEG = 0, CNT_DELTA_POS, CNT_DELTA_MULTI, CNT_ONE_LIMB, CNT_U_LT_V, CNT_V_ZERO,
       CNT_SIGN_NEG, CNT_POW_B, CNT_TILES, CNT_DELTA_NEG_MULTI, CNT_DELTA_OUT_OF_RANGE, CNT_CLIPPED_STEPS,
       CNT_MMA_PRODUCTS, CNT_MMA_WAIT_FAILURES /* filled by the host from mp_mma.cuh */, CNT_SEED_ADDBACK, CNT_SEEDS,
       CNT_MMA_COLSTEPS, CNT_CLUSTER_DIVS, CNT_CHUNKS, CNT_MMA_UNIT_CYCLES };
__device__ __forceinline__ uint32_t cta_rank_in_cluster()
{
    uint32_t r;
    asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// one count per division: the CTAs of a cluster (mp_mul.cuh) all run the same division, rank 0 counts
__device__ __forceinline__ void count(int which, unsigned long long n = 1ull)
{
    if (threadIdx.x == 0 && cta_rank_in_cluster() == 0) atomicAdd(&g_counters[which], n);
}

// Per-block bookkeeping for the scans/reductions: a double-buffered word per warp.
struct BlkScratch {
    uint32_t code[2][32];
    unsigned long long io_bar;   // mbarrier of the block's bulk copies (mp_io.cuh)
    uint32_t pad_[2];            // keeps whatever follows 16-byte aligned
};

struct Blk {
    BlkScratch *sc;
    uint32_t parity;   // which half of sc->code the next collective uses
    uint32_t tiles;    // 8x8-limb tile products this thread has executed (debug counter)
    uint32_t cl;       // cluster form (mp_mul.cuh): rank | size << 8 | staging set of the next product << 16; else 0
};

// ---------------------------------------------------------------------------------------
// block collectives
// ---------------------------------------------------------------------------------------
// Every primitive is a template on T = the number of threads that take part.  T = 32 is the "narrow"
// form: warp 0 of a larger block runs the operation alone (the early Newton iterations, whose operands
// are a few tiles long), the group barrier is a __syncwarp and the other warps neither spend issue slots
// nor meet a block barrier.
template <int T>
__device__ __forceinline__ void grp_sync()
{
    if (T == 32) __syncwarp();
    else __syncthreads();
}
template <int T>
__device__ __forceinline__ bool grp_or(bool pred)
{
    if (T == 32) return __any_sync(0xffffffffu, pred) != 0;
    return __syncthreads_or(pred) != 0;
}
// The per-warp words of a collective, through explicit shared-memory instructions (a volatile generic pointer compiles to
// LD.E.STRONG.SYS / ST.E.STRONG.SYS).
__device__ __forceinline__ uint32_t code_base(const Blk &blk)
{
    return (uint32_t)__cvta_generic_to_shared(blk.sc->code[blk.parity & 1]);
}
__device__ __forceinline__ void code_put(uint32_t base, uint32_t idx, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(base + 4u * idx), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t code_get(uint32_t base, uint32_t idx)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(base + 4u * idx) : "memory");
    return v;
}

template <int T>
__device__ __forceinline__ int block_max(int v, Blk &blk)
{
    constexpr int NW = T / 32;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = __reduce_max_sync(0xffffffffu, v);
    const uint32_t code = code_base(blk);
    blk.parity++;
    if (lane == 0) code_put(code, warp, (uint32_t)v);
    grp_sync<T>();
    int r = (lane < NW) ? (int)code_get(code, lane) : INT32_MIN;
    return __reduce_max_sync(0xffffffffu, r);
}

// Carry/borrow prefix over the block.  Thread t contributes g (its chunk generates a carry) and
// p (its chunk propagates an incoming carry), never both; cin enters below thread 0.
// Returns the carry into this thread's chunk; cout = carry out of the last thread.
template <int T>
__device__ __forceinline__ uint32_t carry_scan(uint32_t g, uint32_t p, uint32_t cin, Blk &blk,
                                               uint32_t &cout)
{
    constexpr int NW = T / 32;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t G = __ballot_sync(0xffffffffu, g != 0);
    const uint32_t P = __ballot_sync(0xffffffffu, p != 0);
    const uint32_t a = G | P, b = G;
    const uint32_t wg = (uint32_t)(((uint64_t)a + b) >> 32);   // warp generates
    const uint32_t wp = (P == 0xffffffffu) ? 2u : 0u;          // warp propagates
    const uint32_t code = code_base(blk);
    blk.parity++;
    if (lane == 0) code_put(code, warp, wg | wp);
    grp_sync<T>();
    const uint32_t c = (lane < NW) ? code_get(code, lane) : 0u;
    const uint64_t GW = __ballot_sync(0xffffffffu, (c & 1u) != 0);
    const uint64_t PW = __ballot_sync(0xffffffffu, (c & 2u) != 0);
    const uint64_t aw = GW | PW, bw = GW;
    const uint64_t cw = (aw + bw + cin) ^ aw ^ bw;             // bit w = carry into warp w
    cout = (uint32_t)(cw >> NW) & 1u;
    const uint32_t cwarp = (uint32_t)(cw >> warp) & 1u;
    const uint32_t cl = (a + b + cwarp) ^ a ^ b;               // bit l = carry into lane l
    return (cl >> lane) & 1u;
}

// ---------------------------------------------------------------------------------------
// 8-limb chunk arithmetic (in registers)
// ---------------------------------------------------------------------------------------
// r = a + b, returns carry out
__device__ __forceinline__ uint32_t add8(limb (&r)[8], const limb (&a)[8], const limb (&b)[8])
{
    uint32_t c;
    asm("add.cc.u32 %0, %9, %17;\n\t"
        "addc.cc.u32 %1, %10, %18;\n\t"
        "addc.cc.u32 %2, %11, %19;\n\t"
        "addc.cc.u32 %3, %12, %20;\n\t"
        "addc.cc.u32 %4, %13, %21;\n\t"
        "addc.cc.u32 %5, %14, %22;\n\t"
        "addc.cc.u32 %6, %15, %23;\n\t"
        "addc.cc.u32 %7, %16, %24;\n\t"
        "addc.u32 %8, 0, 0;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
          "=r"(r[7]), "=r"(c)
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]), "r"(a[7]),
          "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(b[4]), "r"(b[5]), "r"(b[6]), "r"(b[7]));
    return c;
}

// r = a - b, returns borrow out (0/1)
__device__ __forceinline__ uint32_t sub8(limb (&r)[8], const limb (&a)[8], const limb (&b)[8])
{
    uint32_t c;
    asm("sub.cc.u32 %0, %9, %17;\n\t"
        "subc.cc.u32 %1, %10, %18;\n\t"
        "subc.cc.u32 %2, %11, %19;\n\t"
        "subc.cc.u32 %3, %12, %20;\n\t"
        "subc.cc.u32 %4, %13, %21;\n\t"
        "subc.cc.u32 %5, %14, %22;\n\t"
        "subc.cc.u32 %6, %15, %23;\n\t"
        "subc.cc.u32 %7, %16, %24;\n\t"
        "subc.u32 %8, 0, 0;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
          "=r"(r[7]), "=r"(c)
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]), "r"(a[7]),
          "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(b[4]), "r"(b[5]), "r"(b[6]), "r"(b[7]));
    return c & 1u;
}

// r += c (c small), returns carry out
__device__ __forceinline__ uint32_t inc8(limb (&r)[8], uint32_t cin)
{
    uint32_t c;
    asm("add.cc.u32 %0, %0, %9;\n\t"
        "addc.cc.u32 %1, %1, 0;\n\t"
        "addc.cc.u32 %2, %2, 0;\n\t"
        "addc.cc.u32 %3, %3, 0;\n\t"
        "addc.cc.u32 %4, %4, 0;\n\t"
        "addc.cc.u32 %5, %5, 0;\n\t"
        "addc.cc.u32 %6, %6, 0;\n\t"
        "addc.cc.u32 %7, %7, 0;\n\t"
        "addc.u32 %8, 0, 0;"
        : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]),
          "+r"(r[7]), "=r"(c)
        : "r"(cin));
    return c;
}

// r -= c (c in {0,1}), returns borrow out
__device__ __forceinline__ uint32_t dec8(limb (&r)[8], uint32_t cin)
{
    uint32_t c;
    asm("sub.cc.u32 %0, %0, %9;\n\t"
        "subc.cc.u32 %1, %1, 0;\n\t"
        "subc.cc.u32 %2, %2, 0;\n\t"
        "subc.cc.u32 %3, %3, 0;\n\t"
        "subc.cc.u32 %4, %4, 0;\n\t"
        "subc.cc.u32 %5, %5, 0;\n\t"
        "subc.cc.u32 %6, %6, 0;\n\t"
        "subc.cc.u32 %7, %7, 0;\n\t"
        "subc.u32 %8, 0, 0;"
        : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]),
          "+r"(r[7]), "=r"(c)
        : "r"(cin));
    return c & 1u;
}

__device__ __forceinline__ bool all_eq8(const limb (&r)[8], limb x)
{
    return ((r[0] ^ x) | (r[1] ^ x) | (r[2] ^ x) | (r[3] ^ x) | (r[4] ^ x) | (r[5] ^ x) |
            (r[6] ^ x) | (r[7] ^ x)) == 0;
}

// ---------------------------------------------------------------------------------------
// linear operations on shared-memory numbers
// ---------------------------------------------------------------------------------------
// dst[i] = fa(i) +/- fb(i) +/- carry for i in [0, len), len a multiple of 8.  fa/fb return the
// limb of each operand at index i (0 outside the operand): shifts by whole limbs
// (shift_n) are folded into these index maps instead of being
// materialised.  Map-scan-map of PAPER.md:423-432.  Returns the final carry (borrow).
// dst may alias an operand only when that operand is read at the same index it is written.
// Ends with a __syncthreads: dst is visible to the whole block on return.
// one chunk of lin_addsub: r = fa +/- fb over limbs i0 .. i0 + 7; g = carry (borrow) out, p = an incoming one passes through
template <bool SUB, class FA, class FB>
__device__ __forceinline__ void lin_chunk(limb (&r)[8], uint32_t &g, uint32_t &p, int i0, const FA &fa, const FB &fb)
{
    limb a[8], b[8];
#pragma unroll
    for (int j = 0; j < 8; j++) {
        a[j] = fa(i0 + j);
        b[j] = fb(i0 + j);
    }
    if (SUB) {
        g = sub8(r, a, b);
        p = all_eq8(r, 0u);
    } else {
        g = add8(r, a, b);
        p = all_eq8(r, 0xffffffffu);
    }
}
template <bool SUB>
__device__ __forceinline__ void lin_finish(limb *dst, limb (&r)[8], uint32_t c)
{
    if (SUB) dec8(r, c); else inc8(r, c);
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    d4[0] = make_uint4(r[0], r[1], r[2], r[3]);
    d4[1] = make_uint4(r[4], r[5], r[6], r[7]);
}

// (A form in which warp 0 also takes up to 32 tail chunks in the same scan -- the operands of a division are a few guard
// limbs longer than 8 T, so full-size operations need a second pass for a handful of limbs -- was measured and lost
// 2 % even at a single call site, 19 % everywhere: the inlined code doubles.)
template <int T, bool SUB, class FA, class FB>
__device__ __forceinline__ uint32_t lin_addsub(limb *dst, int len, FA fa, FB fb, uint32_t cin,
                                               Blk &blk)
{
    for (int base = 0; base < len; base += CHUNK * T) {
        const int i0 = base + CHUNK * (int)threadIdx.x;
        limb r[8];
        const bool active = i0 < len;
        uint32_t g = 0, p = active ? 0u : 1u;   // idle threads pass the carry on to the block's cout
        if (active) lin_chunk<SUB>(r, g, p, i0, fa, fb);
        uint32_t cout;
        const uint32_t c = carry_scan<T>(g, p, cin, blk, cout);
        if (active) lin_finish<SUB>(dst + i0, r, c);
        cin = cout;
    }
    grp_sync<T>();
    return cin;
}

// limb i of a number stored at p with n valid limbs, read at index i + off (0 outside)
struct LimbView {
    const limb *p;
    int n;
    int off;
    __device__ __forceinline__ limb operator()(int i) const
    {
        const int j = i + off;
        return (j >= 0 && j < n) ? p[j] : 0u;
    }
};
struct NotView {   // ~x over [0, n), 0 outside: used for B^n - x = ~x + 1.
    const limb *p; // x has `valid` readable limbs (zero beyond)
    int n;
    int valid;
    __device__ __forceinline__ limb operator()(int i) const
    {
        return (i < n) ? ~((i < valid) ? p[i] : 0u) : 0u;
    }
};
struct ZeroView {
    __device__ __forceinline__ limb operator()(int) const { return 0u; }
};

// dst[0..len) = src[i + off] (0 outside [0, n)); len multiple of 4.  Whole-limb shift / masked copy.
template <int T>
__device__ __forceinline__ void lin_copy(limb *dst, int len, const limb *src, int n, int off)
{
    for (int i = threadIdx.x; i < len; i += T) {
        const int j = i + off;
        dst[i] = (j >= 0 && j < n) ? src[j] : 0u;
    }
    grp_sync<T>();
}

template <int T>
__device__ __forceinline__ void lin_zero(limb *dst, int len)
{
    for (int i = threadIdx.x; i < len; i += T) dst[i] = 0u;
    grp_sync<T>();
}

// any limb of a[lo, hi) non-zero?  (block-uniform result)
template <int T>
__device__ __forceinline__ bool any_nonzero(const limb *a, int lo, int hi)
{
    uint32_t acc = 0;
    for (int i = lo + (int)threadIdx.x; i < hi; i += T) acc |= a[i];
    return grp_or<T>(acc != 0);
}

// a >= b for a of `len` limbs and b of nb <= len limbs (zero above): the less-than of PAPER.md:331-335 as ONE reduction --
// the highest limb in which the numbers differ decides -- instead of a subtraction with a borrow scan whose
// result would be thrown away.  Block-uniform; one block barrier.
template <int T>
__device__ __forceinline__ bool big_ge(const limb *a, int len, const limb *b, int nb, Blk &blk)
{
    int top = -1;
    for (int i = threadIdx.x; i < len; i += T)
        if (a[i] != (i < nb ? b[i] : 0u)) top = i;    // i increases: the last hit is this thread's highest
    top = block_max<T>(top, blk);
    if (top < 0) return true;
    return a[top] > (top < nb ? b[top] : 0u);
}

// number of significant limbs of a[0, n)  ("prec")
template <int T>
__device__ __forceinline__ int prec_of(const limb *a, int n, Blk &blk)
{
    int top = 0;
    for (int i = threadIdx.x; i < n; i += T)
        if (a[i] != 0u) top = i + 1;   // i increases, so the last hit is this thread's highest
    return block_max<T>(top, blk);
}

}  // namespace mpd
