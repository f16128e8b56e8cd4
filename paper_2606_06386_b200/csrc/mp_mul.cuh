// Block-level schoolbook multiplier on 32-bit limbs for sm_100a.
//
// The product of two shared-memory numbers is cut into 8x8-limb tiles (I, J) of the operand
// grid.  A thread owns whole tile DIAGONALS K = I + J (all tiles of a diagonal land on the same
// 16 output limbs 8K..8K+15), so it accumulates a diagonal in registers and touches shared
// memory only to fetch 16 operand limbs per 64 limb products.  Diagonals are dealt to threads
// cyclically (K = t, t + T, ...): for the shapes the division produces (n x n, 2n x n with
// T = n/8 threads) the lengths of a thread's diagonals add up to the same number of tiles for
// every thread -- the load-balancing idea of PAPER.md:446-448 / Fig. 2 (first-half columns paired
// with mirrored second-half columns), re-expressed on tiles.
//
// Inner tile: 64 x IMAD.WIDE.U32 with the carry in a predicate.  For a fixed a_i the products
// a_i*b_j with i+j even fill the aligned register pairs (c, c+1) of accumulator E, those with
// i+j odd the pairs of accumulator O (O is the same number shifted by one limb), so each
// parity class is ONE carry chain  mad.lo.cc / madc.hi.cc ... which ptxas fuses into
// IMAD.WIDE.U32 R, P = a, b, R (.X for the carry-in): one multiply-pipe slot per limb product.
// The carry out of a chain goes to a small counter (one IADD per 4 products, on the ALU pipe).
//
// Truncated ("close") products, MULTMOD of PAPER.md:105-106, simply stop at the diagonal that
// holds limb L-1: the skipped tiles are never computed.
//
// Carry resolution (once per product): diagonal K leaves 17 limbs D_K = LO (8) | HI (8) | OV (1).
// Column block K of the result is LO[K] + HI[K-1] + OV[K-2] plus the carry from below, resolved
// with the block carry scan of mp_block.cuh.
#pragma once
#include "mp_block.cuh"

namespace mpd {

// four limb products of one parity class of row a: the 8-limb window held in the four 64-bit
// accumulators (x0..x3) += a * (b0, b1, b2, b3) at limb offsets 0, 2, 4, 6; the carry out of the
// window is counted in cy.  The accumulators are 64-bit registers so that ptxas keeps them in aligned
// register pairs for the whole loop (with 32-bit halves it re-pairs them with moves and XOR swaps).
__device__ __forceinline__ void chain4(uint64_t &x0, uint64_t &x1, uint64_t &x2, uint64_t &x3,
                                       uint32_t &cy, uint32_t a, uint32_t b0, uint32_t b1,
                                       uint32_t b2, uint32_t b3)
{
    asm("{\n\t"
        ".reg .u32 l0, h0, l1, h1, l2, h2, l3, h3;\n\t"
        "mov.b64 {l0, h0}, %0;\n\t"
        "mov.b64 {l1, h1}, %1;\n\t"
        "mov.b64 {l2, h2}, %2;\n\t"
        "mov.b64 {l3, h3}, %3;\n\t"
        "mad.lo.cc.u32 l0, %5, %6, l0;\n\t"
        "madc.hi.cc.u32 h0, %5, %6, h0;\n\t"
        "madc.lo.cc.u32 l1, %5, %7, l1;\n\t"
        "madc.hi.cc.u32 h1, %5, %7, h1;\n\t"
        "madc.lo.cc.u32 l2, %5, %8, l2;\n\t"
        "madc.hi.cc.u32 h2, %5, %8, h2;\n\t"
        "madc.lo.cc.u32 l3, %5, %9, l3;\n\t"
        "madc.hi.cc.u32 h3, %5, %9, h3;\n\t"
        "addc.u32 %4, %4, 0;\n\t"
        "mov.b64 %0, {l0, h0};\n\t"
        "mov.b64 %1, {l1, h1};\n\t"
        "mov.b64 %2, {l2, h2};\n\t"
        "mov.b64 %3, {l3, h3};\n\t"
        "}"
        : "+l"(x0), "+l"(x1), "+l"(x2), "+l"(x3), "+r"(cy)
        : "r"(a), "r"(b0), "r"(b1), "r"(b2), "r"(b3));
}

// Accumulators of one tile diagonal: E[p] holds limbs 2p, 2p+1 (limbs 0..15), O[p] limbs 2p+1, 2p+2
// (limbs 1..14), CY the chain-end carries of limbs 8..16.
struct DiagAcc {
    uint64_t E[8];
    uint64_t O[7];
    uint32_t CY[9];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int i = 0; i < 8; i++) E[i] = 0;
#pragma unroll
        for (int i = 0; i < 7; i++) O[i] = 0;
#pragma unroll
        for (int i = 0; i < 9; i++) CY[i] = 0;
    }
};

template <int I>
__device__ __forceinline__ void tile_row(DiagAcc &s, uint32_t a, const uint32_t (&b)[8])
{
    if ((I & 1) == 0) {
        constexpr int p = I / 2;
        // j even -> limb i+j even -> E pairs p..p+3 (limbs i..i+7), carry into limb i+8
        chain4(s.E[p], s.E[p + 1], s.E[p + 2], s.E[p + 3], s.CY[I], a, b[0], b[2], b[4], b[6]);
        // j odd -> limbs i+1..i+8 = O pairs p..p+3, carry into limb i+9
        chain4(s.O[p], s.O[p + 1], s.O[p + 2], s.O[p + 3], s.CY[I + 1], a, b[1], b[3], b[5], b[7]);
    } else {
        constexpr int p = (I - 1) / 2;
        // j even -> limbs i..i+7 = O pairs p..p+3, carry into limb i+8
        chain4(s.O[p], s.O[p + 1], s.O[p + 2], s.O[p + 3], s.CY[I], a, b[0], b[2], b[4], b[6]);
        // j odd -> limbs i+1..i+8 = E pairs p+1..p+4, carry into limb i+9
        chain4(s.E[p + 1], s.E[p + 2], s.E[p + 3], s.E[p + 4], s.CY[I + 1], a, b[1], b[3], b[5], b[7]);
    }
}

__device__ __forceinline__ void tile_mac(DiagAcc &s, const uint32_t (&a)[8], const uint32_t (&b)[8])
{
    tile_row<0>(s, a[0], b);
    tile_row<1>(s, a[1], b);
    tile_row<2>(s, a[2], b);
    tile_row<3>(s, a[3], b);
    tile_row<4>(s, a[4], b);
    tile_row<5>(s, a[5], b);
    tile_row<6>(s, a[6], b);
    tile_row<7>(s, a[7], b);
}

// d[0..N) += x[0..N) + cin as ONE add.cc/addc.cc chain (N = 8 or 9); returns the carry out.
template <int N>
__device__ __forceinline__ uint32_t acc_chain(uint32_t *d, const uint32_t *x, uint32_t cin)
{
    static_assert(N == 8 || N == 9, "chain length");
    uint32_t c;
    if (N == 8) {
        asm("add.cc.u32 %8, %17, 0xffffffff;\n\t"
            "addc.cc.u32 %0, %0, %9;\n\t"
            "addc.cc.u32 %1, %1, %10;\n\t"
            "addc.cc.u32 %2, %2, %11;\n\t"
            "addc.cc.u32 %3, %3, %12;\n\t"
            "addc.cc.u32 %4, %4, %13;\n\t"
            "addc.cc.u32 %5, %5, %14;\n\t"
            "addc.cc.u32 %6, %6, %15;\n\t"
            "addc.cc.u32 %7, %7, %16;\n\t"
            "addc.u32 %8, 0, 0;"
            : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3]), "+r"(d[4]), "+r"(d[5]), "+r"(d[6]), "+r"(d[7]),
              "=&r"(c)
            : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]), "r"(cin));
    } else {
        asm("add.cc.u32 %9, %19, 0xffffffff;\n\t"
            "addc.cc.u32 %0, %0, %10;\n\t"
            "addc.cc.u32 %1, %1, %11;\n\t"
            "addc.cc.u32 %2, %2, %12;\n\t"
            "addc.cc.u32 %3, %3, %13;\n\t"
            "addc.cc.u32 %4, %4, %14;\n\t"
            "addc.cc.u32 %5, %5, %15;\n\t"
            "addc.cc.u32 %6, %6, %16;\n\t"
            "addc.cc.u32 %7, %7, %17;\n\t"
            "addc.cc.u32 %8, %8, %18;\n\t"
            "addc.u32 %9, 0, 0;"
            : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3]), "+r"(d[4]), "+r"(d[5]), "+r"(d[6]), "+r"(d[7]),
              "+r"(d[8]), "=&r"(c)
            : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]), "r"(x[8]),
              "r"(cin));
    }
    return c;
}

// d += x over 17 limbs (no carry out: the top limb of a diagonal sum is small)
__device__ __forceinline__ void add17(uint32_t (&d)[17], const uint32_t (&x)[17])
{
    const uint32_t c = acc_chain<8>(d, x, 0u);
    acc_chain<9>(d + 8, x + 8, c);
}

// D[0..16] = E + (O << 1 limb) + (CY << 8 limbs).
__device__ __forceinline__ void diag_finish(const DiagAcc &s, uint32_t (&d)[17])
{
    uint32_t e[17], o[17];
#pragma unroll
    for (int i = 0; i < 8; i++) { e[2 * i] = (uint32_t)s.E[i]; e[2 * i + 1] = (uint32_t)(s.E[i] >> 32); }
    e[16] = 0u;
    o[0] = 0u;
#pragma unroll
    for (int i = 0; i < 7; i++) { o[2 * i + 1] = (uint32_t)s.O[i]; o[2 * i + 2] = (uint32_t)(s.O[i] >> 32); }
    o[15] = 0u; o[16] = 0u;
#pragma unroll
    for (int i = 0; i < 17; i++) d[i] = e[i];
    const uint32_t c = acc_chain<8>(d, o, 0u);                // limbs 0..7
    acc_chain<9>(d + 8, o + 8, c);                            // limbs 8..16
    acc_chain<9>(d + 8, s.CY, 0u);                            // chain-end carries enter at limb 8
}

// 8 limbs from shared memory at the 32-bit shared-window address `saddr` (16-byte aligned).
__device__ __forceinline__ void load_tile(uint32_t (&x)[8], uint32_t saddr)
{
    asm("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x[0]), "=r"(x[1]), "=r"(x[2]), "=r"(x[3]) : "r"(saddr));
    asm("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(x[4]), "=r"(x[5]), "=r"(x[6]), "=r"(x[7]) : "r"(saddr));
}
__device__ __forceinline__ void load_tile(uint32_t (&x)[8], const limb *p)
{
    const uint4 lo = reinterpret_cast<const uint4 *>(p)[0];
    const uint4 hi = reinterpret_cast<const uint4 *>(p)[1];
    x[0] = lo.x; x[1] = lo.y; x[2] = lo.z; x[3] = lo.w;
    x[4] = hi.x; x[5] = hi.y; x[6] = hi.z; x[7] = hi.w;
}

// Scratch of one product: P (in/out, product-sized), HI (product-sized), OV and C3 (one word per
// column block).  All sized for KdMax column blocks by the caller.
struct MulScratch {
    limb *HI;
    uint32_t *OV;
    uint32_t *C3;
    limb *ST;        // cluster form only: two staging sets of (LO | HI | OV), stage_cap limbs per LO and per HI
    int stage_cap;
};

// ---------------------------------------------------------------------------------------
// A thread-block CLUSTER per division (a batch smaller than the GPU leaves
// most SMs idle and a lone block spends more than half of a 2^15-bit division in its tile diagonals).  Every CTA of the
// cluster holds the whole state of the division and runs every linear operation itself -- those are latency bound
// and gain nothing from more threads -- but a product's tile diagonals are dealt over ALL lanes of the cluster: a CTA
// accumulates its share and writes each finished diagonal (LO | HI | OV) into the staging set of EVERY CTA through
// distributed shared memory (mapa + st.shared::cluster), one cluster barrier makes the sets complete, and each CTA
// resolves the carries from its own copy into its own product buffer.  The staging sets alternate between
// products, so one barrier per product suffices: a CTA that is writing set s for product i + 2 has passed the barrier
// of product i + 1, which every CTA reaches only after it has read set s of product i.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_size()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_map(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cluster_st4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    asm volatile("st.shared::cluster.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void cluster_st1(uint32_t addr, uint32_t a)
{
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(a) : "memory");
}

// Phase 1: tile diagonals 0..Kd-1 of A (Na tiles) x Bp (Nb tiles) -> P (low 8 limbs of each
// diagonal), HI, OV.  Operands must be 16-byte aligned and zero padded to whole tiles.
//
// A diagonal is shared by a GROUP of C = 2^sh consecutive lanes (C >= 4): lane c of the group takes
// tiles I = Ilo + c, Ilo + c + C, ... and the C partial 17-limb sums are added with a shuffle
// butterfly.  Consecutive groups of a warp own consecutive diagonals, whose lengths differ by one
// tile, so the trip counts of the 32 lanes of a warp differ by at most ceil(8 / C) -- the ramps of
// the product no longer idle three lanes in four -- and a block has C times more threads than
// diagonals per pass, which is what small products (config 1) need.  Diagonals are dealt in passes of
// T / 4 (cyclically: the up-ramp / plateau / down-ramp profile of a full product balances over the
// passes; snake = true reverses odd passes, which balances the single ramp of a truncated product).
// A pass that has fewer diagonals left than groups widens its groups (up to a whole warp).
// CL: the cluster form (above): crank / csize = this CTA's rank in its cluster and the cluster's size; P, HI, OV are the
// staging set of this product.
// COMPACT: one copy of the 64-product tile in a plain loop instead of two in a ping-pong loop plus a tail copy.  A
// latency-bound division runs ONE warp per scheduler through code that is cold at every call (a tile is ~165
// instructions = 21 lines of instruction cache): at config 1 a tile then costs ~750 cycles of instruction fetch against
// ~300 once its code is resident, so fewer copies of it beat the hidden operand latency of the ping-pong form.
template <int T, bool CL, bool COMPACT = false>
__device__ __forceinline__ uint32_t mul_diagonals_body(const limb *A, int Na, const limb *Bp, int Nb, int Klo, int Kd,
                                                       limb *P, limb *HI, uint32_t *OV, bool snake, int crank, int csize)
{   // everything by value: a reference argument of a noinline function lives in local memory
    // lanes per diagonal: 4 for long diagonals, fewer when a diagonal has only a tile or two (the shuffle
    // reduction then costs more than it saves); a pass with spare threads widens its groups, but never
    // beyond one lane per two tiles
    const int maxlen = min(Na, Nb);
    const int sh0 = maxlen <= 2 ? 0 : (maxlen <= 4 ? 1 : 2);
    int shmax = sh0;
    while (shmax < 5 && (2 << shmax) <= maxlen) ++shmax;
    const int TT = CL ? T * csize : T;              // lanes that share the product
    const int G0 = TT >> sh0;                       // diagonals per full pass
    int pass = 0;
    uint32_t tiles = 0;
    for (int base = Klo; base < Kd; base += G0, ++pass) {
        const int ndiag = min(G0, Kd - base);
        int sh = sh0;
        while (sh < shmax && (ndiag << (sh + 1)) <= TT) ++sh;
        const int C = 1 << sh;
        // the groups of the cluster's CTAs interleave, so that neighbouring diagonals (similar lengths) go to different CTAs
        // (giving a group a PAIR of diagonals of complementary lengths to level a single-ramp product was measured and
        // lost 15 %: the fixed cost per diagonal -- first loads, finish, lane reduction, stores -- outweighs the balance)
        const int g = CL ? ((int)threadIdx.x >> sh) * csize + crank : (int)threadIdx.x >> sh;
        const int c = (int)threadIdx.x & (C - 1);
        const bool act = g < ndiag;
        const int K = base + ((snake && (pass & 1)) ? (ndiag - 1 - g) : g);
        const int Ilo = max(0, K - Nb + 1), Ihi = act ? min(Na - 1, K) : -1;
        DiagAcc s;
        s.clear();
        int I = Ilo + c;
        if (I <= Ihi) {
            tiles += ((uint32_t)(Ihi - I) >> sh) + 1u;
            uint32_t a0[8], b0[8], a1[8], b1[8];
            const int step = 4 * TILE * C;                  // bytes between a lane's consecutive tiles
            uint32_t pa = (uint32_t)__cvta_generic_to_shared(A) + 4 * TILE * I;
            uint32_t pb = (uint32_t)__cvta_generic_to_shared(Bp) + 4 * TILE * (K - I);
            if (COMPACT) {
#pragma unroll 1
                for (; I <= Ihi; I += C) {
                    load_tile(a0, pa);
                    load_tile(b0, pb);
                    pa += step; pb -= step;
                    tile_mac(s, a0, b0);
                }
            } else {
            load_tile(a0, pa);
            load_tile(b0, pb);
            // two tiles per trip with ping-pong operand registers (no register copies)
            for (; I + C <= Ihi; I += 2 * C) {
                pa += step; pb -= step;
                load_tile(a1, pa);
                load_tile(b1, pb);
                tile_mac(s, a0, b0);
                if (I + 2 * C <= Ihi) {
                    pa += step; pb -= step;
                    load_tile(a0, pa);
                    load_tile(b0, pb);
                }
                tile_mac(s, a1, b1);
            }
            if (I <= Ihi) tile_mac(s, a0, b0);
            }
        }
        uint32_t d[17];
        diag_finish(s, d);
        for (int off = 1; off < C; off <<= 1) {
            uint32_t x[17];
#pragma unroll
            for (int i = 0; i < 17; i++) x[i] = __shfl_xor_sync(0xffffffffu, d[i], off);
            add17(d, x);
        }
        if (CL) {
            if (act && c == 0) {                     // the finished diagonal goes to the staging set of every CTA
                const uint32_t lp = (uint32_t)__cvta_generic_to_shared(P + TILE * K);
                const uint32_t lh = (uint32_t)__cvta_generic_to_shared(HI + TILE * K);
                const uint32_t lo = (uint32_t)__cvta_generic_to_shared(OV + K);
                for (int rk = 0; rk < csize; ++rk) {
                    const uint32_t rp = cluster_map(lp, (uint32_t)rk), rh = cluster_map(lh, (uint32_t)rk);
                    cluster_st4(rp, d[0], d[1], d[2], d[3]);
                    cluster_st4(rp + 16, d[4], d[5], d[6], d[7]);
                    cluster_st4(rh, d[8], d[9], d[10], d[11]);
                    cluster_st4(rh + 16, d[12], d[13], d[14], d[15]);
                    cluster_st1(cluster_map(lo, (uint32_t)rk), d[16]);
                }
            }
        } else if (act && c == 0) {
            uint4 *p4 = reinterpret_cast<uint4 *>(P + TILE * K);
            uint4 *h4 = reinterpret_cast<uint4 *>(HI + TILE * K);
            p4[0] = make_uint4(d[0], d[1], d[2], d[3]);
            p4[1] = make_uint4(d[4], d[5], d[6], d[7]);
            h4[0] = make_uint4(d[8], d[9], d[10], d[11]);
            h4[1] = make_uint4(d[12], d[13], d[14], d[15]);
            OV[K] = d[16];
        }
    }
    if (CL) cluster_sync_all();
    else grp_sync<T>();
    return tiles;
}

template <int T>
__device__ __noinline__ uint32_t mul_diagonals(const limb *A, int Na, const limb *Bp, int Nb, int Klo, int Kd,
                                                  limb *P, limb *HI, uint32_t *OV, bool snake)
{
    return mul_diagonals_body<T, false>(A, Na, Bp, Nb, Klo, Kd, P, HI, OV, snake, 0, 1);
}
template <int T>
__device__ __noinline__ uint32_t mul_diagonals_cluster(const limb *A, int Na, const limb *Bp, int Nb, int Klo, int Kd,
                                                       limb *P, limb *HI, uint32_t *OV, bool snake, int crank, int csize)
{
    return mul_diagonals_body<T, true, true>(A, Na, Bp, Nb, Klo, Kd, P, HI, OV, snake, crank, csize);
}
template <int T>
__device__ __noinline__ uint32_t mul_diagonals_compact(const limb *A, int Na, const limb *Bp, int Nb, int Klo, int Kd,
                                                       limb *P, limb *HI, uint32_t *OV, bool snake)
{
    return mul_diagonals_body<T, false, true>(A, Na, Bp, Nb, Klo, Kd, P, HI, OV, snake, 0, 1);
}

// Phase 2: resolve column blocks Klo..Kc-1 in place: P[K] = P[K] + HI[K-1] + OV[K-2] + carries,
// where only diagonals Klo <= K < Kd contribute (nothing enters from below column block Klo).
// Kc <= Kd + 2.  Ends with __syncthreads.
// Pin: where the low halves of the diagonals are (P itself, or the staging set of the cluster form).
template <int T>
__device__ __forceinline__ uint32_t mul_resolve_body(limb *P, const limb *Pin, int Klo, int Kd, int Kc, const limb *HI,
                                                     const uint32_t *OV, uint32_t *C3, Blk blk)
{   // blk by value (registers); the advanced collective parity is returned
    uint32_t cin = 0;
    for (int base = Klo; base < Kc; base += T) {
        const int K = base + (int)threadIdx.x;
        const bool active = K < Kc;
        limb s[8];
        uint32_t c3 = 0;
        if (active) {
            limb lo[8], hi[8];
            if (K < Kd) load_tile(lo, Pin + TILE * K);
            else {
#pragma unroll
                for (int j = 0; j < 8; j++) lo[j] = 0;
            }
            if (K > Klo && K - 1 < Kd) load_tile(hi, HI + TILE * (K - 1));
            else {
#pragma unroll
                for (int j = 0; j < 8; j++) hi[j] = 0;
            }
            const uint32_t ov = (K - 2 >= Klo && K - 2 < Kd) ? OV[K - 2] : 0u;
            c3 = add8(s, lo, hi);
            c3 += inc8(s, ov);
            C3[K] = c3;
        }
        grp_sync<T>();
        uint32_t g = 0, p = 0;
        if (active) {
            const uint32_t cprev = (K > Klo) ? C3[K - 1] : 0u;
            g = inc8(s, cprev);
            p = all_eq8(s, 0xffffffffu);
        }
        uint32_t cout;
        const uint32_t c = carry_scan<T>(g, p, cin, blk, cout);
        if (active) {
            inc8(s, c);
            uint4 *p4 = reinterpret_cast<uint4 *>(P + TILE * K);
            p4[0] = make_uint4(s[0], s[1], s[2], s[3]);
            p4[1] = make_uint4(s[4], s[5], s[6], s[7]);
        }
        cin = cout;
    }
    grp_sync<T>();
    return blk.parity;
}

template <int T>
__device__ __noinline__ uint32_t mul_resolve(limb *P, int Klo, int Kd, int Kc, limb *HI, uint32_t *OV,
                                                uint32_t *C3, Blk blk)
{
    return mul_resolve_body<T>(P, P, Klo, Kd, Kc, HI, OV, C3, blk);
}
template <int T>
__device__ __noinline__ uint32_t mul_resolve_cluster(limb *P, const limb *Pin, int Klo, int Kd, int Kc, const limb *HI,
                                                     const uint32_t *OV, uint32_t *C3, Blk blk)
{
    return mul_resolve_body<T>(P, Pin, Klo, Kd, Kc, HI, OV, C3, blk);
}

// words of one staging set: LO (cap) | HI (cap) | OV (one word per diagonal), cap a multiple of 32
__host__ __device__ constexpr int stage_set_words(int cap) { return 2 * cap + cap / TILE + 4; }

// The two phases of a product, block form or cluster form (CL).  Pd, HId, OVd, C3d are already offset so that index K
// addresses diagonal K.  In the cluster form the diagonals pass through the staging set blk.cl selects.
template <int T, bool CL>
__device__ __forceinline__ void mul_phases(const limb *A, int Na, const limb *Bp, int Nb, int Klo, int Kd, int Kc, limb *Pd,
                                           limb *HId, uint32_t *OVd, uint32_t *C3d, const MulScratch &ms, Blk &blk, bool snake)
{
    // cluster form: a product of so few diagonals that one CTA covers them in a single pass is computed by every CTA
    // for itself (the state is replicated): the barrier and the remote stores would cost more than the share saves
    if (CL && (Kd - Klo) * 4 > T) {
        const int cap = ms.stage_cap;
        limb *S = ms.ST + ((blk.cl >> 16) & 1u) * (uint32_t)stage_set_words(cap);
        limb *Ps = S - TILE * Klo, *HIs = S + cap - TILE * Klo;
        uint32_t *OVs = S + 2 * cap - Klo;
        blk.tiles += mul_diagonals_cluster<T>(A, Na, Bp, Nb, Klo, Kd, Ps, HIs, OVs, snake, (int)(blk.cl & 0xffu),
                                              (int)((blk.cl >> 8) & 0xffu));
        blk.parity = mul_resolve_cluster<T>(Pd, Ps, Klo, Kd, Kc, HIs, OVs, C3d, blk);
        blk.cl ^= 1u << 16;
    } else {
        if (CL) blk.tiles += mul_diagonals_compact<T>(A, Na, Bp, Nb, Klo, Kd, Pd, HId, OVd, snake);
        else blk.tiles += mul_diagonals<T>(A, Na, Bp, Nb, Klo, Kd, Pd, HId, OVd, snake);
        blk.parity = mul_resolve<T>(Pd, Klo, Kd, Kc, HId, OVd, C3d, blk);
    }
}

// P[0 .. 8*Kc) = (A * Bp) restricted to tile diagonals < Kd, carries resolved.
//   full product      : Kd = Na + Nb - 1 (or more), Kc = Na + Nb
//   product mod B^L   : Kd = Kc = ceil(L / 8); limbs >= L of the last block are not meaningful
// na, nb in limbs; operands zero padded to whole tiles.
template <int T, bool CL = false>
__device__ __forceinline__ void mul_full(const limb *A, int na, const limb *Bp, int nb, limb *P,
                                         const MulScratch &ms, Blk &blk)
{
    const int Na = (na + TILE - 1) / TILE, Nb = (nb + TILE - 1) / TILE;
    const int Kd = Na + Nb - 1;
    mul_phases<T, CL>(A, Na, Bp, Nb, 0, Kd, Na + Nb, P, ms.HI, ms.OV, ms.C3, ms, blk, false);
}

template <int T, bool CL = false>
__device__ __forceinline__ void mul_low(const limb *A, int na, const limb *Bp, int nb, int L, limb *P,
                                        const MulScratch &ms, Blk &blk)
{
    const int Na = (na + TILE - 1) / TILE, Nb = (nb + TILE - 1) / TILE;
    const int Kfull = Na + Nb;
    const int Kc = min((L + TILE - 1) / TILE, Kfull);
    const int Kd = min(Kc, Kfull - 1);
    mul_phases<T, CL>(A, Na, Bp, Nb, 0, Kd, Kc, P, ms.HI, ms.OV, ms.C3, ms, blk, Kd < Kfull - 1);
}

// Clipped ("range") product: only tile diagonals Klo <= K < Khi are computed, so the result is
//     ((A * Bp) - E) mod B^(8*Khi),   0 <= E < B^(8*Klo + 9)
// (E = the omitted low diagonals: column i+j = t holds at most t+1 products < B^2, and the omitted
// columns end at 8*Klo + 6).  The block stores limb 8*Klo + i of that value at P[i] -- the buffers
// only need 8*(Khi - Klo) limbs -- and limbs below 8*Klo are not produced.  Khi is clamped to the
// size of the full product.  Returns the number of limbs stored.
template <int T, bool CL = false>
__device__ __forceinline__ int mul_range(const limb *A, int na, const limb *Bp, int nb, int Klo, int Khi,
                                         limb *P, const MulScratch &ms, Blk &blk)
{
    const int Na = (na + TILE - 1) / TILE, Nb = (nb + TILE - 1) / TILE;
    const int Kfull = Na + Nb;
    const int Kc = min(Khi, Kfull);
    const int Kd = min(Kc, Kfull - 1);
    limb *Pd = P - TILE * Klo, *HId = ms.HI - TILE * Klo;
    uint32_t *OVd = ms.OV - Klo, *C3d = ms.C3 - Klo;
    mul_phases<T, CL>(A, Na, Bp, Nb, Klo, Kd, Kc, Pd, HId, OVd, C3d, ms, blk, true);
    return TILE * max(Kc - Klo, 0);
}

}  // namespace mpd
