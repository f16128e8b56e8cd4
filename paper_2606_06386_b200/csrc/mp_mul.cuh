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

// four limb products of one parity class of row a: (r0..r7) += a * (b0, b1, b2, b3) at limb
// offsets 0, 2, 4, 6; the carry out of limb 7 is counted in cy.
__device__ __forceinline__ void chain4(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3,
                                       uint32_t &r4, uint32_t &r5, uint32_t &r6, uint32_t &r7,
                                       uint32_t &cy, uint32_t a, uint32_t b0, uint32_t b1,
                                       uint32_t b2, uint32_t b3)
{
    asm("mad.lo.cc.u32 %0, %9, %10, %0;\n\t"
        "madc.hi.cc.u32 %1, %9, %10, %1;\n\t"
        "madc.lo.cc.u32 %2, %9, %11, %2;\n\t"
        "madc.hi.cc.u32 %3, %9, %11, %3;\n\t"
        "madc.lo.cc.u32 %4, %9, %12, %4;\n\t"
        "madc.hi.cc.u32 %5, %9, %12, %5;\n\t"
        "madc.lo.cc.u32 %6, %9, %13, %6;\n\t"
        "madc.hi.cc.u32 %7, %9, %13, %7;\n\t"
        "addc.u32 %8, %8, 0;"
        : "+r"(r0), "+r"(r1), "+r"(r2), "+r"(r3), "+r"(r4), "+r"(r5), "+r"(r6), "+r"(r7), "+r"(cy)
        : "r"(a), "r"(b0), "r"(b1), "r"(b2), "r"(b3));
}

// Accumulators of one tile diagonal: E holds limbs 0..15, O limbs 1..14 (index = limb - 1),
// CY the chain-end carries of limbs 8..16.
struct DiagAcc {
    uint32_t E[16];
    uint32_t O[14];
    uint32_t CY[9];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int i = 0; i < 16; i++) E[i] = 0;
#pragma unroll
        for (int i = 0; i < 14; i++) O[i] = 0;
#pragma unroll
        for (int i = 0; i < 9; i++) CY[i] = 0;
    }
};

template <int I>
__device__ __forceinline__ void tile_row(DiagAcc &s, uint32_t a, const uint32_t (&b)[8])
{
    if ((I & 1) == 0) {
        // j even -> column i+j even -> E[i..i+7], carry into limb i+8
        chain4(s.E[I], s.E[I + 1], s.E[I + 2], s.E[I + 3], s.E[I + 4], s.E[I + 5], s.E[I + 6],
               s.E[I + 7], s.CY[I], a, b[0], b[2], b[4], b[6]);
        // j odd -> column odd -> limbs i+1..i+8 = O[i..i+7], carry into limb i+9
        chain4(s.O[I], s.O[I + 1], s.O[I + 2], s.O[I + 3], s.O[I + 4], s.O[I + 5], s.O[I + 6],
               s.O[I + 7], s.CY[I + 1], a, b[1], b[3], b[5], b[7]);
    } else {
        // j even -> column odd -> limbs i..i+7 = O[i-1..i+6], carry into limb i+8
        chain4(s.O[I - 1], s.O[I], s.O[I + 1], s.O[I + 2], s.O[I + 3], s.O[I + 4], s.O[I + 5],
               s.O[I + 6], s.CY[I], a, b[0], b[2], b[4], b[6]);
        // j odd -> column even -> limbs i+1..i+8 = E[i+1..i+8], carry into limb i+9
        chain4(s.E[I + 1], s.E[I + 2], s.E[I + 3], s.E[I + 4], s.E[I + 5], s.E[I + 6], s.E[I + 7],
               s.E[I + 8], s.CY[I + 1], a, b[1], b[3], b[5], b[7]);
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

// D[0..16] = E + (O << 1 limb) + (CY << 8 limbs).  Each asm block is a self-contained carry chain
// (the condition code never has to survive between two asm statements).
__device__ __forceinline__ void diag_finish(const DiagAcc &s, uint32_t (&d)[17])
{
    uint32_t c1;
    d[0] = s.E[0];
    // limbs 1..8 = E[1..8] + O[0..7]
    asm("add.cc.u32 %0, %9, %17;\n\t"
        "addc.cc.u32 %1, %10, %18;\n\t"
        "addc.cc.u32 %2, %11, %19;\n\t"
        "addc.cc.u32 %3, %12, %20;\n\t"
        "addc.cc.u32 %4, %13, %21;\n\t"
        "addc.cc.u32 %5, %14, %22;\n\t"
        "addc.cc.u32 %6, %15, %23;\n\t"
        "addc.cc.u32 %7, %16, %24;\n\t"
        "addc.u32 %8, 0, 0;"
        : "=r"(d[1]), "=r"(d[2]), "=r"(d[3]), "=r"(d[4]), "=r"(d[5]), "=r"(d[6]), "=r"(d[7]),
          "=r"(d[8]), "=r"(c1)
        : "r"(s.E[1]), "r"(s.E[2]), "r"(s.E[3]), "r"(s.E[4]), "r"(s.E[5]), "r"(s.E[6]),
          "r"(s.E[7]), "r"(s.E[8]), "r"(s.O[0]), "r"(s.O[1]), "r"(s.O[2]), "r"(s.O[3]),
          "r"(s.O[4]), "r"(s.O[5]), "r"(s.O[6]), "r"(s.O[7]));
    // limbs 9..16 = E[9..15] + O[8..13] + c1   (add.cc c1 + 0xffffffff recreates the carry)
    asm("add.cc.u32 %0, %8, 0xffffffff;\n\t"
        "addc.cc.u32 %0, %9, %16;\n\t"
        "addc.cc.u32 %1, %10, %17;\n\t"
        "addc.cc.u32 %2, %11, %18;\n\t"
        "addc.cc.u32 %3, %12, %19;\n\t"
        "addc.cc.u32 %4, %13, %20;\n\t"
        "addc.cc.u32 %5, %14, %21;\n\t"
        "addc.cc.u32 %6, %15, 0;\n\t"
        "addc.u32 %7, 0, 0;"
        : "=&r"(d[9]), "=r"(d[10]), "=r"(d[11]), "=r"(d[12]), "=r"(d[13]), "=r"(d[14]),
          "=r"(d[15]), "=r"(d[16])
        : "r"(c1), "r"(s.E[9]), "r"(s.E[10]), "r"(s.E[11]), "r"(s.E[12]), "r"(s.E[13]),
          "r"(s.E[14]), "r"(s.E[15]), "r"(s.O[8]), "r"(s.O[9]), "r"(s.O[10]), "r"(s.O[11]),
          "r"(s.O[12]), "r"(s.O[13]));
    // limbs 8..16 += CY[0..8]
    asm("add.cc.u32 %0, %0, %9;\n\t"
        "addc.cc.u32 %1, %1, %10;\n\t"
        "addc.cc.u32 %2, %2, %11;\n\t"
        "addc.cc.u32 %3, %3, %12;\n\t"
        "addc.cc.u32 %4, %4, %13;\n\t"
        "addc.cc.u32 %5, %5, %14;\n\t"
        "addc.cc.u32 %6, %6, %15;\n\t"
        "addc.cc.u32 %7, %7, %16;\n\t"
        "addc.u32 %8, %8, %17;"
        : "+r"(d[8]), "+r"(d[9]), "+r"(d[10]), "+r"(d[11]), "+r"(d[12]), "+r"(d[13]),
          "+r"(d[14]), "+r"(d[15]), "+r"(d[16])
        : "r"(s.CY[0]), "r"(s.CY[1]), "r"(s.CY[2]), "r"(s.CY[3]), "r"(s.CY[4]), "r"(s.CY[5]),
          "r"(s.CY[6]), "r"(s.CY[7]), "r"(s.CY[8]));
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
};

// Phase 1: tile diagonals 0..Kd-1 of A (Na tiles) x Bp (Nb tiles) -> P (low 8 limbs of each
// diagonal), HI, OV.  Operands must be 16-byte aligned and zero padded to whole tiles.
// Diagonals are dealt in rounds of T: cyclically (thread t takes t, t+T, ...), which balances the
// up-ramp / plateau / down-ramp length profile of a full product, or -- snake = true -- in
// boustrophedon order (odd rounds reversed), which balances the single ramp of a truncated product.
template <int T>
__device__ __noinline__ void mul_diagonals(const limb *A, int Na, const limb *Bp, int Nb, int Kd,
                                              limb *P, const MulScratch &ms, bool snake)
{
    for (int base = 0; base < Kd; base += T) {
        const int j = (snake && ((base / T) & 1)) ? (T - 1 - (int)threadIdx.x) : (int)threadIdx.x;
        const int K = base + j;
        if (K >= Kd) continue;
        const int Ilo = max(0, K - Nb + 1), Ihi = min(Na - 1, K);
        DiagAcc s;
        s.clear();
        if (Ilo <= Ihi) {
            uint32_t a[8], b[8];
            const limb *pa = A + TILE * Ilo;
            const limb *pb = Bp + TILE * (K - Ilo);
            load_tile(a, pa);
            load_tile(b, pb);
            for (int I = Ilo; I < Ihi; ++I) {
                uint32_t an[8], bn[8];
                pa += TILE;
                pb -= TILE;
                load_tile(an, pa);
                load_tile(bn, pb);
                tile_mac(s, a, b);
#pragma unroll
                for (int jj = 0; jj < 8; jj++) { a[jj] = an[jj]; b[jj] = bn[jj]; }
            }
            tile_mac(s, a, b);
        }
        uint32_t d[17];
        diag_finish(s, d);
        uint4 *p4 = reinterpret_cast<uint4 *>(P + TILE * K);
        uint4 *h4 = reinterpret_cast<uint4 *>(ms.HI + TILE * K);
        p4[0] = make_uint4(d[0], d[1], d[2], d[3]);
        p4[1] = make_uint4(d[4], d[5], d[6], d[7]);
        h4[0] = make_uint4(d[8], d[9], d[10], d[11]);
        h4[1] = make_uint4(d[12], d[13], d[14], d[15]);
        ms.OV[K] = d[16];
    }
    __syncthreads();
}

// Phase 2: resolve column blocks 0..Kc-1 in place: P[K] = P[K] + HI[K-1] + OV[K-2] + carries,
// where diagonals >= Kd contribute nothing.  Kc <= Kd + 2.  Ends with __syncthreads.
template <int T>
__device__ __noinline__ void mul_resolve(limb *P, int Kd, int Kc, const MulScratch &ms, Blk &blk)
{
    uint32_t cin = 0;
    for (int base = 0; base < Kc; base += T) {
        const int K = base + (int)threadIdx.x;
        const bool active = K < Kc;
        limb s[8];
        uint32_t c3 = 0;
        if (active) {
            limb lo[8], hi[8];
            if (K < Kd) load_tile(lo, P + TILE * K);
            else {
#pragma unroll
                for (int j = 0; j < 8; j++) lo[j] = 0;
            }
            if (K >= 1 && K - 1 < Kd) load_tile(hi, ms.HI + TILE * (K - 1));
            else {
#pragma unroll
                for (int j = 0; j < 8; j++) hi[j] = 0;
            }
            const uint32_t ov = (K >= 2 && K - 2 < Kd) ? ms.OV[K - 2] : 0u;
            c3 = add8(s, lo, hi);
            c3 += inc8(s, ov);
            ms.C3[K] = c3;
        }
        __syncthreads();
        uint32_t g = 0, p = 0;
        if (active) {
            const uint32_t cprev = (K >= 1) ? ms.C3[K - 1] : 0u;
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
    __syncthreads();
}

// P[0 .. 8*Kc) = (A * Bp) restricted to tile diagonals < Kd, carries resolved.
//   full product      : Kd = Na + Nb - 1 (or more), Kc = Na + Nb
//   product mod B^L   : Kd = Kc = ceil(L / 8); limbs >= L of the last block are not meaningful
// na, nb in limbs; operands zero padded to whole tiles.
template <int T>
__device__ __forceinline__ void mul_full(const limb *A, int na, const limb *Bp, int nb, limb *P,
                                         const MulScratch &ms, Blk &blk)
{
    const int Na = (na + TILE - 1) / TILE, Nb = (nb + TILE - 1) / TILE;
    const int Kd = Na + Nb - 1;
    mul_diagonals<T>(A, Na, Bp, Nb, Kd, P, ms, false);
    mul_resolve<T>(P, Kd, Na + Nb, ms, blk);
}

template <int T>
__device__ __forceinline__ void mul_low(const limb *A, int na, const limb *Bp, int nb, int L, limb *P,
                                        const MulScratch &ms, Blk &blk)
{
    const int Na = (na + TILE - 1) / TILE, Nb = (nb + TILE - 1) / TILE;
    const int Kfull = Na + Nb;
    const int Kc = min((L + TILE - 1) / TILE, Kfull);
    const int Kd = min(Kc, Kfull - 1);
    mul_diagonals<T>(A, Na, Bp, Nb, Kd, P, ms, Kd < Kfull - 1);
    mul_resolve<T>(P, Kd, Kc, ms, blk);
}

}  // namespace mpd
