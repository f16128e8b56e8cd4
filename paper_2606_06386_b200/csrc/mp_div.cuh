// Whole shifted inverse (Alg. 1-2) and division (Alg. 3) for
// one big integer per thread block, operands resident in shared memory.
//
// Reading of the garbled Algorithm 1:
//   * the loop runs  ceil(log2(H-1)) + 2  times with H = max(h-k, 2)            (printed bound)
//   * guard digits g = 2; the final shift is -(g + H - (h-k))                   (PAPER.md:92 l.26-27)
//   * Step's negative branch subtracts one more when the discarded low limbs of w*x are
//     non-zero (floor of a negative number, eq. (2))
//   * the divisor prefix drops s limbs with s rounded DOWN to a multiple of 4 so that the prefix
//     stays 16-byte aligned in shared memory; a longer prefix is always admissible.
//   * one-limb divisors (Alg. 1 l.6 "divide by 1 digit") are mapped to two-limb ones:
//     floor(B^h / v) = floor(B^(h+1) / (v*B)), and (u*B) div (v*B) = u div v with remainder r*B.
//
// Variants.  MPDIV_VARIANT_PRINTED runs Alg. 1-3 as printed: full products w*x, u*shinv, v*q and the
// close product v'w mod B^L.  MPDIV_VARIANT_CLIPPED (default) is the paper's first future-work item
// (clipped products): every product computes only the tile
// diagonals whose limbs the step keeps --
//   * v'w : columns [c, L) only, c = 8*(floor((c_x - 9)/8) - 1), c_x = d + 1 - prec(w) the lowest limb
//           of x that can still move a kept limb of w*x;  x = P or ~P on those limbs (no borrow scan)
//   * w*x : columns >= d + 1 - 9 only (the shift drops d + 1 limbs)
//   * u*shinv : columns >= h - 9 only;   v*q : columns < k + 3 only (|u - v q0| < 4v)
// An omitted low part E satisfies 0 <= E < B^(8 Klo + 9) (mp_mul.cuh), i.e. less than one unit of the
// lowest kept limb, so every iterate moves by a few units of its lowest GUARD limb, the shifted inverse
// by at most one unit (lambda in {-1,0,1}) and the quotient estimate by at most 2; the correction of
// Alg. 3 becomes two bounded loops (r < 0: q-1, r+v;  r >= v: q+1, r-v) and the result stays exact.
// Iterations whose operands are too short for the window to clip anything run the printed code.
#pragma once
#include "mp_mul.cuh"
#include "mp_mma.cuh"

namespace mpd {

__device__ __forceinline__ void count_tiles(Blk &blk)
{
    uint32_t t = __reduce_add_sync(0xffffffffu, blk.tiles);
    if ((threadIdx.x & 31) == 0 && t != 0) atomicAdd(&g_counters[CNT_TILES], (unsigned long long)t);
    blk.tiles = 0;
}

// significant limbs of a shared-memory number known to have at most `bound` limbs.
// Every warp scans the same (stable) words from the top, 32 per step (lane j looks at limb bound - 1 - j), so the
// result is block-uniform without a barrier; the calling warps must be converged.
__device__ __forceinline__ int top_prec(const limb *a, int bound)
{
    const int lane = (int)(threadIdx.x & 31);
    while (bound > 0) {
        const int i = bound - 1 - lane;
        const uint32_t nz = __ballot_sync(0xffffffffu, i >= 0 && a[i] != 0u);
        if (nz) return bound - (__ffs(nz) - 1);
        bound -= 32;
    }
    return 0;
}

struct UnitView {   // B^pos
    int pos;
    __device__ __forceinline__ limb operator()(int i) const { return i == pos ? 1u : 0u; }
};

// Shared-memory working set of one Shinv: two iterate buffers, x, and the product scratch.
struct ShinvBufs {
    limb *WA, *WB;   // iterates w (ping-pong); capacity >= round_up(H + 6, 8) limbs each
    limb *X;         // |B^h'' - v'w|; capacity >= k + 48 limbs
    limb *P;         // product; capacity >= h + 40 limbs
    MulScratch ms;
};

// Block sizes whose kernels carry the tensor-core multiplier (mp_mma.cuh); the others never see an MmaCtx.
template <int T>
struct MmaEnabled { static constexpr bool value = (T == 512 || T == 256 || T == 128); };
// (128-thread blocks, 2^16 bits: no gain while the MMAs were issued by a single thread of a diverged warp; +23 % at
// config 2 with the warp-issued loop of mp_mma.cuh.  The latency kernel of small batches keeps the IMAD path:
// its instantiation carries no tensor-core code: MMA template flag of shinv_block / refine_step / try_mma_range.)

// Range product on the tensor core when the plan says it wins, else -1 (caller runs the IMAD path).
// P[i] = limb 32*dlo + i.
template <int T, bool MMA = MmaEnabled<T>::value>
__device__ __forceinline__ int try_mma_range(const MmaRef &mma, const limb *A, int na, const limb *Bp, int nb, int dlo, int dhi,
                                             limb *P, limb *HI, Blk &blk)
{
    if constexpr (MMA) {
        bool swap;
        if (mma_plan<T>(mma, na, nb, dlo, dhi, swap))
            return swap ? mma_mul_range<T>(*mma.cx, Bp, nb, A, na, dlo, dhi, P, HI, blk)
                        : mma_mul_range<T>(*mma.cx, A, na, Bp, nb, dlo, dhi, P, HI, blk);
    }
    return -1;
}

// One Refine iteration (Alg. 1 lines 19-25 with Step and PowDiff inlined) run by a group of TT threads:
// the whole block (TT = T) or, for the early iterations whose operands are a few tiles long, warp 0 alone
// (TT = 32: warp-level barriers only; the other warps wait at the block barrier that ends the narrow phase
// and leave their issue slots to the other blocks of the SM).
template <int TT, bool MMA = false, bool CL = false>
__device__ __forceinline__ void refine_step(const limb *V, int k, int H, int it, int l, int wlen, limb *Wc, limb *Wn,
                                            limb *X, limb *P, const MulScratch &ms, Blk &blk, bool clip, const MmaRef &mma)
{
    const int g = 2;
    const int m = min(H + 1 - l, l);
    int s = max(0, k - 2 * l + 1 - g);
    s &= ~3;                                               // keep the divisor prefix 16-byte aligned
    const limb *Vp = V + s;                                // shift_{-s}(v)
    const int pv = k + 1 - s;
    const int hp = k + l + m - s + g;                      // h' of Step
    const int hpp = hp - m;                                // h'' of PowDiff
    const int pw = top_prec(Wc, min(wlen, l + g + 2));
    const int d = hp - 2 * m;                              // limbs of w*x that shift_{2m-h'} drops

    // ---- PowDiff (Alg. 2): (sign, x) = (B^h'' >= v'w, |B^h'' - v'w|) -------
    const int L = pv + pw - (l - g) + 1;
    bool positive;
    int xl;                                                // limbs of x (upper bound)
    int c = 0;                                             // X holds x / B^c
    if (L >= hpp) {
        // no room to truncate: full product and a comparison with B^h''
        mul_full<TT, CL>(Vp, pv, Wc, pw, P, ms, blk);
        const int pl = round_up(pv, TILE) + round_up(pw, TILE);
        positive = !any_nonzero<TT>(P, hpp, pl);            // v'w < B^h''  (v'w != B^h'' here or x = 0)
        if (positive) {
            xl = hpp;                                      // x = B^h'' - p = ~p + 1 over h'' limbs
            lin_addsub<TT, false>(X, round_up(xl, TILE), NotView{P, xl, pl}, ZeroView{}, 1u, blk);
            // p = 0 cannot happen (v', w > 0); p = B^h'' exactly falls in the other branch
        } else {
            xl = pv + pw;                                  // x = p - B^h''
            lin_addsub<TT, true>(X, round_up(xl, TILE), LimbView{P, pl, 0}, UnitView{hpp}, 0u, blk);
        }
    } else {
        // c_x: x must be right down to limb c_x for w*x to be right down to limb d + 1
        const int cx = d + 1 - pw;
        const int Klo2 = (clip && cx >= 25) ? (cx - 9) / 8 - 1 : 0;
        if (Klo2 <= 0) {
            // close product: only the L low limbs of v'w (MULTMOD)
            mul_low<TT, CL>(Vp, pv, Wc, pw, L, P, ms, blk);
            positive = P[L - 1] != 0u;                     // top limb set: v'w just below B^h''
            xl = L;
            if (positive)
                lin_addsub<TT, false>(X, round_up(xl, TILE), NotView{P, xl, xl}, ZeroView{}, 1u, blk);
            else
                lin_copy<TT>(X, round_up(xl, TILE), P, xl, 0);  // v'w = B^h'' + P, P small (or P = 0)
        } else {
            // clipped close product: limbs [c, L) of v'w only; X holds x / B^c (low limbs taken as 0)
            count(CNT_CLIPPED_STEPS);
            const int dlo = (cx - 1) / 32;               // tensor-core form: blocks of 32 limbs, E < B^(32 dlo + 1)
            if (try_mma_range<TT, MMA>(mma, Vp, pv, Wc, pw, dlo, (L + 31) / 32, P, ms.HI, blk) >= 0) {
                c = 32 * dlo;
                count(CNT_MMA_PRODUCTS);
            } else {
                c = TILE * Klo2;
                mul_range<TT, CL>(Vp, pv, Wc, pw, Klo2, (L + TILE - 1) / TILE, P, ms, blk);
            }
            xl = L - c;
            positive = P[xl - 1] != 0u;
            for (int i = threadIdx.x; i < round_up(xl, TILE); i += TT)
                X[i] = (i < xl) ? (positive ? ~P[i] : P[i]) : 0u;
            grp_sync<TT>();
        }
    }
    if (!positive) count(CNT_SIGN_NEG);
    xl = top_prec(X, xl);

    // ---- Step (Alg. 1 lines 29-37): w <- shift_m(w) +- shift_{2m-h'}(w x), then shift_{-1} ----
    const int nlen = round_up(l + m + g + 2, TILE);
    if (xl == 0) {
        lin_copy<TT>(Wn, nlen, Wc, wlen, 1 - m);
    } else {
        // w*x / B^(d+1): the shift_{2m-h'} of Step and the shift_{-1} of Refine drop d + 1 limbs
        const int dd = d + 1 - c;
        const int Klo1 = (clip && dd >= 17) ? (dd - 9) / TILE : 0;
        int tl = -1, off = 0;
        bool exact = (Klo1 == 0 && c == 0);
        if (clip && dd >= 33) {
            const int dlo = (dd - 1) / 32;
            tl = try_mma_range<TT, MMA>(mma, Wc, pw, X, xl, dlo, 1 << 20, P, ms.HI, blk);
            if (tl >= 0) { off = dd - 32 * dlo; exact = false; count(CNT_MMA_PRODUCTS); }
        }
        if (tl >= 0) {
        } else if (Klo1 == 0) {
            mul_full<TT, CL>(Wc, pw, X, xl, P, ms, blk);
            tl = round_up(pw, TILE) + round_up(xl, TILE);
            off = dd;
        } else {
            tl = mul_range<TT, CL>(Wc, pw, X, xl, Klo1, 1 << 20, P, ms, blk);
            off = dd - TILE * Klo1;
        }
        if (positive) {
            lin_addsub<TT, false>(Wn, nlen, LimbView{Wc, wlen, 1 - m}, LimbView{P, tl, off}, 0u, blk);
        } else {
            // floor of a negative: borrow one when any dropped limb of w*x is non-zero (exact path only;
            // a clipped step is off by less than a guard-limb unit either way)
            uint32_t bin = 0u;
            if (exact) bin = any_nonzero<TT>(P, 0, min(dd, tl)) ? 1u : 0u;
            lin_addsub<TT, true>(Wn, nlen, LimbView{Wc, wlen, 1 - m}, LimbView{P, tl, off}, bin, blk);
        }
    }
}

// ---------------------------------------------------------------------------------------
// Seed of Refine with 17 correct digits, computed by one warp (clipped variant only).
//
// Refine's iterate with l correct digits is w ~ B^(k+l+g) / v (PAPER.md:92 l.15-25).  The first four
// iterations (l = 2, 3, 5, 9 -> 17) multiply numbers of 4 to 40 limbs and cost ~10 000 cycles each in
// block-wide barriers and scans; they are replaced by the exact quotient
//      w = floor(B^38 / D),   D = floor(v / B^(k-19))   (the top 20 limbs of v; v * B^(19-k) when k < 19),
// which satisfies  B^(k+19)/v - 1 < w <= B^(k+19)/v + 1  because D <= v/B^(k-19) < D + 1 and D >= B^19:
// a better iterate than the one Refine would hold at l = 17 (whose error is several units of a guard limb).
// The quotient comes from schoolbook long division (Knuth, TAOCP vol. 2, 4.3.1 Algorithm D) with one limb
// per lane: lane j holds limb j of the normalised divisor and of the 21-limb remainder window; a quotient
// digit is a 2-by-1 division by the top divisor limb through its precomputed reciprocal (Moeller and
// Granlund, "Improved division by invariant integers", Alg. 4), Knuth's two-digit test, a multiply-subtract
// whose carries and borrows are resolved by two ballots and an integer add, and a rare add-back.
// ---------------------------------------------------------------------------------------
constexpr int SEED_L = 17;                 // correct digits of the seed
constexpr int SEED_ITERS = 4;              // Refine iterations it replaces (l = 2 -> 3 -> 5 -> 9 -> 17)
constexpr int SEED_LIMBS = SEED_L + 3;     // limbs of D and of the quotient (l + g + 1)

// carries into each lane from generate / propagate masks: bit j of the result = carry into lane j
__device__ __forceinline__ uint32_t lane_carries(uint32_t G, uint32_t P)
{
    return ((G | P) + G) ^ P;              // G and P are disjoint
}

// Runs on one full warp.  W receives SEED_LIMBS limbs and zeros up to 24 (the wlen of iteration 4).
__device__ __forceinline__ void warp_seed(const limb *V, int k, limb *W)
{
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int ND = SEED_LIMBS;
    const int lane = threadIdx.x & 31;
    const int idx = k - (ND - 1) + lane;
    const uint32_t dj = (lane < ND && idx >= 0) ? V[idx] : 0u;
    // D1: normalise so that the top limb has its high bit set (the dividend B^38 shifts with it)
    const int sh = __clz(__shfl_sync(FULL, dj, ND - 1));
    uint32_t dl = __shfl_up_sync(FULL, dj, 1);
    if (lane == 0) dl = 0u;
    const uint32_t d = (lane < ND) ? __funnelshift_l(dl, dj, sh) : 0u;
    const uint32_t d1 = __shfl_sync(FULL, d, ND - 1), d0 = __shfl_sync(FULL, d, ND - 2);
    const uint32_t dinv = (uint32_t)(0xffffffffffffffffull / d1);      // floor((B^2 - 1) / d1) - B
    // remainder window: lane j holds limb i + j of the running remainder at quotient digit i; digit ND-1 first,
    // where the only non-zero limb of B^38 << sh is limb 38 = lane 19
    uint32_t r = (lane == ND - 1) ? (1u << sh) : 0u;
    uint32_t qd = 0u;
    uint32_t addbacks = 0u;
#pragma unroll 1
    for (int i = ND - 1; i >= 0; --i) {
        const uint32_t r2 = __shfl_sync(FULL, r, ND), r1 = __shfl_sync(FULL, r, ND - 1), r0 = __shfl_sync(FULL, r, ND - 2);
        // D3: qhat = min(floor((r2 B + r1) / d1), B - 1), rhat the remainder; then the two-digit test
        uint32_t qh, rh;
        bool test = true;
        if (r2 >= d1) {                                       // r2 = d1 (r2 > d1 cannot happen)
            qh = 0xffffffffu;
            rh = r1 + d1;
            test = rh >= d1;                                  // no overflow: rhat < B
        } else {
            const uint64_t pq = (uint64_t)dinv * r2 + (((uint64_t)r2 << 32) | r1);
            uint32_t q1 = (uint32_t)(pq >> 32) + 1u;
            const uint32_t q0 = (uint32_t)pq;
            rh = r1 - q1 * d1;
            if (rh > q0) { q1 -= 1u; rh += d1; }
            if (rh >= d1) { q1 += 1u; rh -= d1; }
            qh = q1;
        }
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            if (test && (uint64_t)qh * d0 > (((uint64_t)rh << 32) | r0)) {
                qh -= 1u;
                const uint32_t nr = rh + d1;
                test = nr >= rh;                              // stop once rhat >= B
                rh = nr;
            }
        }
        // D4: r -= qhat * D over the 21 lanes
        const uint64_t p = (uint64_t)qh * d;
        uint32_t hp = __shfl_up_sync(FULL, (uint32_t)(p >> 32), 1);
        if (lane == 0) hp = 0u;
        uint32_t t = (uint32_t)p + hp;
        uint32_t G = __ballot_sync(FULL, t < hp), P = __ballot_sync(FULL, t == 0xffffffffu);
        t += (lane_carries(G, P) >> lane) & 1u;
        uint32_t s = r - t;
        G = __ballot_sync(FULL, r < t);
        P = __ballot_sync(FULL, r == t);
        uint32_t bw = lane_carries(G, P);
        s -= (bw >> lane) & 1u;
        // D5/D6: negative remainder (borrow out of lane ND): add the divisor back (probability ~2/B per digit)
        bool neg = ((bw >> (ND + 1)) & 1u) != 0u;
        while (neg) {
            qh -= 1u;
            addbacks += 1u;
            const uint32_t s2 = s + d;
            G = __ballot_sync(FULL, s2 < s);
            P = __ballot_sync(FULL, s2 == 0xffffffffu);
            const uint32_t cw = lane_carries(G, P);
            s = s2 + ((cw >> lane) & 1u);
            neg = ((cw >> (ND + 1)) & 1u) == 0u;              // the carry out of lane ND cancels the borrow
        }
        if (lane == i) qd = qh;
        // D7: next digit: the window moves one limb down (the dividend's lower limbs are all zero)
        r = __shfl_up_sync(FULL, s, 1);
        if (lane == 0) r = 0u;
    }
    if (lane < 24) W[lane] = (lane < ND) ? qd : 0u;
    if (lane == 0 && addbacks) atomicAdd(&g_counters[CNT_SEED_ADDBACK], (unsigned long long)addbacks);
}

// Refine's trip count for H = max(h - k, 2) (PAPER.md:92 l.18-19; "+1" for the clipped variant, see shinv_block).
__device__ __forceinline__ int refine_iters(int H, bool clip)
{
    return ((H - 1 > 1) ? (32 - __clz(H - 2)) : 0) + (clip ? 1 : 2);
}

// ---------------------------------------------------------------------------------------
// Head of Refine (clipped variant, throughput batches).  The iterations up to l = HEAD_L handle operands of
// at most ~270 limbs: a few thousand limb products each, but thousands of cycles of dependent latency.  When
// the blocks of a batch run them inside the division kernel, all resident blocks of an SM sit in these phases
// at the same time (same sizes, same schedule) and the multiplier pipe idles.  A batch therefore runs them in a
// kernel of its own, one WARP per divisor and up to 16 divisors per SM, which leaves the seed and the iterate
// after the head (at most WMID_STRIDE limbs) in a workspace row; the division kernel starts Refine from there.
// Both kernels derive the split from H alone (head_plan), so no flag travels with the row.
// ---------------------------------------------------------------------------------------
constexpr int HEAD_L = 129;                // the head runs the iterations that start with l <= HEAD_L ...
constexpr int WMID_STRIDE = 272;           // ... and leaves at most 2 HEAD_L + g + 2 limbs, rounded up to tiles
struct HeadPlan { int it_end, l_end, wlen_end; };   // it_end = 0: no head (Refine starts in the division kernel)

__device__ __forceinline__ HeadPlan head_plan(int H, int iters)
{
    HeadPlan p{0, 0, 0};
    if (H < SEED_L) return p;
    int l = SEED_L, it = SEED_ITERS, wlen = 24;
    while (l <= HEAD_L && it + 2 < iters) {                   // the last two iterations stay with the block
        const int m = min(H + 1 - l, l);
        wlen = round_up(l + m + 2 + 2, TILE);
        l += m - 1;
        ++it;
    }
    if (it == SEED_ITERS) return p;
    p.it_end = it; p.l_end = l; p.wlen_end = wlen;
    return p;
}

// w = Shinv(v, h) for B <= v (k = prec(v) - 1 >= 1), v zero padded to whole tiles above limb k.
// The result lands in bufs.WA, zero padded to whole tiles; returns an upper bound of its limb count.
template <int T, bool MMA = false, bool CL = false>
__device__ __forceinline__ int shinv_block(const limb *V, int k, int h, const ShinvBufs &bufs, Blk &blk,
                                           bool clip, const MmaRef &mma = MmaRef{nullptr, 0, 0}, int narrow_l = 0, bool seed = true,
                                           const limb *wmid = nullptr)
{
    limb *WA = bufs.WA, *WB = bufs.WB, *X = bufs.X, *P = bufs.P;
    const MulScratch &ms = bufs.ms;
    const int g = 2;

    // ---- special cases (Alg. 1 lines 5-10) -------------------------------------
    const limb vtop = V[k];
    // the limbs below the top one only matter when the top limb is 1 (v = B^k?) or 2^31 (2v > B^h?)
    const bool low_nz = (vtop == 1u || vtop == 0x80000000u) ? any_nonzero<T>(V, 0, k) : true;
    const bool pow_b = (vtop == 1u) && !low_nz;               // v = B^k
    int special = -1;                                          // value of a one-limb result
    if (k > h || (k == h && !pow_b)) special = 0;              // v > B^h
    else if (!pow_b && k == h - 1 &&
             (vtop > 0x80000000u || (vtop == 0x80000000u && low_nz))) special = 1;   // 2v > B^h
    if (special >= 0) {
        for (int i = threadIdx.x; i < TILE; i += T) WA[i] = (i == 0) ? (limb)special : 0u;
        __syncthreads();
        return 1;
    }
    if (pow_b) {                                               // v = B^k  ->  B^(h-k)
        count(CNT_POW_B);
        const int len = round_up(h - k + 1, TILE);
        for (int i = threadIdx.x; i < len; i += T) WA[i] = (i == h - k) ? 1u : 0u;
        __syncthreads();
        return h - k + 1;
    }

    // ---- initial approximation (Alg. 1 lines 11-13): w = B^3 quo (v[k-1] + v[k] B), l = 2 ----
    const int H = max(h - k, 2);
    // printed bound: ceil(log2(H-1)) + 2 (PAPER.md:92 l.18-19).  The clipped variant runs one trailing iteration
    // fewer (SURVEY G4 "+1"): the last doubling step already reaches all H digits, one repeat at full size
    // repairs its truncation errors, and whatever is left is absorbed by the bounded correction loops of Div
    // (lambda stayed in {-1,0,1} on 60 000 random and directed cases of the big-integer model; a plain
    // `while l < H`, i.e. "+0", is wrong).
    const int iters = refine_iters(H, clip);
    limb *Wc = ((iters + 1) & 1) ? WB : WA;                    // so that write number iters+1 hits WA
    limb *Wn = (Wc == WA) ? WB : WA;
    int l = 2;
    int wlen = TILE;                                           // valid (zero padded) words of Wc
    int it0 = 0;
    const HeadPlan hp = (clip && wmid) ? head_plan(H, iters) : HeadPlan{0, 0, 0};
    if (hp.it_end) {
        // the head kernel left the iterate after it_end iterations in the workspace row
        // The division kernel is launched with programmatic stream serialisation behind the head kernel: its blocks
        // start while the head still runs (their set-up, loads and precisions need nothing from it) and wait HERE for
        // the head grid to have completed and flushed its rows.
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (hp.it_end & 1) { limb *t = Wc; Wc = Wn; Wn = t; }
        for (int i = threadIdx.x; i < hp.wlen_end; i += T) Wc[i] = __ldcg(wmid + i);
        l = hp.l_end;
        wlen = hp.wlen_end;
        it0 = hp.it_end;
    } else if (clip && seed && H >= SEED_L) {
        // the first four iterations would all double l (m = l up to l = 9 needs H + 1 - 9 >= 9): start from the
        // 17-digit seed instead; Wc is the buffer iteration 4 reads (an even number of swaps away)
        if (threadIdx.x < 32) warp_seed(V, k, Wc);
        count(CNT_SEEDS);
        l = SEED_L;
        wlen = 24;
        it0 = SEED_ITERS;
    } else if (threadIdx.x == 0) {
        const unsigned long long V2 = ((unsigned long long)V[k] << 32) | V[k - 1];
        const unsigned __int128 w0 = (((unsigned __int128)1) << 96) / V2;
        Wc[0] = 0u; Wc[1] = 0u;                                // shift_g(w), g = 2 (Alg. 1 line 17)
        Wc[2] = (limb)w0; Wc[3] = (limb)(w0 >> 32); Wc[4] = (limb)(w0 >> 64);
        Wc[5] = 0u; Wc[6] = 0u; Wc[7] = 0u;
    }
    __syncthreads();

    // ---- Refine (Alg. 1 lines 15-28) ------------------------------------------------------------
    // The early iterations (l <= NARROW_L: operands of at most ~40 x 70 limbs) run on warp 0 alone.
    // (narrow_l = 33 when the grid has more blocks than SMs: a lone block per SM is latency bound and keeps all
    // its threads; 0 disables)
    bool narrow_open = false;
    for (int it = it0; it < iters; ++it) {
        const int m = min(H + 1 - l, l);
        const int nlen = round_up(l + m + g + 2, TILE);
        if (T > 32 && l <= narrow_l && it + 2 < iters) {
            narrow_open = true;
            if (threadIdx.x < 32) refine_step<32>(V, k, H, it, l, wlen, Wc, Wn, X, P, ms, blk, clip, MmaRef{nullptr, 0, 0});
        } else {
            if (narrow_open) {                                 // leave the narrow phase: one block barrier,
                narrow_open = false;                           // and a common collective parity again
                __syncthreads();
                blk.parity = 0;
            }
            refine_step<T, MMA, CL>(V, k, H, it, l, wlen, Wc, Wn, X, P, ms, blk, clip, mma);
        }
        l = l + m - 1;
        wlen = nlen;
        limb *t = Wc; Wc = Wn; Wn = t;
    }

    // ---- final shift_{-g - (H - (h-k))} (Alg. 1 lines 26-27) -------------------------------------
    const int sh = g + (H - (h - k));
    const int rlen = round_up(h - k + 2, TILE);
    lin_copy<T>(Wn, rlen, Wc, wlen, sh);                       // Wn == WA by construction
    return h - k + 1;
}

// One divisor's head on one warp (blockDim.x == 32): seed, then the iterations head_plan assigns to it; the
// iterate goes to wrow (hp.wlen_end limbs).  smem: HEAD_SMEM_WORDS words, 16-byte aligned.  vg is the divisor's
// row in global memory; only its top 2 HEAD_L + 4 limbs are read.
constexpr int HEAD_V = 288, HEAD_W = 272, HEAD_X = 288, HEAD_P = 448, HEAD_OV = 64;
constexpr int HEAD_SMEM_WORDS = HEAD_V + 2 * HEAD_W + HEAD_X + 2 * HEAD_P + 2 * HEAD_OV + (int)(sizeof(BlkScratch) / 4);

__device__ __forceinline__ void shinv_head_warp(const limb *__restrict__ vg, int k, int h, uint32_t *smem,
                                                limb *__restrict__ wrow)
{
    const int lane = threadIdx.x;
    const int H = max(h - k, 2);
    const HeadPlan hp = head_plan(H, refine_iters(H, true));
    if (!hp.it_end) return;
    limb *Vs = smem, *Wc = Vs + HEAD_V, *Wn = Wc + HEAD_W, *X = Wn + HEAD_W, *P = X + HEAD_X;
    MulScratch ms;
    ms.HI = P + HEAD_P;
    ms.OV = ms.HI + HEAD_P;
    ms.C3 = ms.OV + HEAD_OV;
    ms.ST = nullptr;
    ms.stage_cap = 0;
    Blk blk{reinterpret_cast<BlkScratch *>(ms.C3 + HEAD_OV), 0u, 0u};
    // divisor prefix: limbs s_lo..k, s_lo the s of an iteration at l = HEAD_L (no head iteration reaches lower),
    // zeros above limb k
    const int s_lo = max(0, k - 2 * HEAD_L + 1 - 2) & ~3;
    const int cnt = k + 1 - s_lo;
    for (int i = lane; i < HEAD_V; i += 32) Vs[i] = (i < cnt) ? __ldg(vg + s_lo + i) : 0u;
    __syncwarp();
    const limb *V = Vs - s_lo;                                 // V[i] = limb i of v for i >= s_lo
    warp_seed(V, k, Wc);
    count(CNT_SEEDS);
    __syncwarp();
    int l = SEED_L, wlen = 24;
    for (int it = SEED_ITERS; it < hp.it_end; ++it) {
        const int m = min(H + 1 - l, l);
        const int nlen = round_up(l + m + 2 + 2, TILE);
        refine_step<32>(V, k, H, it, l, wlen, Wc, Wn, X, P, ms, blk, true, MmaRef{nullptr, 0, 0});
        l = l + m - 1;
        wlen = nlen;
        limb *t = Wc; Wc = Wn; Wn = t;
    }
    for (int i = lane; i < hp.wlen_end; i += 32) wrow[i] = Wc[i];
    count_tiles(blk);
}

}  // namespace mpd
