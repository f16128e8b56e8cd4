// mpdiv_batch / shinv_batch kernels and the rest of the C ABI (included by mpdiv.cu).

// ---------------------------------------------------------------------------------------
// shared-memory arena of one division (word offsets).  Phases reuse the same words:
//   Refine   : V | WB (=U area) | WA | X  P  HI  OV  C3            (u is not resident)
//   quotient : V | U            | WA (= shinv, then q) | P  HI  OV  C3   (P up to 2M+2 limbs)
// ---------------------------------------------------------------------------------------
struct DivLayout {
    int v_off, u_off, wa_off, big_off, sc_off, total_words;
    int mma_off;      // word offset (1024-byte aligned) of the tensor-core scratch (rows | ring), or -1
    int bar_off;      // word offset of the engine's mbarriers (MMA_BAR_BYTES that no buffer of either layout overlaps)
    int mma_rows;     // rows of 128 bytes available for the row operand
    int mma_cols;     // TMEM columns to allocate
    int x_words;      // Refine: X at big_off, P behind it
    int p_words_r;    // Refine: capacity of P and of HI
    int p_words_q;    // quotient phase: capacity of P and of HI
    int hcap;         // the layout holds instances with H = max(h - k, 2) <= hcap
    int qb_off;       // chunked form (mpdiv_kernel<.., BIG>): the quotient chunk's own buffer; otherwise = wa_off
    int stage_off;    // cluster form (mpdiv_kernel<.., CL>): two staging sets of stage_set_words(stage_cap) words, or -1
    int stage_cap;
};

// M: limbs of the dividend side (u stride, or h for shinv_batch); n: divisor stride;
// with_quotient: reserve the product scratch of u * shinv and v * q; clip: MPDIV_VARIANT_CLIPPED, whose
// products only store the limbs they keep (about M/2 in Refine, M in the quotient phase).
// hcap: 0 = any instance of these strides (H up to M: a short divisor has a long inverse and a long quotient);
// otherwise the COMPACT layout for instances with H <= hcap: the iterate / quotient buffer WA and the quotient-phase
// product shrink to what such instances need -- at the configs' shape (H = M/2 + 1) that is 8 KB of 40 at
// 2^16 bits, the room the tensor-core scratch needs to keep four blocks on an SM.  V, U and the block scratch sit
// at the same offsets in both layouts, so the operands are loaded before the layout of the instance is known.
static DivLayout div_layout(int M, int n, bool with_quotient, bool clip, int hcap = 0)
{
    DivLayout L;
    const int Mp = round_up(M, TILE);
    const int np = round_up(n, TILE);
    const int hc = (hcap > 0 && hcap < Mp) ? round_up(hcap, TILE) : Mp;
    if (clip) {
        L.x_words = round_up(Mp / 2 + 96, TILE);
        L.p_words_r = round_up(Mp / 2 + 160, TILE);
        L.p_words_q = with_quotient ? (hc > np ? hc : np) + 104 : 0;
    } else {
        L.x_words = np + 48;
        L.p_words_r = Mp + 48;
        L.p_words_q = with_quotient ? 2 * Mp + 32 : 0;
    }
    const int ovr = round_up(L.p_words_r / TILE, 4), ovq = round_up(L.p_words_q / TILE, 4);
    const int big_r = L.x_words + 2 * L.p_words_r + 2 * ovr;
    const int big_q = 2 * L.p_words_q + 2 * ovq;
    int o = 0;
    L.sc_off = o; o += (int)(sizeof(BlkScratch) / 4);
    L.v_off = o; o += np + 16;
    L.u_off = o; o += Mp + 16;
    L.wa_off = o; o += hc + 24;
    L.big_off = o; o += (big_r > big_q ? big_r : big_q);
    L.total_words = o;
    L.mma_off = -1;
    L.bar_off = -1;
    L.mma_rows = 0;
    L.mma_cols = 0;
    L.hcap = hc;
    L.qb_off = L.wa_off;
    L.stage_off = -1;
    L.stage_cap = 0;
    return L;
}

// Adds the staging sets of the cluster form (mp_mul.cuh) behind layout L; returns the bytes.
static size_t div_layout_add_stage(DivLayout &L)
{
    const int pw = L.p_words_r > L.p_words_q ? L.p_words_r : L.p_words_q;
    L.stage_cap = round_up(pw + 2 * TILE, 32);
    L.stage_off = round_up(L.total_words, 4);
    L.total_words = L.stage_off + 2 * stage_set_words(L.stage_cap);
    return (size_t)L.total_words * 4;
}

// H up to which an instance takes the compact layout: the configs' shape H = M/2 + 1 with room to spare.
static int compact_hcap(int M) { return round_up(M, TILE) / 2 + 40; }

// Places the scratch of the tensor-core multiplier (mp_mma.cuh) behind layout Lx: the rows of the row operand (output
// blocks + steps rows of 128 bytes) and the ring of the Toeplitz operand.  Returns the word offset where the scratch
// ends, or -1 (and leaves Lx without an engine) when that would pass limit_words.  threads = block size.
static int div_layout_place_mma(DivLayout &Lx, int M, int limit_words, int threads)
{
    const int blocks = (M / 2 + 1 + 9 + 31) / 32 + 2;             // output blocks of u * shinv at n = M/2
    const int nn = (blocks + 15) & ~15;
    const int want = 2 * nn;                                      // one accumulator set per issuing warp (mp_mma.cuh)
    const int cols = want <= 32 ? 32 : want <= 64 ? 64 : want <= 128 ? 128 : want <= 256 ? 256 : 512;
    const int rows = round_up(nn + blocks, 8);
    const int off = round_up(Lx.total_words, 256);
    const int end = off + mma_scratch_bytes(rows, threads) / 4;
    if (end > limit_words) return -1;
    Lx.mma_off = off;
    Lx.mma_rows = rows;
    Lx.mma_cols = cols;
    return end;
}

// The two layouts of a division kernel that carries the engine, and the bytes to allocate.
//   Lc  compact layout (instances with H <= Lc.hcap) + scratch: the common case, and the fastest arrangement
//   Lf  full layout (any instance); it gets a scratch of its own behind it when that still keeps per_sm blocks on an
//       SM (2^17 bits and up), otherwise its instances run without the engine and may overrun Lc's scratch, which every
//       product rewrites.  The mbarriers sit behind everything (Lc.bar_off == Lf.bar_off).
static size_t div_layouts_with_mma(DivLayout &Lf, DivLayout &Lc, int u_limbs, int v_limbs, bool clip, int threads, int per_sm,
                                   int max_smem)
{
    Lf = div_layout(u_limbs + 1, v_limbs, true, clip);
    Lc = div_layout(u_limbs + 1, v_limbs, true, clip, compact_hcap(u_limbs + 1));
    const int bar_words = MMA_BAR_BYTES / 4;
    const int budget = (max_smem + 1024) / per_sm - 1024;        // shared memory of an SM = the per-block maximum + 1 KB
    int limit = (budget < max_smem ? budget : max_smem) / 4 - bar_words;
    int end_c = div_layout_place_mma(Lc, u_limbs, limit, threads);
    if (end_c < 0) {                                             // give up occupancy before giving up the engine
        limit = max_smem / 4 - bar_words;
        end_c = div_layout_place_mma(Lc, u_limbs, limit, threads);
    }
    int end = Lf.total_words;
    if (end_c >= 0) {
        if (end_c > end) end = end_c;
        const int end_f = div_layout_place_mma(Lf, u_limbs, limit, threads);
        if (end_f > end) end = end_f;
        end = round_up(end, 4);
        Lc.bar_off = Lf.bar_off = end;
        end += bar_words;
    }
    Lc.total_words = Lf.total_words = end;
    return (size_t)end * 4;
}

// Layout of the CHUNKED division (mpdiv_kernel<.., BIG>; dividends above MPDIV_MAX_OPERAND_LIMBS limbs, whose rows do not
// fit beside the divisor and the product scratch): the dividend is not resident.  The quotient is produced t limbs at a
// time from a WINDOW of at most k + 1 + t limbs (the running remainder above the next t limbs of u, streamed from HBM),
// with one shifted inverse of t + 2 limbs for all windows.  V | window (the U area; Refine's second iterate buffer) |
// WA (iterates, shinv) | QB (quotient chunk) | product scratch | tensor-core scratch | mbarriers.  Sized like a regular
// division of a (v_limbs + 1 + t)-limb dividend whose inverse has at most t + 2 limbs.  Returns the bytes, 0 when t does
// not fit max_smem.
static size_t div_layout_big(DivLayout &L, int v_limbs, int t, int threads, int max_smem)
{
    const int np = round_up(v_limbs, TILE);
    L = div_layout(np + 1 + t + 1, v_limbs, true, true, t + 40);
    L.qb_off = L.total_words;
    L.total_words += round_up(t + 32, TILE);
    const int bar_words = MMA_BAR_BYTES / 4;
    // tensor-core scratch: v * q_chunk needs ceil((k + 3) / 32) output blocks (one accumulator set when that exceeds 256
    // columns) and one row per block and per 128-byte chunk of the quotient chunk
    const int blocks = (np + 8 + 31) / 32 + 1;
    const int nn = (blocks + 15) & ~15;
    const int want = nn > 256 ? nn : 2 * nn;
    const int cols = want <= 32 ? 32 : want <= 64 ? 64 : want <= 128 ? 128 : want <= 256 ? 256 : 512;
    const int rows = round_up(nn + (t + 2 + 31) / 32 + 2, 8);
    const int off = round_up(L.total_words, 256);
    const int end = off + mma_scratch_bytes(rows, threads) / 4;
    if (nn <= 512 && (end + bar_words) * 4 <= max_smem) {
        L.mma_off = off;
        L.mma_rows = rows;
        L.mma_cols = cols;
        L.bar_off = end;
        L.total_words = end + bar_words;
    }
    return (size_t)L.total_words * 4 <= (size_t)max_smem ? (size_t)L.total_words * 4 : 0;
}

__device__ __forceinline__ ShinvBufs refine_bufs(uint32_t *smem, const DivLayout &L)
{
    ShinvBufs b;
    b.WA = smem + L.wa_off;
    b.WB = smem + L.u_off;
    b.X = smem + L.big_off;
    b.P = b.X + L.x_words;
    const int ov = round_up(L.p_words_r / TILE, 4);
    b.ms.HI = b.P + L.p_words_r;
    b.ms.OV = b.ms.HI + L.p_words_r;
    b.ms.C3 = b.ms.OV + ov;
    b.ms.ST = L.stage_off >= 0 ? smem + L.stage_off : nullptr;
    b.ms.stage_cap = L.stage_cap;
    return b;
}

// ---------------------------------------------------------------------------------------
// mpdiv_seed_batch kernel: the 17-digit seed of Refine on its own (one warp per divisor, v read from HBM)
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
seed_kernel(const limb *__restrict__ v, int v_limbs, limb *__restrict__ w, int batch)
{
    const int inst = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (inst >= batch) return;
    const limb *V = v + (size_t)inst * v_limbs;
    int top = -1;                                             // index of the top non-zero limb
    for (int i0 = 0; i0 < v_limbs; i0 += 32) {
        const int i = i0 + lane;
        const uint32_t nz = __ballot_sync(0xffffffffu, i < v_limbs && V[i] != 0u);
        if (nz) top = i0 + 31 - __clz(nz);
    }
    limb *W = w + (size_t)inst * 24;
    if (top < 1) { if (lane < 24) W[lane] = 0u; return; }
    warp_seed(V, top, W);
}

// ---------------------------------------------------------------------------------------
// head of Refine for a whole batch: one warp (= one block) per division (mp_div.cuh "Head of Refine")
// ---------------------------------------------------------------------------------------
// significant limbs of a row in global memory (n a multiple of 4, row 16-byte aligned), scanned from the top
// 512 limbs at a time with four 16-byte loads in flight per lane
__device__ __forceinline__ int warp_prec(const limb *__restrict__ a, int n)
{
    const uint4 *a4 = reinterpret_cast<const uint4 *>(a);
    const int n4 = n >> 2, lane = (int)threadIdx.x;
    for (int hi = n4; hi > 0; hi -= 128) {
        uint4 x[4];
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const int i = hi - 128 + 32 * j + lane;          // 16-byte word index
            x[j] = (i >= 0) ? __ldg(a4 + i) : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int j = 3; j >= 0; j--) {
            const uint32_t nz = __ballot_sync(0xffffffffu, (x[j].x | x[j].y | x[j].z | x[j].w) != 0u);
            if (nz) {
                const int top_lane = 31 - __clz(nz);
                const uint32_t xx = __shfl_sync(0xffffffffu, x[j].x, top_lane), xy = __shfl_sync(0xffffffffu, x[j].y, top_lane);
                const uint32_t xz = __shfl_sync(0xffffffffu, x[j].z, top_lane), xw = __shfl_sync(0xffffffffu, x[j].w, top_lane);
                const int i = hi - 128 + 32 * j + top_lane;
                return 4 * i + (xw ? 4 : xz ? 3 : xy ? 2 : (xx ? 1 : 0));
            }
        }
    }
    return 0;
}

__global__ void __launch_bounds__(32, 16)
shinv_head_kernel(const limb *__restrict__ u, int u_limbs, const limb *__restrict__ v, int v_limbs,
                  limb *__restrict__ wmid, int batch, int tchunk)
{
    extern __shared__ __align__(1024) uint32_t smem[];
    asm volatile("griddepcontrol.launch_dependents;");     // the division kernel may start its blocks (see shinv_block)
    const int inst = blockIdx.x;
    if (inst >= batch) return;
    const int h = warp_prec(u + (size_t)inst * u_limbs, u_limbs);
    const int pv = warp_prec(v + (size_t)inst * v_limbs, v_limbs);
    if (pv < 2 || pv > h) return;                        // zero and one-limb divisors, u < v: the division kernel's own paths
    int hx = h;                                          // chunked form (tchunk > 0): the inverse all windows share
    if (tchunk > 0 && (h - (pv - 1) + tchunk - 1) / tchunk > 1) hx = pv + tchunk;
    shinv_head_warp(v + (size_t)inst * v_limbs, pv - 1, hx, smem, wmid + (size_t)inst * WMID_STRIDE);
}

// ---------------------------------------------------------------------------------------
// shinv_batch kernel
// ---------------------------------------------------------------------------------------
template <int T>
__global__ void __launch_bounds__(T, 512 / T)
shinv_kernel(const limb *__restrict__ v, int v_limbs, int h, limb *__restrict__ w, int w_limbs, int batch,
             DivLayout L, int clip, int narrow_l)
{
    extern __shared__ __align__(1024) uint32_t smem[];
    limb *V = smem + L.v_off;
    Blk blk{reinterpret_cast<BlkScratch *>(smem + L.sc_off), 0u};
    const ShinvBufs bufs = refine_bufs(smem, L);
    const int vpad = round_up(v_limbs, TILE) + 16;

    for (int inst = blockIdx.x; inst < batch; inst += gridDim.x) {
        limb *wout = w + (size_t)inst * w_limbs;
        load_number<T>(V + 4, v + (size_t)inst * v_limbs, v_limbs, vpad - 4);   // room to shift by one limb
        if (threadIdx.x < 4) V[threadIdx.x] = 0u;
        __syncthreads();
        const int pv = prec_of<T>(V + 4, v_limbs, blk);
        if (pv == 0) {                                   // v = 0: undefined
            count(CNT_V_ZERO);
            raise_status(ST_V_ZERO);
            for (int i = threadIdx.x; i < w_limbs; i += T) wout[i] = 0xffffffffu;
            __syncthreads();
            continue;
        }
        int nw;
        if (pv == 1) {                                   // one-limb divisor: Shinv(v*B, h+1)
            count(CNT_ONE_LIMB);
            if (threadIdx.x == 0) { V[1] = V[4]; V[4] = 0u; }   // v*B at the (aligned) base V
            __syncthreads();
            nw = shinv_block<T>(V, 1, h + 1, bufs, blk, clip != 0, MmaRef{nullptr, 0, 0}, narrow_l & 255, !(narrow_l & 256));
        } else {
            nw = shinv_block<T>(V + 4, pv - 1, h, bufs, blk, clip != 0, MmaRef{nullptr, 0, 0}, narrow_l & 255, !(narrow_l & 256));
        }
        store_number<T>(wout, bufs.WA, w_limbs, round_up(nw, TILE));
        __syncthreads();
    }
    count_tiles(blk);
}

// ---------------------------------------------------------------------------------------
// mpdiv_batch kernel: Alg. 3, one division per block
// ---------------------------------------------------------------------------------------
// LAT = false: 128 registers per thread, 512 threads per SM (throughput: the batch fills the SMs several
// times over).  LAT = true: up to 255 registers, for batches that leave an SM one or two blocks -- the kernel
// body keeps ~20 values live across the multiplier calls and spills them at 128 registers, which costs a
// latency-bound division 20 % (config 1: 102 -> 81 us).
// Bound of the two correction loops of Div.  Theorem 2 needs one step; the clipped variant two or three; the
// bound only has to keep |delta| * v below B^(k+2), the range of the remainder arithmetic.
constexpr int CORR_MAX = 64;

// Which division kernels carry the tensor-core engine: a latency-bound batch of 128-thread blocks is faster on the
// IMAD path alone (config 1: 68 us against 100 us per division), and without the engine's code in the kernel.
template <int T, bool LAT>
struct DivMma { static constexpr bool value = MmaEnabled<T>::value && !(LAT && T <= 128); };

// significant limbs of a row in global memory (n a multiple of 4, 16-byte aligned), by the whole block
template <int T>
__device__ __forceinline__ int global_prec(const limb *__restrict__ a, int n, Blk &blk)
{
    const uint4 *a4 = reinterpret_cast<const uint4 *>(a);
    int top = 0;
    for (int i = threadIdx.x; i < n / 4; i += T) {
        const uint4 x = __ldg(a4 + i);
        if (x.x | x.y | x.z | x.w) top = 4 * i + (x.w ? 4 : x.z ? 3 : x.y ? 2 : 1);
    }
    return block_max<T>(top, blk);
}

// dst[0..n) = (i < valid) ? src[i] : 0, both rows in global memory (n a multiple of 4, 16-byte aligned)
template <int T>
__device__ __forceinline__ void copy_row_global(limb *__restrict__ dst, const limb *__restrict__ src, int n, int valid)
{
    const uint4 *s4 = reinterpret_cast<const uint4 *>(src);
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    for (int i = threadIdx.x; i < n / 4; i += T) {
        const int b = 4 * i;
        uint4 x = (b < valid) ? __ldg(s4 + i) : make_uint4(0u, 0u, 0u, 0u);
        if (b + 1 >= valid) x.y = 0u;
        if (b + 2 >= valid) x.z = 0u;
        if (b + 3 >= valid) x.w = 0u;
        d4[i] = x;
    }
}

// MMA = this instantiation carries the engine (at most DivMma<T, LAT>; 128-thread throughput blocks also exist
// without it, for the sizes that never use it: its mere presence costs 2^15-bit batches 4 %).
// BIG = the chunked form for dividends that do not fit on chip (div_layout_big: the
// paper stops at 2^18 bits for lack of shared memory).  u stays in HBM; with D = h - k quotient limbs to produce and
// chunks of t limbs, chunk c (from the top) divides the window x_c = r_(c-1) B^t + (the next t limbs of u) by v:
// x_c < v B^t, so its quotient has t limbs, and ONE inverse w = Shinv(v, k + 1 + t) serves every window
// (q0 = floor(x w / B^(k+1+t)) is within the range of the bounded correction loops for any x < B^(k+1+t)).
// A division with D <= t is a single window with h_w = h: exactly the resident algorithm.
// CL = the cluster form (mp_mul.cuh): the CTAs of a thread-block cluster all run the division of instance
// %clusterid.x on their own copy of the state and share the tile diagonals of every product; rank 0 stores.
template <int T, bool LAT, bool MMA, bool BIG = false, bool CL = false>
__global__ void __launch_bounds__(T, LAT ? (T <= 128 ? 2 : 1) : 512 / T)
mpdiv_kernel(const limb *__restrict__ u, int u_limbs, const limb *__restrict__ v, int v_limbs,
             limb *__restrict__ q, limb *__restrict__ r, int batch, DivLayout L, DivLayout Lc, int clip, int narrow_l,
             const limb *__restrict__ wmid, int tchunk)
{
    // L: the layout for any instance of these strides; Lc: the compact layout (H <= Lc.hcap); each with the tensor-core
    // scratch behind it or mma_off < 0 (div_layouts_with_mma).  V, U and the block scratch coincide.  BIG: L == Lc.
    extern __shared__ __align__(1024) uint32_t smem[];
    limb *V = smem + L.v_off;          // divisor at V + 4 (one-limb divisors are re-based to V)
    limb *U = smem + L.u_off;          // dividend (BIG: the window) at U + 4 (same)
    limb *WA = smem + L.wa_off;        // shinv, then the quotient
    Blk blk{reinterpret_cast<BlkScratch *>(smem + L.sc_off), 0u};
    const int vpad = round_up(v_limbs, TILE) + 16, upad = round_up(u_limbs, TILE) + 16;
    static_assert(!MMA || DivMma<T, LAT>::value, "no tensor-core engine for this block size");
    static_assert(!BIG || !LAT, "the chunked form is a throughput kernel");
    static_assert(!CL || (LAT && !MMA && !BIG), "the cluster form is a latency kernel on the IMAD engine");
    uint32_t crank = 0, inst0 = blockIdx.x, inst_step = gridDim.x;
    if constexpr (CL) {
        crank = cluster_rank();
        blk.cl = crank | (cluster_size() << 8);
        asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(inst0));
        asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(inst_step));
    }
    MmaCtx mcx;
    MmaCtx *mma = nullptr;
    if constexpr (MMA) {
        if (Lc.mma_off >= 0 && clip) {
            mma_init<T>(mcx, reinterpret_cast<uint8_t *>(smem + Lc.mma_off), Lc.mma_rows,
                        reinterpret_cast<uint8_t *>(smem + Lc.bar_off), Lc.mma_cols);
            mma = &mcx;
        } else {
            mma_decline();
        }
    }
    IoBar io;
    io_init<T>(io, blk.sc);
    if constexpr (CL) cluster_sync_all();                  // every CTA of the cluster is running before any remote store

    for (int inst = (int)inst0; inst < batch; inst += (int)inst_step) {
        const limb *ug = u + (size_t)inst * u_limbs;
        const limb *vg = v + (size_t)inst * v_limbs;
        limb *qg = q + (size_t)inst * u_limbs;
        limb *rg = r + (size_t)inst * v_limbs;

        // a1/a2: load (one bulk copy per row), precisions ("h <- prec(u)")
        if (threadIdx.x < 4) { V[threadIdx.x] = 0u; U[threadIdx.x] = 0u; }
        int h;
        if constexpr (BIG) {
            load_rows<T>(io, V + 4, vg, v_limbs, vpad - 4, nullptr, nullptr, 0, 0);
            h = global_prec<T>(ug, u_limbs, blk);
        } else {
            load_rows<T>(io, V + 4, vg, v_limbs, vpad - 4, U + 4, ug, u_limbs, upad - 4, true);   // u comes back after Refine
            h = prec_of<T>(U + 4, u_limbs, blk);
        }
        const int pv = prec_of<T>(V + 4, v_limbs, blk);

        if (pv == 0) {                                     // v = 0: q = all ones, r = low limbs of u
            count(CNT_V_ZERO);
            raise_status(ST_V_ZERO);
            if (crank == 0) {
                for (int i = threadIdx.x; i < u_limbs; i += T) qg[i] = 0xffffffffu;
                if constexpr (BIG) copy_row_global<T>(rg, ug, v_limbs, min(u_limbs, v_limbs));
                else store_number<T>(rg, U + 4, v_limbs, min(u_limbs, v_limbs));
            }
            __syncthreads();
            continue;
        }
        if (pv > h) {                                      // u < v: (0, u)
            count(CNT_U_LT_V);
            if (crank == 0) {
                store_row<T>(qg, U + 4, u_limbs, 0);
                if constexpr (BIG) copy_row_global<T>(rg, ug, v_limbs, h);
                else store_number<T>(rg, U + 4, v_limbs, h);
            }
            __syncthreads();
            continue;
        }

        // one-limb divisor: divide u*B by v*B (same quotient, remainder r*B)
        const bool one_limb = (pv == 1);
        const limb *Vb = V + 4;
        limb *Ub = U + 4;
        int k = pv - 1;
        if (one_limb) {
            count(CNT_ONE_LIMB);
            if (threadIdx.x == 0) { V[1] = V[4]; V[4] = 0u; }
            __syncthreads();
            Vb = V; k = 1; h = h + 1;
        }

        // the layout of this instance: compact (and with it the tensor-core engine) when its inverse and quotient are
        // short enough, the full one otherwise
        const bool compact = BIG || (mma != nullptr && max(h - k, 2) <= Lc.hcap);
        const DivLayout &Li = compact ? Lc : L;
        const MmaRef mma_i{(mma != nullptr && Li.mma_off >= 0) ? mma : nullptr, Lc.mma_cols, Li.mma_rows};
        if (mma_i.cx) {                                    // the scratch of this instance's layout
            mcx.brows = reinterpret_cast<uint8_t *>(smem + Li.mma_off);
            mcx.ring = mcx.brows + Li.mma_rows * 128;
            mcx.brows_cap = Li.mma_rows;
        }
        const ShinvBufs rb = refine_bufs(smem, Li);
        limb *PQ = smem + Li.big_off;      // quotient-phase product scratch
        MulScratch mq;
        mq.HI = PQ + Li.p_words_q;
        mq.OV = mq.HI + Li.p_words_q;
        mq.C3 = mq.OV + round_up(Li.p_words_q / TILE, 4);
        mq.ST = rb.ms.ST;
        mq.stage_cap = rb.ms.stage_cap;

        // chunks of the quotient (BIG; otherwise one window = the whole dividend)
        const int D = h - k;                               // q < B^D
        const int nchunks = BIG ? max(1, (D + tchunk - 1) / tchunk) : 1;
        const int hx = (BIG && nchunks > 1) ? k + 1 + tchunk : h;     // every window is < B^hx

        // a3..a8: shifted inverse (U area is reused as the second iterate buffer)
        const int nw = shinv_block<T, MMA, CL>(Vb, k, hx, rb, blk, clip != 0, mma_i, narrow_l & 255, !(narrow_l & 256),
                                      (wmid && !one_limb) ? wmid + (size_t)inst * WMID_STRIDE : nullptr);
        const int psh = top_prec(WA, nw);

        const int nq = hx - k + 1;                         // q0 <= B^(hx-k): at most hx-k+1 limbs
        const int qlen = round_up(nq + 1, TILE);
        limb *Q = BIG ? smem + Li.qb_off : WA;             // resident form: WA (shinv) is dead once q0 is formed
        limb *R = PQ, *R2 = mq.HI;                         // r in place over p; HI is free after the product
        int rlen = 0;                                      // limbs of the remainder arithmetic

        for (int c = 0; c < nchunks; ++c) {
        const int lo = BIG ? (nchunks - 1 - c) * tchunk : 0;          // this chunk gives the quotient limbs from lo up
        if constexpr (BIG) {
            // the window: x_c = r_(c-1) B^t + u[lo, lo + t), or the top h - lo limbs of u for c = 0
            const int nu = (c == 0) ? h - lo : tchunk;                // limbs taken from u (h counts the B of u*B)
            const int wtop = round_up(hx + 1, TILE) + 8;
            const int n4 = one_limb ? nu : min(round_up(nu, 4), u_limbs - lo);   // limbs of u above h are zero
            if (c > 0) {
                for (int i = threadIdx.x; i < wtop - tchunk; i += T) Ub[tchunk + i] = (i <= k) ? R[i] : 0u;
            } else {
                for (int i = n4 + (int)threadIdx.x; i < wtop; i += T) Ub[i] = 0u;
            }
            if (one_limb) {                                // limb i of u*B is limb i - 1 of u
                for (int i = threadIdx.x; i < nu; i += T) {
                    const int j = lo + i - 1;
                    Ub[i] = (j >= 0 && j < u_limbs) ? __ldg(ug + j) : 0u;
                }
                __syncthreads();
            } else {
                load_rows<T>(io, Ub, ug + lo, n4, n4, nullptr, nullptr, 0, 0);
            }
            R = PQ; R2 = mq.HI;
        } else {
            // reload u; for one-limb divisors u*B, re-based to the aligned U (limb i of u at U[i+1])
            if (one_limb) {
                for (int i = threadIdx.x; i < upad; i += T)
                    U[i] = (i >= 1 && i <= u_limbs) ? __ldg(ug + i - 1) : 0u;
                Ub = U;
                __syncthreads();
            } else {
                load_rows<T>(io, U + 4, ug, u_limbs, upad - 4, nullptr, nullptr, 0, 0);
            }
        }
        int minus = 0;
        if (!clip) {
            // a9: q0 = shift_{-h}(u * shinv)  (Alg. 3 line 2); the full product, as printed
            if (psh == 0) {
                lin_zero<T>(Q, qlen);
            } else {
                mul_full<T, CL>(Ub, h, WA, psh, PQ, mq, blk);
                const int pl = round_up(h, TILE) + round_up(psh, TILE);
                lin_copy<T>(Q, qlen, PQ, pl, h);           // WA (shinv) is dead: reuse it for q
            }
            const int pq = top_prec(Q, nq);

            // a10: p = v * q0  (Alg. 3 line 3)
            rlen = round_up(h + 1, TILE);                  // p <= u + v < 2 B^h
            int pl = 0;
            if (pq > 0) {
                mul_full<T, CL>(Vb, k + 1, Q, pq, PQ, mq, blk);
                pl = round_up(k + 1, TILE) + round_up(pq, TILE);
            }

            // a11: corrections (Alg. 3 lines 4-10, Theorem 2)
            const uint32_t borrow =
                lin_addsub<T, true>(R, rlen, LimbView{Ub, h, 0}, LimbView{PQ, pl, 0}, 0u, blk);
            if (borrow) {                                  // u < v*q0: delta = -1
                minus = 1;
                lin_addsub<T, false>(R, rlen, LimbView{R, rlen, 0}, LimbView{Vb, k + 1, 0}, 0u, blk);
                lin_addsub<T, true>(Q, qlen, LimbView{Q, qlen, 0}, ZeroView{}, 1u, blk);
            }
        } else {
            // a9 clipped: only the columns >= hx - 9 of x * shinv; q0' in {q0 - 1, q0}
            if (psh == 0) {
                lin_zero<T>(Q, qlen);
            } else {
                const int dlo = (hx - 1) / 32;             // tensor-core form: E < B^(32 dlo + 1) <= B^hx
                int pl = try_mma_range<T, MMA>(mma_i, Ub, hx, WA, psh, dlo, 1 << 20, PQ, mq.HI, blk);
                if (pl >= 0) {
                    count(CNT_MMA_PRODUCTS);
                    lin_copy<T>(Q, qlen, PQ, pl, hx - 32 * dlo);
                } else {
                    const int Klo = (hx >= 17) ? (hx - 9) / TILE : 0;
                    pl = mul_range<T, CL>(Ub, hx, WA, psh, Klo, 1 << 20, PQ, mq, blk);
                    lin_copy<T>(Q, qlen, PQ, pl, hx - TILE * Klo);
                }
            }
            const int pq = top_prec(Q, nq);

            // a10 clipped: |x - v q0'| < 4v < B^(k+2), so the remainder arithmetic runs mod B^rlen
            rlen = round_up(k + 3, TILE);
            int pl = 0;
            if (pq > 0) {
                pl = try_mma_range<T, MMA>(mma_i, Vb, k + 1, Q, pq, 0, (rlen + 31) / 32, PQ, mq.HI, blk);
                if (pl >= 0) {
                    count(CNT_MMA_PRODUCTS);
                    pl = min(rlen, pl);
                } else {
                    mul_low<T, CL>(Vb, k + 1, Q, pq, rlen, PQ, mq, blk);
                    pl = min(rlen, round_up(k + 1, TILE) + round_up(pq, TILE));
                }
            }
            // a11: r = x - p (mod B^rlen); negative (top limb all ones) -> q - 1, r + v
            lin_addsub<T, true>(R, rlen, LimbView{Ub, hx, 0}, LimbView{PQ, pl, 0}, 0u, blk);
            // the estimate must lie in (-B^(k+2), B^(k+2)): its top limb (index >= k+2) is 0 or all ones
            if (R[rlen - 1] != 0u && R[rlen - 1] != 0xffffffffu) raise_status(ST_REM_RANGE);
            while (R[rlen - 1] != 0u && minus < CORR_MAX) {
                ++minus;
                lin_addsub<T, false>(R, rlen, LimbView{R, rlen, 0}, LimbView{Vb, k + 1, 0}, 0u, blk);
                lin_addsub<T, true>(Q, qlen, LimbView{Q, qlen, 0}, ZeroView{}, 1u, blk);
            }
        }
        if (minus == 1) count(CNT_DELTA_NEG);
        if (minus > 1) count(CNT_DELTA_NEG_MULTI);
        int plus = 0;
        for (int step = 0; step < CORR_MAX; ++step) {      // r >= v: delta = +1 (once by Theorem 2 as printed)
            if (!big_ge<T>(R, rlen, Vb, k + 1, blk)) break;     // the comparison alone: no subtraction to throw away
            lin_addsub<T, true>(R2, rlen, LimbView{R, rlen, 0}, LimbView{Vb, k + 1, 0}, 0u, blk);
            limb *t = R; R = R2; R2 = t;
            const limb qlow = Q[0];
            __syncthreads();                               // every thread has read the limb before it changes
            if (qlow != 0xffffffffu) {                     // q + 1 without a carry: one limb
                if (threadIdx.x == 0) Q[0] = qlow + 1u;
                __syncthreads();
            } else {
                lin_addsub<T, false>(Q, qlen, LimbView{Q, qlen, 0}, ZeroView{}, 1u, blk);
            }
            ++plus;
        }
        if (plus == 1) count(CNT_DELTA_POS);
        if (plus > 1) count(CNT_DELTA_MULTI);
        if (plus >= CORR_MAX || minus >= CORR_MAX) {       // not exact: say so loudly (mpdiv_status)
            count(CNT_DELTA_OUT_OF_RANGE);
            raise_status(ST_CORR_BOUND);
        }

        // a12: the quotient limbs of this window (everything above the top window is zero)
        if constexpr (BIG) {
            if (c == 0) {
                store_row<T>(qg + lo, Q, u_limbs - lo, min(qlen, u_limbs - lo));
            } else {
                if (Q[tchunk] != 0u) raise_status(ST_CORR_BOUND);     // x_c < v B^t: the quotient has t limbs
                store_row<T>(qg + lo, Q, tchunk, tchunk);
            }
            count(CNT_CHUNKS);
            __syncthreads();
        } else if (crank == 0) {
            store_row<T>(qg, Q, u_limbs, min(qlen, u_limbs));
        }
        }   // chunks

        // a12: the remainder (of the scaled problem it is r*B for one-limb divisors)
        if (crank == 0) {
            if (one_limb) store_number<T>(rg, R + 1, v_limbs, 1);
            else store_row<T>(rg, R, v_limbs, min(round_up(k + 1, 4), v_limbs));
        }
        if constexpr (CL) count(CNT_CLUSTER_DIVS);
        __syncthreads();
    }
    count_tiles(blk);
    if constexpr (MMA) {
        if (mma != nullptr) mma_fini<T>(mcx);
    }
}


// ---------------------------------------------------------------------------------------
// mplinop_batch: the linear-cost building blocks of mp_block.cuh on their own (unit tests)
// ---------------------------------------------------------------------------------------
template <int T>
__global__ void __launch_bounds__(T)
mplinop_kernel(int op, const limb *__restrict__ a, int a_limbs, const limb *__restrict__ b, int b_limbs, int shift,
               limb *__restrict__ out, int out_limbs, uint32_t *__restrict__ flag, int batch)
{
    extern __shared__ __align__(1024) uint32_t smem[];
    const int ap = round_up(a_limbs, TILE) + TILE, bp = round_up(b_limbs, TILE) + TILE, op_ = round_up(out_limbs, TILE);
    limb *A = smem, *Bs = A + ap, *O = Bs + bp;
    Blk blk{reinterpret_cast<BlkScratch *>(O + op_ + TILE), 0u, 0u};
    for (int inst = blockIdx.x; inst < batch; inst += gridDim.x) {
        load_number<T>(A, a + (size_t)inst * a_limbs, a_limbs, ap);
        load_number<T>(Bs, b + (size_t)inst * b_limbs, b_limbs, bp);
        __syncthreads();
        uint32_t f = 0;
        switch (op) {
            case MPLINOP_ADD:      // out = (a + shift_n(b)) mod B^out_limbs, flag = carry out
                f = lin_addsub<T, false>(O, op_, LimbView{A, a_limbs, 0}, LimbView{Bs, b_limbs, -shift}, 0u, blk);
                break;
            case MPLINOP_SUB:      // out = (a - shift_n(b)) mod B^out_limbs, flag = borrow = (a < shift_n(b))  (:343-440, :331-335)
                f = lin_addsub<T, true>(O, op_, LimbView{A, a_limbs, 0}, LimbView{Bs, b_limbs, -shift}, 0u, blk);
                break;
            case MPLINOP_NEG:      // out = B^shift - a for a < B^shift (the B^L - P of PowDiff)
                f = lin_addsub<T, false>(O, op_, NotView{A, shift, a_limbs}, ZeroView{}, 1u, blk);
                break;
            case MPLINOP_SHIFT:    // out = shift_n(a), whole limbs, n = shift of either sign   (Definition 1)
                lin_copy<T>(O, op_, A, a_limbs, -shift);
                break;
            case MPLINOP_PREC:     // flag = prec(a); out = a
                f = (uint32_t)prec_of<T>(A, a_limbs, blk);
                lin_copy<T>(O, op_, A, a_limbs, 0);
                break;
            default:               // MPLINOP_ANY: flag = any limb of a[shift, a_limbs) non-zero; out = a
                f = any_nonzero<T>(A, shift, a_limbs) ? 1u : 0u;
                lin_copy<T>(O, op_, A, a_limbs, 0);
                break;
        }
        store_number<T>(out + (size_t)inst * out_limbs, O, out_limbs, min(op_, out_limbs));
        if (threadIdx.x == 0) flag[inst] = f;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------
// host side of mpdiv_batch / shinv_batch / host-buffer form / counters
// ---------------------------------------------------------------------------------------
namespace {

std::mutex g_host_call_mutex;          // serialises mpdiv_batch_host's enqueue (its calls share events)

// Early Newton iterations (l <= 33) run on warp 0 alone when the SMs hold several blocks each: the idle warps
// give their issue slots to the other blocks.  A batch that leaves SMs with a single block is latency bound.
// low byte: l up to which Refine runs on warp 0 alone; bit 8: MPDIV_NO_SEED (tuning: start Refine at l = 2)
int narrow_for(int batch, const Tune &tn) { return (batch > g_sm_count ? 33 : 0) | (tn.no_seed ? 256 : 0); }

// the head kernel pays off when the SMs hold several blocks each and Refine has iterations to hand over
constexpr int HEAD_MIN_LIMBS = 512;
static bool use_head(int u_limbs, int clip, bool lat, const Tune &tn)
{
    return clip && !lat && u_limbs >= HEAD_MIN_LIMBS && !tn.no_head && !tn.no_seed;
}

// Library-owned memory pool of the current device for the head's workspace rows: freed rows stay in the pool
// (release threshold = everything), so a call costs a pool look-up, not a driver allocation.
static cudaMemPool_t head_pool()
{
    static cudaMemPool_t pools[MAX_DEVICES] = {nullptr};
    const int dev = g_dev;                                   // set by device_props() of the calling entry point
    std::lock_guard<std::mutex> lk(g_host_mutex);
    if (!pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t mp = nullptr;
        if (cudaMemPoolCreate(&mp, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &keep);
        pools[dev] = mp;
    }
    return pools[dev];
}

// Runs the head of Refine for a batch in its own kernel and returns the rows it leaves its iterates in (the static
// scratch of mpdiv_batch_noalloc, or a stream-ordered allocation the caller frees with cudaFreeAsync after the division
// kernel); nullptr = no rows (no pool on this device): Refine stays in the block.
static limb *run_head(const limb *u, int u_limbs, const limb *v, int v_limbs, int batch, cudaStream_t st, const Tune &tn,
                      int tchunk)
{
    limb *wmid = tn.wmid_fixed;
    if (!wmid && (!head_pool() ||
                  cudaMallocFromPoolAsync(reinterpret_cast<void **>(&wmid), (size_t)batch * WMID_STRIDE * sizeof(limb), head_pool(),
                                          st) != cudaSuccess)) {
        cudaGetLastError();
        return nullptr;
    }
    shinv_head_kernel<<<batch, 32, HEAD_SMEM_WORDS * 4, st>>>(u, u_limbs, v, v_limbs, wmid, batch, tchunk);
    return wmid;
}

// Launches a division kernel behind the head kernel with programmatic stream serialisation: its blocks start while the
// head still runs and wait for the head grid inside shinv_block (griddepcontrol.wait).
template <class K, class... Args>
static bool launch_behind_head(K kernel, int grid, int threads, size_t bytes, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = bytes;
    cfg.stream = st;
    cudaLaunchAttribute at;
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &at;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kernel, args...) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return true;
}

// A thread-block cluster per division (mpdiv_kernel<128, true, false, false, true>): for batches so small that
// clusters of `cs` CTAs still run all at once.  Returns the largest admissible size in {8, 4, 2} (at most cap), or 1.
static int cluster_size_query(int batch, int cap, size_t bytes)
{
    for (int cs = 8; cs >= 2; cs /= 2) {
        if (cs > cap || batch * cs > g_sm_count) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(batch * cs));
        cfg.blockDim = dim3(128);
        cfg.dynamicSmemBytes = bytes;
        cudaLaunchAttribute at;
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = (unsigned)cs;
        at.val.clusterDim.y = 1;
        at.val.clusterDim.z = 1;
        cfg.attrs = &at;
        cfg.numAttrs = 1;
        int nact = 0;
        if (cudaOccupancyMaxActiveClusters(&nact, mpdiv_kernel<128, true, false, false, true>, &cfg) != cudaSuccess) {
            cudaGetLastError();
            continue;
        }
        if (nact >= batch) return cs;
    }
    return 1;
}

static int cluster_size_for(int batch, int cap, size_t bytes)
{
    // the answer for the last question asked on each device is kept: the occupancy query costs tens of microseconds of
    // host time, and the batches that come here are the latency-bound ones
    struct Memo { int batch, cap, cs; size_t bytes; };
    static Memo memo[MAX_DEVICES] = {};
    {
        std::lock_guard<std::mutex> lk(g_host_mutex);
        const Memo &m = memo[g_dev];
        if (m.cs && m.batch == batch && m.cap == cap && m.bytes == bytes) return m.cs;
    }
    const int cs = cluster_size_query(batch, cap, bytes);
    std::lock_guard<std::mutex> lk(g_host_mutex);
    memo[g_dev] = Memo{batch, cap, cs, bytes};
    return cs;
}

static int launch_div_cluster(const limb *u, int u_limbs, const limb *v, int v_limbs, limb *q, limb *r, int batch,
                              cudaStream_t st, int clip, const Tune &tn)
{
    DivLayout L = div_layout(u_limbs + 1, v_limbs, true, clip != 0);
    const size_t bytes = div_layout_add_stage(L);
    if ((int)bytes > g_max_smem) return -1;
    if (set_smem(mpdiv_kernel<128, true, false, false, true>, bytes) != MPDIV_OK) return -1;
    const int cs = cluster_size_for(batch, tn.cluster_cap, bytes);
    if (cs < 2 || (cs == 2 && !tn.cluster_forced && u_limbs < 1536)) return -1;   // two CTAs do not pay below 2^16 bits
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(batch * cs));
    cfg.blockDim = dim3(128);
    cfg.dynamicSmemBytes = bytes;
    cfg.stream = st;
    cudaLaunchAttribute at;
    at.id = cudaLaunchAttributeClusterDimension;
    at.val.clusterDim.x = (unsigned)cs;
    at.val.clusterDim.y = 1;
    at.val.clusterDim.z = 1;
    cfg.attrs = &at;
    cfg.numAttrs = 1;
    const limb *wmid = nullptr;
    const int narrow = tn.no_seed ? 256 : 0;                 // never the narrow mode: every thread takes part in every product
    if (cudaLaunchKernelEx(&cfg, mpdiv_kernel<128, true, false, false, true>, u, u_limbs, v, v_limbs, q, r, batch, L, L, clip,
                           narrow, wmid, 0) != cudaSuccess) {
        cudaGetLastError();
        return MPDIV_ERR_CUDA;
    }
    return MPDIV_OK;
}

template <int T, bool LAT, bool MMA>
int launch_div_m(const limb *u, int u_limbs, const limb *v, int v_limbs, limb *q, limb *r, int batch,
                 cudaStream_t st, int clip, int sched, bool tensor, const Tune &tn)
{
    if constexpr (T == 128 && LAT && !MMA) {
        // a batch that leaves most SMs idle: a cluster of CTAs per division shares the tile diagonals of every product
        // (measured, 32 divisions: 2^16 bits 121 -> 99 us on four CTAs, 105 us on two; 2^15 bits 73 us either way on four,
        // 75 us on two; 2^14 bits 56 -> 60 us: the cluster barrier and the remote stores cost ~700 cycles per product)
        if (!tn.no_cluster && tn.threads == 0 && 2 * batch <= g_sm_count && (u_limbs >= 1024 || tn.cluster_forced)) {
            const int rc = launch_div_cluster(u, u_limbs, v, v_limbs, q, r, batch, st, clip, tn);
            if (rc >= 0) return rc;
        }
    }
    DivLayout L = div_layout(u_limbs + 1, v_limbs, true, clip != 0);
    DivLayout Lc = L;                                        // Lc.mma_off < 0: no engine, Lc unused
    size_t bytes = (size_t)L.total_words * 4;
    if (MMA && tensor) bytes = div_layouts_with_mma(L, Lc, u_limbs, v_limbs, clip != 0, T, LAT ? 1 : 512 / T, g_max_smem);
    int rc = set_smem(mpdiv_kernel<T, LAT, MMA>, bytes);
    if (rc != MPDIV_OK) return rc;
    // throughput batches: the head of Refine runs in its own kernel, one warp per division, and hands the
    // iterate over in a stream-ordered workspace (mp_div.cuh "Head of Refine")
    limb *wmid = use_head(u_limbs, clip, LAT, tn) ? run_head(u, u_limbs, v, v_limbs, batch, st, tn, 0) : nullptr;
    bool ok;
    if (wmid) {
        const limb *wm = wmid;
        ok = launch_behind_head(mpdiv_kernel<T, LAT, MMA>, batch, T, bytes, st, u, u_limbs, v, v_limbs, q, r, batch, L, Lc, clip,
                                narrow_for(sched, tn), wm, 0);
    } else {
        mpdiv_kernel<T, LAT, MMA><<<batch, T, bytes, st>>>(u, u_limbs, v, v_limbs, q, r, batch, L, Lc, clip, narrow_for(sched, tn), wmid, 0);
        ok = cudaGetLastError() == cudaSuccess;
    }
    if (wmid && !tn.wmid_fixed) cudaFreeAsync(wmid, st);
    return ok ? MPDIV_OK : MPDIV_ERR_CUDA;
}

// Dividends above MPDIV_MAX_OPERAND_LIMBS limbs: the chunked form (mpdiv_kernel<512, false, true, true>), clipped variant
// only, divisor strides up to MPDIV_MAX_OPERAND_LIMBS.  The chunk is the largest of 2048, 1024, 512 limbs whose layout fits.
int launch_div_big(const limb *u, int u_limbs, const limb *v, int v_limbs, limb *q, limb *r, int batch,
                   cudaStream_t st, int sched, const Tune &tn)
{
    constexpr int T = 512;
    DivLayout L;
    size_t bytes = 0;
    int t = 2048;
    for (; t >= 512; t /= 2) {
        bytes = div_layout_big(L, v_limbs, t, T, g_max_smem);
        if (bytes) break;
    }
    if (!bytes) return MPDIV_ERR_UNSUPPORTED;
    if (tn.no_mma) L.mma_off = -1;
    int rc = set_smem(mpdiv_kernel<T, false, true, true>, bytes);
    if (rc != MPDIV_OK) return rc;
    // the head of Refine in its own kernel, as for the resident form: one warp per division instead of 512 threads
    limb *wmid = (!tn.no_head && !tn.no_seed) ? run_head(u, u_limbs, v, v_limbs, batch, st, tn, t) : nullptr;
    const limb *wm = wmid;
    bool ok;
    if (wmid) {
        ok = launch_behind_head(mpdiv_kernel<T, false, true, true>, batch, T, bytes, st, u, u_limbs, v, v_limbs, q, r, batch, L, L, 1,
                                narrow_for(sched, tn), wm, t);
    } else {
        mpdiv_kernel<T, false, true, true><<<batch, T, bytes, st>>>(u, u_limbs, v, v_limbs, q, r, batch, L, L, 1, narrow_for(sched, tn),
                                                                    wm, t);
        ok = cudaGetLastError() == cudaSuccess;
    }
    if (wmid && !tn.wmid_fixed) cudaFreeAsync(wmid, st);
    return ok ? MPDIV_OK : MPDIV_ERR_CUDA;
}

template <int T, bool LAT>
int launch_div_k(const limb *u, int u_limbs, const limb *v, int v_limbs, limb *q, limb *r, int batch,
                 cudaStream_t st, int clip, int sched, const Tune &tn)
{
    // tensor-core range products: clipped variant only; 128-thread blocks from 2^16 bits up (throughput batches of
    // 2^15 bits are faster on the IMAD path alone, 7.05 M against 6.64 M div/s, and run the instantiation without
    // the engine)
    const bool tensor = DivMma<T, LAT>::value && clip && !(T <= 128 && u_limbs < 1536) && !tn.no_mma;
    if constexpr (T == 128 && !LAT) {
        if (!tensor) return launch_div_m<T, LAT, false>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, false, tn);
    }
    return launch_div_m<T, LAT, DivMma<T, LAT>::value>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tensor, tn);
}

// sched = the number of divisions that share the GPU with this launch (the batch itself, or the whole batch
// when the host path launches it chunk by chunk on several streams): it picks the kernel flavour.
template <int T>
int launch_div(const limb *u, int u_limbs, const limb *v, int v_limbs, limb *q, limb *r, int batch,
               cudaStream_t st, int clip, int sched, const Tune &tn)
{
    // a batch that fits the SMs at the latency kernel's occupancy (two blocks per SM up to 128 threads, one at
    // 256) is latency bound: give its threads all the registers they want
    if constexpr (T <= 256) {
        if (sched <= (T <= 128 ? 2 : 1) * g_sm_count)
            return launch_div_k<T, true>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
    }
    return launch_div_k<T, false>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
}

template <int T>
int launch_shinv(const limb *v, int v_limbs, int h, limb *w, int w_limbs, int batch, cudaStream_t st, int clip,
                 const Tune &tn)
{
    const DivLayout L = div_layout(h + 1, v_limbs, false, clip != 0);
    const size_t bytes = (size_t)L.total_words * 4;
    int rc = set_smem(shinv_kernel<T>, bytes);
    if (rc != MPDIV_OK) return rc;
    shinv_kernel<T><<<batch, T, bytes, st>>>(v, v_limbs, h, w, w_limbs, batch, L, clip, narrow_for(batch, tn));
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

int check_div_args(const void *u, int u_limbs, const void *v, int v_limbs, const void *q, const void *r,
                   int batch)
{
    if (!u || !v || !q || !r || u_limbs <= 0 || v_limbs <= 0 || batch <= 0) return MPDIV_ERR_BAD_ARG;
    if ((u_limbs | v_limbs) & 3) return MPDIV_ERR_BAD_ARG;
    if (u_limbs > MPDIV_MAX_LIMBS || v_limbs > MPDIV_MAX_OPERAND_LIMBS) return MPDIV_ERR_UNSUPPORTED;
    return MPDIV_OK;
}

}  // namespace

extern "C" {

int mpdiv_batch(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs, uint32_t *q, uint32_t *r,
                int batch, mpdiv_stream_t stream)
{
    return mpdiv_batch_ex(u, u_limbs, v, v_limbs, q, r, batch, MPDIV_VARIANT_DEFAULT, stream);
}

static int div_dispatch(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs, uint32_t *q, uint32_t *r,
                        int batch, int clip, cudaStream_t st, int sched, const Tune &tn)
{
    if (u_limbs > MPDIV_MAX_OPERAND_LIMBS) {                   // the dividend does not fit on chip: chunked form
        if (!clip) return MPDIV_ERR_UNSUPPORTED;
        return launch_div_big(u, u_limbs, v, v_limbs, q, r, batch, st, sched, tn);
    }
    switch (threads_for(u_limbs, tn.threads, sched)) {
        case 32: return launch_div<32>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
        case 64: return launch_div<64>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
        case 128: return launch_div<128>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
        case 256: return launch_div<256>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
        default: return launch_div<512>(u, u_limbs, v, v_limbs, q, r, batch, st, clip, sched, tn);
    }
}

int mpdiv_batch_ex(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs, uint32_t *q, uint32_t *r,
                   int batch, int flags, mpdiv_stream_t stream)
{
    if (!flags_ok(flags)) return MPDIV_ERR_BAD_ARG;
    const int clip = (flags & MPDIV_VARIANT_MASK) == MPDIV_VARIANT_CLIPPED;
    int rc = check_div_args(u, u_limbs, v, v_limbs, q, r, batch);
    if (rc != MPDIV_OK) return rc;
    if (!aligned16(u) || !aligned16(v) || !aligned16(q) || !aligned16(r)) return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    return div_dispatch(u, u_limbs, v, v_limbs, q, r, batch, clip, reinterpret_cast<cudaStream_t>(stream), batch, tune_of(flags));
}

int shinv_batch(const uint32_t *v, int v_limbs, int h, uint32_t *w, int w_limbs, int batch,
                mpdiv_stream_t stream)
{
    // Theorem 2's value, lambda in {0, 1}: the algorithm as printed
    return shinv_batch_ex(v, v_limbs, h, w, w_limbs, batch, MPDIV_VARIANT_PRINTED, stream);
}

int shinv_batch_ex(const uint32_t *v, int v_limbs, int h, uint32_t *w, int w_limbs, int batch, int flags,
                   mpdiv_stream_t stream)
{
    if (!flags_ok(flags)) return MPDIV_ERR_BAD_ARG;
    const int clip = (flags & MPDIV_VARIANT_MASK) == MPDIV_VARIANT_CLIPPED;
    const Tune tn = tune_of(flags);
    if (!v || !w || v_limbs <= 0 || w_limbs <= 0 || batch <= 0 || h < 1) return MPDIV_ERR_BAD_ARG;
    if ((v_limbs | w_limbs) & 3) return MPDIV_ERR_BAD_ARG;
    if (w_limbs < h + 1) return MPDIV_ERR_BAD_ARG;
    if (!aligned16(v) || !aligned16(w)) return MPDIV_ERR_BAD_ARG;
    if (h > MPDIV_MAX_OPERAND_LIMBS || v_limbs > MPDIV_MAX_OPERAND_LIMBS) return MPDIV_ERR_UNSUPPORTED;
    if (!device_props()) return MPDIV_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    switch (threads_for(h, tn.threads)) {
        case 64: return launch_shinv<64>(v, v_limbs, h, w, w_limbs, batch, st, clip, tn);
        case 128: return launch_shinv<128>(v, v_limbs, h, w, w_limbs, batch, st, clip, tn);
        case 256: return launch_shinv<256>(v, v_limbs, h, w, w_limbs, batch, st, clip, tn);
        default: return launch_shinv<512>(v, v_limbs, h, w, w_limbs, batch, st, clip, tn);
    }
}


int mplinop_batch(int op, const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs, int shift, uint32_t *out,
                  int out_limbs, uint32_t *flag, int batch, mpdiv_stream_t stream)
{
    if (!a || !b || !out || !flag || a_limbs <= 0 || b_limbs <= 0 || out_limbs <= 0 || batch <= 0) return MPDIV_ERR_BAD_ARG;
    if (op < MPLINOP_ADD || op > MPLINOP_ANY) return MPDIV_ERR_BAD_ARG;
    if ((a_limbs | b_limbs | out_limbs) & 3) return MPDIV_ERR_BAD_ARG;
    if (!aligned16(a) || !aligned16(b) || !aligned16(out)) return MPDIV_ERR_BAD_ARG;
    if (a_limbs > MPDIV_MAX_OPERAND_LIMBS || b_limbs > MPDIV_MAX_OPERAND_LIMBS || out_limbs > 2 * MPDIV_MAX_OPERAND_LIMBS) return MPDIV_ERR_UNSUPPORTED;
    if (shift < -2 * MPDIV_MAX_OPERAND_LIMBS || shift > 2 * MPDIV_MAX_OPERAND_LIMBS) return MPDIV_ERR_BAD_ARG;
    if ((op == MPLINOP_NEG && (shift < 0 || shift > out_limbs)) || (op == MPLINOP_ANY && shift < 0)) return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const size_t words = (size_t)round_up(a_limbs, TILE) + round_up(b_limbs, TILE) + round_up(out_limbs, TILE) + 3 * TILE +
                         sizeof(BlkScratch) / 4;
    const size_t bytes = words * 4;
    const int big = out_limbs > a_limbs ? out_limbs : a_limbs;
    if (big <= 1024) {
        int rc = set_smem(mplinop_kernel<128>, bytes);
        if (rc != MPDIV_OK) return rc;
        mplinop_kernel<128><<<batch, 128, bytes, st>>>(op, a, a_limbs, b, b_limbs, shift, out, out_limbs, flag, batch);
    } else {
        int rc = set_smem(mplinop_kernel<512>, bytes);
        if (rc != MPDIV_OK) return rc;
        mplinop_kernel<512><<<batch, 512, bytes, st>>>(op, a, a_limbs, b, b_limbs, shift, out, out_limbs, flag, batch);
    }
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

size_t mpdiv_host_workspace_bytes(int u_limbs, int v_limbs, int batch)
{
    if (u_limbs <= 0 || v_limbs <= 0 || batch <= 0) return 0;
    return (size_t)batch * 2 * ((size_t)u_limbs + (size_t)v_limbs) * sizeof(uint32_t);
}

int mpdiv_batch_host(const uint32_t *u_host, int u_limbs, const uint32_t *v_host, int v_limbs,
                     uint32_t *q_host, uint32_t *r_host, int batch, void *workspace, size_t workspace_bytes,
                     mpdiv_stream_t stream)
{
    int rc = check_div_args(u_host, u_limbs, v_host, v_limbs, q_host, r_host, batch);
    if (rc != MPDIV_OK) return rc;
    if (!workspace || !aligned16(workspace)) return MPDIV_ERR_BAD_ARG;
    if (workspace_bytes < mpdiv_host_workspace_bytes(u_limbs, v_limbs, batch)) return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    uint32_t *du = static_cast<uint32_t *>(workspace);
    uint32_t *dv = du + (size_t)batch * u_limbs;
    uint32_t *dq = dv + (size_t)batch * v_limbs;
    uint32_t *dr = dq + (size_t)batch * u_limbs;

    // Chunks of one division per SM, two up to 2048 limbs (at most MAXC chunks).  The upload of chunk i+1 and the download of chunk
    // i-1 overlap the division of chunk i, and the chunk kernels go round NK streams so that the blocks of
    // consecutive chunks share the SMs like the blocks of one launch would (a chunk alone would leave each SM
    // with a single block); the kernel flavour is the one the whole batch would get.
    constexpr int MAXC = 16, NK = 4;
    // (measured at config 2: 4 chunks 590 us, 8 chunks 620-640 us, 2 chunks 640 us, 1 chunk 850 us per batch; at configs 3 and
    // 4, whose kernels take as long as their copies, one division per SM and chunk is 7-10 % faster than two)
    int nchunks = batch / ((u_limbs <= 2048 ? 2 : 1) * g_sm_count);
    if (nchunks < 1) nchunks = 1;
    if (nchunks > MAXC) nchunks = MAXC;
    const int chunk = (batch + nchunks - 1) / nchunks;
    nchunks = (batch + chunk - 1) / chunk;

    // helper streams and events of the current device: created once, all or nothing, under the host lock;
    // the lock also serialises the enqueue of concurrent calls (they share the events)
    struct HostRes {
        bool ok = false;
        cudaStream_t s_in = nullptr, s_out = nullptr, s_k[NK] = {};
        cudaEvent_t ev_start = nullptr, ev_done = nullptr, ev_in[MAXC] = {}, ev_k[MAXC] = {};
    };
    static HostRes res[MAX_DEVICES];
    std::lock_guard<std::mutex> lk(g_host_call_mutex);
    HostRes &hr = res[g_dev];
    if (!hr.ok) {
        HostRes t;
        bool good = cudaStreamCreateWithFlags(&t.s_in, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaStreamCreateWithFlags(&t.s_out, cudaStreamNonBlocking) == cudaSuccess &&
                    cudaEventCreateWithFlags(&t.ev_start, cudaEventDisableTiming) == cudaSuccess &&
                    cudaEventCreateWithFlags(&t.ev_done, cudaEventDisableTiming) == cudaSuccess;
        for (int i = 0; good && i < NK; i++) good = cudaStreamCreateWithFlags(&t.s_k[i], cudaStreamNonBlocking) == cudaSuccess;
        for (int i = 0; good && i < MAXC; i++)
            good = cudaEventCreateWithFlags(&t.ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
                   cudaEventCreateWithFlags(&t.ev_k[i], cudaEventDisableTiming) == cudaSuccess;
        if (!good) {                                          // nothing half-made survives
            cudaGetLastError();
            if (t.s_in) cudaStreamDestroy(t.s_in);
            if (t.s_out) cudaStreamDestroy(t.s_out);
            if (t.ev_start) cudaEventDestroy(t.ev_start);
            if (t.ev_done) cudaEventDestroy(t.ev_done);
            for (int i = 0; i < NK; i++) if (t.s_k[i]) cudaStreamDestroy(t.s_k[i]);
            for (int i = 0; i < MAXC; i++) {
                if (t.ev_in[i]) cudaEventDestroy(t.ev_in[i]);
                if (t.ev_k[i]) cudaEventDestroy(t.ev_k[i]);
            }
            return MPDIV_ERR_CUDA;
        }
        t.ok = true;
        hr = t;
    }
    // on an error part of the batch may be in flight on the helper streams: wait for it, so that the caller may
    // reuse or free its buffers as soon as the call has returned
    auto fail = [&](int code) {
        cudaGetLastError();
        cudaStreamSynchronize(hr.s_in);
        for (int i = 0; i < NK; i++) cudaStreamSynchronize(hr.s_k[i]);
        cudaStreamSynchronize(hr.s_out);
        cudaGetLastError();
        return code;
    };
#define MPDIV_CK(x) do { if ((x) != cudaSuccess) return fail(MPDIV_ERR_CUDA); } while (0)
    const Tune tn = tune_of(0);
    MPDIV_CK(cudaEventRecord(hr.ev_start, st));               // the helpers start after earlier work on `stream`
    MPDIV_CK(cudaStreamWaitEvent(hr.s_in, hr.ev_start, 0));
    for (int c = 0; c < nchunks; c++) {
        const size_t lo = (size_t)c * chunk;
        const int cnt = (int)((size_t)batch - lo < (size_t)chunk ? (size_t)batch - lo : (size_t)chunk);
        const size_t uo = lo * u_limbs, vo = lo * v_limbs;
        cudaStream_t sk = hr.s_k[c % NK];
        MPDIV_CK(cudaMemcpyAsync(du + uo, u_host + uo, (size_t)cnt * u_limbs * 4, cudaMemcpyHostToDevice, hr.s_in));
        MPDIV_CK(cudaMemcpyAsync(dv + vo, v_host + vo, (size_t)cnt * v_limbs * 4, cudaMemcpyHostToDevice, hr.s_in));
        MPDIV_CK(cudaEventRecord(hr.ev_in[c], hr.s_in));
        MPDIV_CK(cudaStreamWaitEvent(sk, hr.ev_in[c], 0));    // ev_in follows ev_start on s_in
        rc = div_dispatch(du + uo, u_limbs, dv + vo, v_limbs, dq + uo, dr + vo, cnt, 1, sk, batch, tn);
        if (rc != MPDIV_OK) return fail(rc);
        MPDIV_CK(cudaEventRecord(hr.ev_k[c], sk));
        MPDIV_CK(cudaStreamWaitEvent(hr.s_out, hr.ev_k[c], 0));
        MPDIV_CK(cudaMemcpyAsync(q_host + uo, dq + uo, (size_t)cnt * u_limbs * 4, cudaMemcpyDeviceToHost, hr.s_out));
        MPDIV_CK(cudaMemcpyAsync(r_host + vo, dr + vo, (size_t)cnt * v_limbs * 4, cudaMemcpyDeviceToHost, hr.s_out));
    }
    MPDIV_CK(cudaEventRecord(hr.ev_done, hr.s_out));          // s_out has waited for every chunk kernel
    MPDIV_CK(cudaStreamWaitEvent(st, hr.ev_done, 0));         // `stream` completes when the last download has
#undef MPDIV_CK
    return MPDIV_OK;
}

int mpdiv_batch_launches(int u_limbs, int batch, int flags)
{
    if (u_limbs <= 0 || batch <= 0 || !flags_ok(flags) || !device_props()) return 0;
    const Tune tn = tune_of(flags);
    if (u_limbs > MPDIV_MAX_OPERAND_LIMBS) return (!tn.no_head && !tn.no_seed) ? 2 : 1;
    const int T = threads_for(u_limbs, tn.threads, batch);
    const bool lat = T <= 256 && batch <= (T <= 128 ? 2 : 1) * g_sm_count;
    return use_head(u_limbs, (flags & MPDIV_VARIANT_MASK) == MPDIV_VARIANT_CLIPPED, lat, tn) ? 2 : 1;
}

int mpdiv_seed_batch(const uint32_t *v, int v_limbs, uint32_t *w, int batch, mpdiv_stream_t stream)
{
    if (!v || !w || v_limbs <= 0 || batch <= 0) return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    seed_kernel<<<(batch + 3) / 4, 128, 0, reinterpret_cast<cudaStream_t>(stream)>>>(v, v_limbs, w, batch);
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

int mpdiv_debug_counters(unsigned long long out[MPDIV_NUM_COUNTERS], int reset, mpdiv_stream_t stream)
{
    static_assert(MPDIV_NUM_COUNTERS == NUM_COUNTERS, "header and device counters agree");
    if (!out) return MPDIV_ERR_BAD_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (cudaStreamSynchronize(st) != cudaSuccess) return MPDIV_ERR_CUDA;
    if (cudaMemcpyFromSymbol(out, g_counters, NUM_COUNTERS * sizeof(unsigned long long)) != cudaSuccess) return MPDIV_ERR_CUDA;
    unsigned int mma_fail = 0;
    if (cudaMemcpyFromSymbol(&mma_fail, g_mma_fail, sizeof(mma_fail)) != cudaSuccess) return MPDIV_ERR_CUDA;
    out[CNT_MMA_WAIT_FAILURES] = mma_fail;
    if (reset) {
        const unsigned int zf = 0;
        if (cudaMemcpyToSymbol(g_mma_fail, &zf, sizeof(zf)) != cudaSuccess) return MPDIV_ERR_CUDA;
        unsigned long long z[NUM_COUNTERS] = {0};
        if (cudaMemcpyToSymbol(g_counters, z, sizeof(z)) != cudaSuccess) return MPDIV_ERR_CUDA;
    }
    return MPDIV_OK;
}

int mpdiv_status(mpdiv_stream_t stream, unsigned int *flags, int reset)
{
    static_assert(MPDIV_STATUS_MMA_WAIT == ST_MMA_WAIT && MPDIV_STATUS_CORR_BOUND == ST_CORR_BOUND &&
                  MPDIV_STATUS_REM_RANGE == ST_REM_RANGE && MPDIV_STATUS_V_ZERO == ST_V_ZERO && MPDIV_STATUS_IO_WAIT == ST_IO_WAIT,
                  "status bits agree");
    if (!flags) return MPDIV_ERR_BAD_ARG;
    if (cudaStreamSynchronize(reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess) return MPDIV_ERR_CUDA;
    if (cudaMemcpyFromSymbol(flags, g_status, sizeof(unsigned int)) != cudaSuccess) return MPDIV_ERR_CUDA;
    if (reset) {
        const unsigned int z = 0;
        if (cudaMemcpyToSymbol(g_status, &z, sizeof(z)) != cudaSuccess) return MPDIV_ERR_CUDA;
    }
    return MPDIV_OK;
}

}  // extern "C"
