// libmpdiv.so -- kernels and C ABI (include/mpdiv.h).  sm_100a only.
#include <atomic>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <unordered_map>
#include <cuda_runtime.h>

#include "../../include/mpdiv.h"
#include "mp_block.cuh"
#include "mp_mul.cuh"
#include "mp_div.cuh"
#include "mp_io.cuh"

using namespace mpd;

#define MPDIV_VERSION_STR "mpdiv 0.7 sm_100a (B200) limbs=u32 imad.wide 8x8 tiles + int8 tcgen05 range products, bulk-copy rows, warp/block/cluster per division, dividends to 2^19 bits"

// ---------------------------------------------------------------------------------------
// mpmul_batch
// ---------------------------------------------------------------------------------------
struct MulLayout {
    int a_off, b_off, p_off, hi_off, ov_off, c3_off, sc_off, total_words;
    int mma_off, mma_rows, mma_cols;     // tensor-core scratch (mp_mma.cuh), mma_off = -1 when absent
};

static MulLayout mul_layout(int a_limbs, int b_limbs, int c_limbs)
{
    MulLayout L;
    const int pa = round_up(a_limbs, TILE) + TILE;
    const int pb = round_up(b_limbs, TILE) + TILE;
    const int full = round_up(a_limbs, TILE) + round_up(b_limbs, TILE);
    const int pc = round_up(c_limbs < full ? c_limbs : full, TILE) + 2 * TILE;
    int o = 0;
    L.a_off = o; o += pa;
    L.b_off = o; o += pb;
    L.p_off = o; o += pc;
    L.hi_off = o; o += pc;
    L.ov_off = o; o += round_up(pc / TILE, 4);
    L.c3_off = o; o += round_up(pc / TILE, 4);
    L.sc_off = o; o += (int)(sizeof(BlkScratch) / 4);
    L.total_words = o;
    L.mma_off = -1;
    L.mma_rows = 0;
    L.mma_cols = 0;
    return L;
}

// Scratch of the tensor-core engine for a product of a_limbs x b_limbs truncated to c_limbs; false if the
// request does not fit (TMEM has 512 columns = 512 output blocks of 32 limbs; shared memory max_smem bytes).
static bool mul_layout_add_mma(MulLayout &L, int a_limbs, int b_limbs, int c_limbs, int max_smem)
{
    const int full = (a_limbs + b_limbs + 31) / 32, want = (c_limbs + 31) / 32;
    const int blocks = want < full ? want : full;
    const int nn = (blocks + 15) & ~15;
    if (nn > 512) return false;
    const int sets = 2 * nn;                                     // one accumulator set per issuing warp when they fit
    const int cols = sets <= 32 ? 32 : sets <= 64 ? 64 : sets <= 128 ? 128 : sets <= 256 ? 256 : 512;
    const int small = a_limbs < b_limbs ? a_limbs : b_limbs;
    const int rows = round_up(nn + (small + 31) / 32 + 8, 8);
    // P and HI must hold 32 limbs per output block
    const int pc = 32 * blocks + 2 * TILE;
    const int grow = pc - (L.hi_off - L.p_off);
    if (grow > 0) {                       // re-lay P, HI, OV, C3, scratch with the larger product buffers
        int o = L.p_off;
        L.p_off = o; o += pc;
        L.hi_off = o; o += pc;
        L.ov_off = o; o += round_up(pc / TILE, 4);
        L.c3_off = o; o += round_up(pc / TILE, 4);
        L.sc_off = o; o += (int)(sizeof(BlkScratch) / 4);
        L.total_words = o;
    }
    const int off = round_up(L.total_words, 256);
    const int words = (mma_scratch_bytes(rows, 512) + MMA_BAR_BYTES) / 4;     // launch_mul<512> runs this engine
    if ((off + words) * 4 > max_smem) return false;
    L.mma_off = off;
    L.mma_rows = rows;
    L.mma_cols = cols;
    L.total_words = off + words;
    return true;
}

template <int T>
__global__ void __launch_bounds__(T, 512 / T)
mpmul_kernel(const limb *__restrict__ a, int a_limbs, const limb *__restrict__ b, int b_limbs,
             limb *__restrict__ c, int c_limbs, int batch, MulLayout L)
{
    extern __shared__ __align__(1024) uint32_t smem[];
    limb *A = smem + L.a_off, *Bs = smem + L.b_off, *P = smem + L.p_off;
    MulScratch ms{smem + L.hi_off, smem + L.ov_off, smem + L.c3_off, nullptr, 0};
    Blk blk{reinterpret_cast<BlkScratch *>(smem + L.sc_off), 0u};
    MmaCtx mcx;
    bool tensor = false;
    if constexpr (MmaEnabled<T>::value) {
        if (L.mma_off >= 0) {
            uint8_t *scratch = reinterpret_cast<uint8_t *>(smem + L.mma_off);
            mma_init<T>(mcx, scratch, L.mma_rows, scratch + mma_scratch_bytes(L.mma_rows, T), L.mma_cols);
            tensor = true;
        } else {
            mma_decline();
        }
    }

    for (int inst = blockIdx.x; inst < batch; inst += gridDim.x) {
        load_number<T>(A, a + (size_t)inst * a_limbs, a_limbs, round_up(a_limbs, TILE) + TILE);
        load_number<T>(Bs, b + (size_t)inst * b_limbs, b_limbs, round_up(b_limbs, TILE) + TILE);
        __syncthreads();
        const int na = prec_of<T>(A, a_limbs, blk);
        const int nb = prec_of<T>(Bs, b_limbs, blk);
        int valid = 0;
        if constexpr (MmaEnabled<T>::value) {
            if (tensor && na > 0 && nb > 0) {
                // the operand with fewer 128-byte chunks becomes the Toeplitz operand (fewer MMA steps)
                const int dhi = (c_limbs + 31) / 32;
                const bool swap = mma_steps(nb, na, 0, dhi) < mma_steps(na, nb, 0, dhi);
                valid = swap ? mma_mul_range<T>(mcx, Bs, nb, A, na, 0, dhi, P, ms.HI, blk)
                             : mma_mul_range<T>(mcx, A, na, Bs, nb, 0, dhi, P, ms.HI, blk);
                if (valid > c_limbs) valid = c_limbs;
            }
        }
        if (valid > 0) {
        } else if (na > 0 && nb > 0) {
            if (c_limbs >= na + nb) {
                mul_full<T>(A, na, Bs, nb, P, ms, blk);
                valid = round_up(na, TILE) + round_up(nb, TILE);
            } else {
                mul_low<T>(A, na, Bs, nb, c_limbs, P, ms, blk);
                valid = c_limbs;
            }
        }
        store_number<T>(c + (size_t)inst * c_limbs, P, c_limbs, valid);
        __syncthreads();
    }
    if constexpr (MmaEnabled<T>::value) {
        if (tensor) mma_fini<T>(mcx);
    }
}

// ---------------------------------------------------------------------------------------
// integer-multiply roofline probe
// ---------------------------------------------------------------------------------------
constexpr int PROBE_THREADS = 256;
constexpr int PROBE_BLOCKS_PER_SM = 4;

template <int KIND>
__global__ void __launch_bounds__(PROBE_THREADS)
imad_probe_kernel(uint32_t *sink, int iters)
{
    if (KIND == 0) {
        // the multiplier's own inner tile: 64 carry-chained IMAD.WIDE.U32 + 16 carry counters
        DiagAcc s;
        s.clear();
        uint32_t a[8], b[8];
#pragma unroll
        for (int j = 0; j < 8; j++) {
            a[j] = threadIdx.x * 2654435761u + j * 40503u + 1u;
            b[j] = blockIdx.x * 2246822519u + j * 9973u + 7u;
        }
        for (int it = 0; it < iters; ++it) {
            tile_mac(s, a, b);
            a[0] ^= s.CY[0];   // keep the operands loop-variant without extra multiplies
        }
        uint32_t d[17];
        diag_finish(s, d);
        uint32_t x = 0;
#pragma unroll
        for (int j = 0; j < 17; j++) x ^= d[j];
        sink[blockIdx.x * PROBE_THREADS + threadIdx.x] = x;
    } else {
        // 64 independent plain 32-bit IMADs per round (no carry, no wide result)
        uint32_t acc[16];
#pragma unroll
        for (int j = 0; j < 16; j++) acc[j] = threadIdx.x + j;
        uint32_t m = blockIdx.x * 2246822519u + 12345u;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 4; r++)
#pragma unroll
                for (int j = 0; j < 16; j++) acc[j] = acc[j] * m + acc[(j + 1) & 15];
        }
        uint32_t x = 0;
#pragma unroll
        for (int j = 0; j < 16; j++) x ^= acc[j];
        sink[blockIdx.x * PROBE_THREADS + threadIdx.x] = x;
    }
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
namespace {

// Per-device facts, cached on first use (any host thread, any device): the entry points call device_props()
// first, which refreshes the thread-local copies for the CURRENT device.
constexpr int MAX_DEVICES = 64;
struct DevInfo { int sm_count, max_smem; };
std::mutex g_host_mutex;                         // guards every lazily created library-owned host object
DevInfo g_devinfo[MAX_DEVICES];
std::atomic<bool> g_devinfo_ok[MAX_DEVICES];
thread_local int g_dev = 0, g_sm_count = 0, g_max_smem = 0;

bool device_props()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return false;
    if (!g_devinfo_ok[dev].load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lk(g_host_mutex);
        DevInfo d{0, 0};
        if (cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return false;
        if (cudaDeviceGetAttribute(&d.max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return false;
        if (d.sm_count <= 0) return false;
        g_devinfo[dev] = d;
        g_devinfo_ok[dev].store(true, std::memory_order_release);
    }
    g_dev = dev;
    g_sm_count = g_devinfo[dev].sm_count;
    g_max_smem = g_devinfo[dev].max_smem;
    return true;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Tuning switches carried by the `flags` argument of the *_ex calls (include/mpdiv.h).
struct Tune {
    bool no_seed, no_head, no_mma, no_cluster;
    int cluster_cap;                             // largest cluster per division (MPDIV_FLAG_CLUSTER; default 4)
    bool cluster_forced;                         // MPDIV_FLAG_CLUSTER given: use clusters wherever they fit
    int threads;                                 // 0 = by size
    limb *wmid_fixed;                            // mpdiv_batch_noalloc: the head kernel's rows live here (no pool allocation)
};
Tune tune_of(int flags)
{
    Tune t;
    t.no_seed = (flags & MPDIV_FLAG_NO_SEED) != 0;
    t.no_head = (flags & MPDIV_FLAG_NO_HEAD) != 0;
    t.no_mma = (flags & MPDIV_FLAG_NO_MMA) != 0;
    t.no_cluster = (flags & MPDIV_FLAG_NO_CLUSTER) != 0;
    const int cc = (flags & MPDIV_FLAG_CLUSTER_MASK) >> 12;
    t.cluster_cap = cc ? 1 << cc : 4;
    t.cluster_forced = cc != 0;
    const int c = (flags & MPDIV_FLAG_THREADS_MASK) >> 8;
    t.threads = c >= 1 && c <= 4 ? 32 << c : (c == 5 ? 32 : 0);
    t.wmid_fixed = nullptr;
    return t;
}
bool flags_ok(int flags)
{
    const int var = flags & MPDIV_VARIANT_MASK;
    if (var != MPDIV_VARIANT_PRINTED && var != MPDIV_VARIANT_CLIPPED) return false;
    if (flags & ~(MPDIV_VARIANT_MASK | MPDIV_FLAG_NO_SEED | MPDIV_FLAG_NO_HEAD | MPDIV_FLAG_NO_MMA | MPDIV_FLAG_NO_CLUSTER |
                  MPDIV_FLAG_THREADS_MASK | MPDIV_FLAG_CLUSTER_MASK)) return false;
    return ((flags & MPDIV_FLAG_THREADS_MASK) >> 8) <= 5;
}

// threads per block for numbers of `limbs` limbs.  Four lanes share a tile diagonal (mp_mul.cuh), so
// a block of T threads covers T/4 diagonals = 2T limbs of product per pass.  256 threads at 128
// registers let two blocks share an SM up to 4096 limbs; above that one block of 512 fills the SM.
// sched = the divisions that share the GPU (0 = unknown).  Small numbers in large batches (the
// paper's "suboptimal number of threads per CUDA block" below 2^15 bits): a block is too big
// a unit, so a division gets ONE WARP (32-thread blocks, 16 resident per SM, warp-level barriers only) up to 512
// limbs and two warps at 1024 -- measured on 4736-9472 divisions: 68.6 M div/s against 40.4 M at 32 limbs, 27.3 M
// against 12.3 M at 256, 16.3 M against 11.4 M at 512, 7.84 M against 7.15 M at 1024 limbs.
int threads_for(int limbs, int override_threads = 0, int sched = 0)
{
    if (override_threads) return override_threads;
    if (limbs <= 512 && sched >= 16 * g_sm_count) return 32;
    if (limbs <= 128) return 64;
    if (limbs <= 1024 && sched >= 8 * g_sm_count) return 64;
    if (limbs <= 2048) return 128;      // four blocks per SM overlap the latency-bound early iterations
    if (limbs <= 4096) return 256;
    return 512;
}

// Opt a kernel in to the device's full dynamic shared memory, once per kernel and device (the launch itself
// states how much it uses, so occupancy is unaffected).
int set_smem(const void *kernel, size_t bytes)
{
    if ((int)bytes > g_max_smem) return MPDIV_ERR_UNSUPPORTED;
    static std::unordered_map<const void *, unsigned long long> done;     // kernel -> mask of devices
    std::lock_guard<std::mutex> lk(g_host_mutex);
    unsigned long long &mask = done[kernel];
    if (mask >> g_dev & 1ull) return MPDIV_OK;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, g_max_smem) != cudaSuccess) {
        cudaGetLastError();
        return MPDIV_ERR_CUDA;
    }
    mask |= 1ull << g_dev;
    return MPDIV_OK;
}
template <class K>
int set_smem(K kernel, size_t bytes) { return set_smem(reinterpret_cast<const void *>(kernel), bytes); }

template <int T>
int launch_mul(const limb *a, int a_limbs, const limb *b, int b_limbs, limb *c, int c_limbs, int batch,
               cudaStream_t st, bool tensor = false)
{
    MulLayout L = mul_layout(a_limbs, b_limbs, c_limbs);
    if (tensor && !(MmaEnabled<T>::value && mul_layout_add_mma(L, a_limbs, b_limbs, c_limbs, g_max_smem)))
        return MPDIV_ERR_UNSUPPORTED;
    const size_t bytes = (size_t)L.total_words * 4;
    int rc = set_smem(mpmul_kernel<T>, bytes);
    if (rc != MPDIV_OK) return rc;
    mpmul_kernel<T><<<batch, T, bytes, st>>>(a, a_limbs, b, b_limbs, c, c_limbs, batch, L);
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

}  // namespace

extern "C" {

int mpmul_batch(const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs, uint32_t *c, int c_limbs,
                int batch, mpdiv_stream_t stream)
{
    return mpmul_batch_ex(a, a_limbs, b, b_limbs, c, c_limbs, batch, MPMUL_ENGINE_IMAD, stream);
}

int mpmul_batch_ex(const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs, uint32_t *c, int c_limbs,
                   int batch, int engine, mpdiv_stream_t stream)
{
    if (engine != MPMUL_ENGINE_IMAD && engine != MPMUL_ENGINE_TENSOR) return MPDIV_ERR_BAD_ARG;
    if (!a || !b || !c || a_limbs <= 0 || b_limbs <= 0 || c_limbs <= 0 || batch <= 0) return MPDIV_ERR_BAD_ARG;
    if ((a_limbs | b_limbs | c_limbs) & 3) return MPDIV_ERR_BAD_ARG;
    if (!aligned16(a) || !aligned16(b) || !aligned16(c)) return MPDIV_ERR_BAD_ARG;
    if (c_limbs > a_limbs + b_limbs) return MPDIV_ERR_BAD_ARG;
    if (a_limbs > MPDIV_MAX_OPERAND_LIMBS || b_limbs > MPDIV_MAX_OPERAND_LIMBS) return MPDIV_ERR_UNSUPPORTED;
    if (!device_props()) return MPDIV_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (engine == MPMUL_ENGINE_TENSOR) return launch_mul<512>(a, a_limbs, b, b_limbs, c, c_limbs, batch, st, true);
    const int big = a_limbs > b_limbs ? a_limbs : b_limbs;
    switch (threads_for(big)) {
        case 64: return launch_mul<64>(a, a_limbs, b, b_limbs, c, c_limbs, batch, st);
        case 128: return launch_mul<128>(a, a_limbs, b, b_limbs, c, c_limbs, batch, st);
        case 256: return launch_mul<256>(a, a_limbs, b, b_limbs, c, c_limbs, batch, st);
        default: return launch_mul<512>(a, a_limbs, b, b_limbs, c, c_limbs, batch, st);
    }
}

int mpdiv_imad_probe_threads(void)
{
    if (!device_props()) return 0;
    return g_sm_count * PROBE_BLOCKS_PER_SM * PROBE_THREADS;
}

int mpdiv_imad_probe(uint32_t *sink, int kind, int iters, unsigned long long *products, mpdiv_stream_t stream)
{
    if (!sink || iters <= 0 || (kind != 0 && kind != 1)) return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int blocks = g_sm_count * PROBE_BLOCKS_PER_SM;
    if (kind == 0) imad_probe_kernel<0><<<blocks, PROBE_THREADS, 0, st>>>(sink, iters);
    else imad_probe_kernel<1><<<blocks, PROBE_THREADS, 0, st>>>(sink, iters);
    if (products) *products = (unsigned long long)blocks * PROBE_THREADS * 64ull * (unsigned long long)iters;
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------
// tensor-core issue-rate probe (include/mpdiv.h: mpdiv_mma_probe)
// ---------------------------------------------------------------------------------------
// One block of 128 threads per SM; `issuers` warps (1 or 2) each issue `iters` steps of four
// tcgen05.mma.kind::i8 (M = 128, K = 32, N = n_cols, B = swizzled shared-memory rows) into their own accumulator
// columns, in the warp form the multiplier uses (mp_mma.cuh: operand words in ordinary registers, one lane elected
// around the four MMAs and the commit).  form 0: A in tensor memory (the pure rate of the pipe: the roofline
// denominator); form 1: A read from shared memory through the overlapped Toeplitz descriptor, as the multiplier
// issues it.  Operand contents are arbitrary; nothing is read back.  cycles[warp] of block 0 = clock64 from the
// first issue to the completion barrier.
}  // extern "C"
constexpr int MMA_PROBE_ROWS = 272;
template <int FORM>
__global__ void __launch_bounds__(128)
mma_probe_kernel(int n_cols, int issuers, int iters, unsigned long long *cycles)
{
    extern __shared__ __align__(1024) uint8_t psm[];
    for (int i = threadIdx.x; i < mma_scratch_bytes(MMA_PROBE_ROWS, 128) / 4; i += 128)
        reinterpret_cast<uint32_t *>(psm)[i] = (uint32_t)i * 2654435761u;
    MmaCtx cx;
    mma_init<128>(cx, psm, MMA_PROBE_ROWS, psm + mma_scratch_bytes(MMA_PROBE_ROWS, 128), 512);
    if (threadIdx.x == 0) {
        mbar_init(cx.bar + 192, 1);                      // the probe's own barriers: one completion barrier and one
        mbar_init(cx.bar + 200, 1);                      // per-step commit target per issuer (nobody waits on those)
        mbar_init(cx.bar + 208, 1);
        mbar_init(cx.bar + 216, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_async_smem();
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    if (warp < issuers) {
        const long long t0 = clock64();
        const uint32_t idesc0 = mma_idesc(n_cols);
        for (int it = 0; it < iters; ++it) {
            uint32_t d_tmem = cx.tmem_base + 128u * (uint32_t)warp, a_tmem = cx.tmem_base + 256u + 32u * (uint32_t)(it & 3);
            uint32_t a_lo = mma_desc_lo(smem_u32(cx.ring) + 128u * (uint32_t)(it % ring_segs(128)));
            uint32_t b_lo = mma_desc_lo(smem_u32(cx.brows + (it & 7) * 128)), idesc = idesc0, ebar = cx.bar + 208 + 8 * warp;
            asm volatile("" : "+r"(d_tmem), "+r"(a_tmem), "+r"(a_lo), "+r"(b_lo), "+r"(idesc), "+r"(ebar));
            if (FORM == 0) {
                if (elect_one()) {
                    tc_mma_i8_ts(d_tmem, a_tmem, b_lo, idesc, 1u);
                    tc_mma_i8_ts(d_tmem, a_tmem + 8, b_lo + 2, idesc, 1u);
                    tc_mma_i8_ts(d_tmem, a_tmem + 16, b_lo + 4, idesc, 1u);
                    tc_mma_i8_ts(d_tmem, a_tmem + 24, b_lo + 6, idesc, 1u);
                    tc_commit(ebar);
                }
            } else {
                if (elect_one()) {
                    tc_mma_i8_ss<128>(d_tmem, a_lo, b_lo, idesc, 1u);
                    tc_mma_i8_ss<128>(d_tmem, a_lo + 2, b_lo + 2, idesc, 1u);
                    tc_mma_i8_ss<128>(d_tmem, a_lo + 4, b_lo + 4, idesc, 1u);
                    tc_mma_i8_ss<128>(d_tmem, a_lo + 6, b_lo + 6, idesc, 1u);
                    tc_commit(ebar);
                }
            }
        }
        if (elect_one()) tc_commit(cx.bar + 192 + 8 * warp);
        __syncwarp();
        const bool ok = mbar_wait(cx.bar + 192 + 8 * warp, 0);
        const long long t1 = clock64();
        if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) cycles[warp] = ok ? (unsigned long long)(t1 - t0) : 0ull;
    }
    mma_fini<128>(cx);
}
extern "C" {

unsigned long long mpdiv_mma_probe_macs(int n_cols, int issuers, int iters)
{
    if (iters <= 0 || (issuers != 1 && issuers != 2) || n_cols < 16 || n_cols > 128 || (n_cols & 15) || !device_props())
        return 0ull;
    return (unsigned long long)g_sm_count * issuers * iters * 4ull * 128ull * (unsigned long long)n_cols * 32ull;
}

int mpdiv_mma_probe(int n_cols, int issuers, int iters, int form, unsigned long long *cycles, mpdiv_stream_t stream)
{
    if (!cycles || iters <= 0 || (issuers != 1 && issuers != 2) || n_cols < 16 || n_cols > 128 || (n_cols & 15) ||
        (form != 0 && form != 1))
        return MPDIV_ERR_BAD_ARG;
    if (!device_props()) return MPDIV_ERR_CUDA;
    const int bytes = mma_scratch_bytes(MMA_PROBE_ROWS, 128) + MMA_BAR_BYTES;
    if (set_smem(form ? mma_probe_kernel<1> : mma_probe_kernel<0>, (size_t)bytes) != MPDIV_OK) return MPDIV_ERR_CUDA;
    if (form) mma_probe_kernel<1><<<g_sm_count, 128, bytes, reinterpret_cast<cudaStream_t>(stream)>>>(n_cols, issuers, iters, cycles);
    else mma_probe_kernel<0><<<g_sm_count, 128, bytes, reinterpret_cast<cudaStream_t>(stream)>>>(n_cols, issuers, iters, cycles);
    return cudaGetLastError() == cudaSuccess ? MPDIV_OK : MPDIV_ERR_CUDA;
}

const char *mpdiv_version(void) { return MPDIV_VERSION_STR; }

const char *mpdiv_strerror(int code)
{
    switch (code) {
        case MPDIV_OK: return "ok";
        case MPDIV_ERR_BAD_ARG: return "bad argument (null pointer, non-positive size, misaligned pointer or stride)";
        case MPDIV_ERR_UNSUPPORTED: return "unsupported size (stride above MPDIV_MAX_LIMBS or shared memory budget exceeded)";
        case MPDIV_ERR_CUDA: return "CUDA runtime error";
        case MPDIV_ERR_TOO_LARGE: return "batch larger than MPDIV_NOALLOC_MAX_BATCH: the static scratch of mpdiv_batch_noalloc holds no more";
        default: return "unknown status";
    }
}

}  // extern "C"

#include "mpdiv_api.inl"

// ---------------------------------------------------------------------------------------
// mpdiv_batch_noalloc (include/mpdiv.h): the division for callers that must not allocate
// ---------------------------------------------------------------------------------------
// The one scratch buffer of the division path is the workspace through which the head-of-Refine kernel hands its
// iterates to the division kernel (batch x WMID_STRIDE limbs; mpdiv_batch takes it from a stream-ordered memory
// pool).  Here it is a file-scope device array: every GPU that loads the library holds these
// MPDIV_NOALLOC_MAX_BATCH x 272 x 4 bytes = 4.25 MiB until the process exits.  In host code the NAME of the array is
// a host-side stand-in, not a device address: its device address is looked up once per device with
// cudaGetSymbolAddress (that device current) and that pointer is what the kernels get.
static __device__ __align__(256) limb g_noalloc_wmid[(size_t)MPDIV_NOALLOC_MAX_BATCH * WMID_STRIDE];

namespace {
limb *noalloc_scratch()
{
    static limb *ptr[MAX_DEVICES] = {nullptr};
    std::lock_guard<std::mutex> lk(g_host_mutex);
    if (!ptr[g_dev]) {                                       // g_dev: the current device, set by device_props()
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_wmid) != cudaSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        ptr[g_dev] = static_cast<limb *>(p);
    }
    return ptr[g_dev];
}
}  // namespace

extern "C" int mpdiv_batch_noalloc(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs, uint32_t *q, uint32_t *r,
                                   int batch, mpdiv_stream_t stream)
{
    int rc = check_div_args(u, u_limbs, v, v_limbs, q, r, batch);
    if (rc != MPDIV_OK) return rc;
    if (!aligned16(u) || !aligned16(v) || !aligned16(q) || !aligned16(r)) return MPDIV_ERR_BAD_ARG;
    if (batch > MPDIV_NOALLOC_MAX_BATCH) return MPDIV_ERR_TOO_LARGE;       // the static scratch holds no more rows
    if (!device_props()) return MPDIV_ERR_CUDA;
    Tune tn = tune_of(MPDIV_VARIANT_DEFAULT);
    tn.wmid_fixed = noalloc_scratch();
    if (!tn.wmid_fixed) return MPDIV_ERR_CUDA;
    // Nothing in the scratch has to start at zero: the head kernel writes the row of every instance whose row the
    // division kernel reads (both derive that from the instance's precisions alone, mp_div.cuh head_plan), so what
    // an earlier call left behind is never read.
    return div_dispatch(u, u_limbs, v, v_limbs, q, r, batch, 1, reinterpret_cast<cudaStream_t>(stream), batch, tn);
}
