/*
 * mpdiv.h -- C ABI of libmpdiv.so: batched exact division of midsize unsigned integers on one
 * NVIDIA B200 (sm_100a), after "On GPU Implementation for Multi-Precision Integer Division"
 * (arxiv/paper_2606_06386; citations are lines of the paper text PAPER.md).
 *
 * Method: one division per thread block; quotient by Newton iteration on Watt's whole shifted
 * inverse shinv_h(v) = floor(B^h / v) (Definition 1; Alg. 1-2),
 * then the +-1 quotient / remainder correction of Alg. 3 (Theorem 2 :156-162).
 * B = 2^32.  All arithmetic is exact integer arithmetic.
 *
 * Conventions common to every entry point
 *   - Numbers are little-endian arrays of uint32 limbs: limb j has weight B^j.
 *     Batches are row-major: instance i of an operand with stride s starts at ptr + i*s.
 *     A value shorter than its stride is zero padded at the top; the kernels find the effective
 *     precision themselves ("Prec").
 *   - Pointers of the *_batch functions are DEVICE pointers owned by the caller (PyTorch allocates
 *     them); they must be 16-byte aligned and every stride must be a multiple of 4 limbs.
 *     Outputs must not overlap inputs.  The library never frees caller memory and the *_batch calls
 *     never synchronise the stream: work is enqueued on `stream` and the call returns.  Library-owned
 *     state, all per device, created on first use and never destroyed: the shared-memory attribute of each
 *     kernel, a memory pool for the stream-ordered workspace of mpdiv_batch (see there), the helper
 *     streams and events of mpdiv_batch_host, and three small device words (counters, status).
 *   - Return value: MPDIV_OK, or an error code; nothing is enqueued when an error is returned.
 *     No exception crosses the ABI.  mpdiv_strerror() gives a text for a code.
 *   - Conditions a kernel can only find while it runs (a tensor-core pipeline wait that gave up, a
 *     correction loop that hit its bound, v = 0) do not change the return value of the asynchronous
 *     call; they set sticky bits of a device status word that mpdiv_status() reads.  A caller that
 *     needs certainty polls it once per batch (tests do so after every batch; it must read 0).
 *   - Supported sizes: operand strides up to MPDIV_MAX_OPERAND_LIMBS limbs (2^18 bits, the paper's range,
 *     its ceiling is the shared memory of an SM); the DIVIDEND of mpdiv_batch may have up to
 *     MPDIV_MAX_LIMBS limbs (2^19 bits: dividends above MPDIV_MAX_OPERAND_LIMBS limbs are not held on chip but
 *     streamed from HBM window by window, see mpdiv_batch).  Any effective precision inside the stride,
 *     including 0.
 */
#ifndef MPDIV_H
#define MPDIV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* binary-compatible with cudaStream_t (0 / NULL = the legacy default stream) */
typedef struct CUstream_st *mpdiv_stream_t;

#define MPDIV_MAX_LIMBS 16384          /* u_limbs of mpdiv_batch (default variant) */
#define MPDIV_MAX_OPERAND_LIMBS 8192   /* every other stride: v_limbs, h of shinv_batch, operands of mpmul_batch, and
                                          u_limbs of MPDIV_VARIANT_PRINTED */

enum {
    MPDIV_OK = 0,
    MPDIV_ERR_BAD_ARG = 1,      /* null pointer, non-positive size, misaligned pointer or stride */
    MPDIV_ERR_UNSUPPORTED = 2,  /* stride above MPDIV_MAX_(OPERAND_)LIMBS, or shared memory budget exceeded */
    MPDIV_ERR_CUDA = 3,         /* a CUDA runtime call failed (launch, attribute, copy) */
    MPDIV_ERR_TOO_LARGE = 4     /* mpdiv_batch_noalloc: batch above MPDIV_NOALLOC_MAX_BATCH */
};

/*
 * Division, Alg. 3: for each i < batch
 *     q_i = floor(u_i / v_i),   r_i = u_i - q_i * v_i        (u = q*v + r, 0 <= r < v)
 *   u : batch x u_limbs (device, read)      v : batch x v_limbs (device, read)
 *   q : batch x u_limbs (device, written)   r : batch x v_limbs (device, written)
 * q has stride u_limbs because the quotient of an M-limb by an n-limb number can need M-n+1
 * limbs, and up to M when the divisor is short; both outputs are zero padded.  v_limbs may exceed
 * u_limbs (an instance whose divisor is really longer than its dividend gives q = 0, r = u).
 * v_i = 0 (undefined in the paper) does not trap: q_i is set to all ones, r_i to the
 * low v_limbs limbs of u_i, and the instance is counted in mpdiv_debug_counters.
 * Launches: one kernel, one division per thread block; a throughput batch of the clipped variant
 * (mpdiv_batch_launches() == 2) runs the short-operand head of Refine in a kernel of its own first, one
 * warp per division, and passes its iterate (batch x 272 limbs) through a stream-ordered allocation from a
 * library-owned memory pool of the current device (created on first use, never destroyed; freed rows stay
 * in the pool).  The division kernel is launched behind that head kernel with programmatic stream serialisation:
 * its blocks start while the head still runs and wait for it (griddepcontrol.wait) where they take its rows over.
 * Everything is enqueued on `stream`; nothing synchronises.
 * Rows travel between HBM and shared memory as 1-D bulk asynchronous copies (cp.async.bulk + mbarrier).
 * A batch of at most half as many divisions as the GPU has SMs, of 1024 limbs or more, runs every division on a
 * thread-block cluster of 2-4 CTAs; small numbers in large batches run one division per warp.
 * MPDIV_MAX_OPERAND_LIMBS < u_limbs <= MPDIV_MAX_LIMBS (2^19 bits; v_limbs <= MPDIV_MAX_OPERAND_LIMBS): the dividend
 * stays in HBM.  The quotient is produced t = 2048 limbs at a time (1024 or 512 if shared memory is short) from a
 * window x = r' B^t + (next t limbs of u), r' the running remainder: x < v B^t, so one shifted inverse
 * Shinv(v, k + 1 + t) of t + 2 limbs serves every window, and each window is the division above on a
 * (k + 1 + t)-limb dividend.  An instance whose quotient has at most t limbs is a single window.  Exact like the rest.
 */
int mpdiv_batch(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs,
                uint32_t *q, uint32_t *r, int batch, mpdiv_stream_t stream);

/*
 * mpdiv_batch for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): same inputs, outputs, exact results and default variant as mpdiv_batch, but the one
 * scratch buffer of the path -- the rows through which the head-of-Refine kernel hands its iterates to the
 * division kernel, which mpdiv_batch takes from a stream-ordered memory pool -- is a static device array inside
 * the library: MPDIV_NOALLOC_MAX_BATCH x 272 limbs = 4.25 MiB that every GPU that loads the library holds until
 * the process exits.  The call makes no cudaMalloc / cudaFree / pool call of any kind (its first use on a device
 * looks the array's address up with cudaGetSymbolAddress and sets kernel attributes, host side only).
 *   batch > MPDIV_NOALLOC_MAX_BATCH returns MPDIV_ERR_TOO_LARGE and enqueues nothing: split the batch.
 *   ALL calls on a device share the one array: calls whose kernels may overlap on the GPU (different streams
 *   without an ordering between them, or several host threads) RACE on it and give wrong quotients; calls on one
 *   stream, or ordered by events, are safe.  The array keeps the last call's contents; nothing in it has to start
 *   at zero (every row that is read was written by the same call).
 */
#define MPDIV_NOALLOC_MAX_BATCH 4096
int mpdiv_batch_noalloc(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs,
                        uint32_t *q, uint32_t *r, int batch, mpdiv_stream_t stream);

/*
 * Variants of the method; both return the same exact (q, r).
 *   MPDIV_VARIANT_PRINTED  Alg. 1-3 as printed: full products w*x, u*shinv, v*q and the close product
 *                          v'w mod B^L.  Needs the 2M-limb product on chip:
 *                          strides with u_limbs + v_limbs > 12288 return MPDIV_ERR_UNSUPPORTED.
 *   MPDIV_VARIANT_CLIPPED  the paper's first future-work item: every product
 *                          computes only the limb range the step keeps (top of w*x and u*shinv, middle
 *                          of v'w, bottom of v*q); the +-1 correction of Alg. 3 becomes two bounded
 *                          loops.  About 0.4 M^2 instead of 1.8 M^2 limb products per division.
 * mpdiv_batch uses MPDIV_VARIANT_DEFAULT; shinv_batch returns Theorem 2's value and uses MPDIV_VARIANT_PRINTED.
 *
 * `flags` of the *_ex calls = a variant, optionally OR-ed with tuning switches (for A/B measurements and the
 * tests; none of them changes a result, q and r are exact either way):
 *   MPDIV_FLAG_NO_SEED     Refine starts at l = 2 as printed instead of the 17-digit seed (clipped variant)
 *   MPDIV_FLAG_NO_HEAD     the head of Refine stays inside the division kernel (see mpdiv_batch_launches)
 *   MPDIV_FLAG_NO_MMA      every product of the division runs on the IMAD engine (no tcgen05 range products)
 *   MPDIV_FLAG_NO_CLUSTER  a small batch keeps one block per division (no thread-block cluster per division)
 *   MPDIV_FLAG_CLUSTER(n)  clusters of at most n CTAs, n in {2, 4, 8}, wherever such clusters all run at once (default:
 *                          at most 4, from 1024 limbs up, 2 only from 1536 limbs up)
 *   MPDIV_FLAG_THREADS(n)  block size override, n in {32, 64, 128, 256, 512}
 */
#define MPDIV_VARIANT_PRINTED 0
#define MPDIV_VARIANT_CLIPPED 1
#define MPDIV_VARIANT_DEFAULT MPDIV_VARIANT_CLIPPED
#define MPDIV_VARIANT_MASK 0x0f
#define MPDIV_FLAG_NO_SEED 0x10
#define MPDIV_FLAG_NO_HEAD 0x20
#define MPDIV_FLAG_NO_MMA 0x40
#define MPDIV_FLAG_NO_CLUSTER 0x80
#define MPDIV_FLAG_THREADS(n) ((n) == 64 ? 0x100 : (n) == 128 ? 0x200 : (n) == 256 ? 0x300 : (n) == 512 ? 0x400 : (n) == 32 ? 0x500 : 0)
#define MPDIV_FLAG_THREADS_MASK 0x700
#define MPDIV_FLAG_CLUSTER(n) ((n) == 2 ? 0x1000 : (n) == 4 ? 0x2000 : (n) == 8 ? 0x3000 : 0)
#define MPDIV_FLAG_CLUSTER_MASK 0x3000
int mpdiv_batch_ex(const uint32_t *u, int u_limbs, const uint32_t *v, int v_limbs,
                   uint32_t *q, uint32_t *r, int batch, int flags, mpdiv_stream_t stream);

/*
 * Multiplication, the unit of the paper's cost model (PAPER.md:105-106 MULT / MULTMOD, :166, :186):
 *     c_i = (a_i * b_i) mod B^c_limbs
 *   a : batch x a_limbs, b : batch x b_limbs (device, read);  c : batch x c_limbs (device, written)
 * c_limbs = a_limbs + b_limbs gives the full product; a smaller c_limbs gives the truncated
 * ("close") product, whose skipped limb products are not computed.  c_limbs <= a_limbs + b_limbs.
 */
int mpmul_batch(const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs,
                uint32_t *c, int c_limbs, int batch, mpdiv_stream_t stream);

/*
 * Same product with an explicit engine.
 *   MPMUL_ENGINE_IMAD    the block-level schoolbook multiplier on IMAD.WIDE (what mpmul_batch runs; the unit
 *                        of the paper's cost model).
 *   MPMUL_ENGINE_TENSOR  the product as an int8 tcgen05 GEMM: byte convolution with Toeplitz tiles generated
 *                        on the fly, accumulators in TMEM (csrc/mp_mma.cuh).  The north star allows tensor
 *                        cores only where measured faster: bench.py times both engines; mpdiv_batch uses this
 *                        engine for its large range products from 2^16 bits up (throughput batches).
 *                        MPDIV_ERR_UNSUPPORTED when the request needs more than 512 output blocks of 32 limbs
 *                        or does not fit shared memory.
 */
#define MPMUL_ENGINE_IMAD 0
#define MPMUL_ENGINE_TENSOR 1
int mpmul_batch_ex(const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs,
                   uint32_t *c, int c_limbs, int batch, int engine, mpdiv_stream_t stream);

/*
 * Whole shifted inverse as the division uses it, Alg. 1-2 and Theorem 2
 * (PAPER.md:160):   w_i = floor(B^h / v_i) + lambda_i,  lambda_i in {0, 1}
 * i.e. the UNCORRECTED Newton result of the algorithm as printed (MPDIV_VARIANT_PRINTED), so that its time
 * is the "2..4 multiplications" of the cost model.
 *   v : batch x v_limbs (device, read);  w : batch x w_limbs (device, written),
 * w_limbs >= h + 1, 1 <= h <= MPDIV_MAX_OPERAND_LIMBS.  v_i = 0 gives w_i = all ones (status bit MPDIV_STATUS_V_ZERO).
 */
int shinv_batch(const uint32_t *v, int v_limbs, int h, uint32_t *w, int w_limbs,
                int batch, mpdiv_stream_t stream);
/*
 * Same with explicit flags (variant | tuning switches, see mpdiv_batch_ex).  MPDIV_VARIANT_CLIPPED is the
 * shifted inverse as the default division computes it (clipped products, "+1" loop, 17-digit seed): it
 * returns floor(B^h / v) + lambda with lambda in {-1, 0, 1}, one unit wider than Theorem 2; Div's bounded
 * correction loops absorb it.
 */
int shinv_batch_ex(const uint32_t *v, int v_limbs, int h, uint32_t *w, int w_limbs,
                   int batch, int flags, mpdiv_stream_t stream);

/*
 * The linear-cost building blocks of the method on their own (PAPER.md 3.2-3.3), exported so that they can
 * be unit-tested: each is the block-level map-scan-map the division uses internally.
 *   a : batch x a_limbs, b : batch x b_limbs (device, read);  out : batch x out_limbs, flag : batch words
 *   (device, written).  shift counts whole limbs; shift_n(x) = floor(x * B^n) (Definition 1).
 *   MPLINOP_ADD    out = (a + shift_n(b)) mod B^out_limbs,  flag = carry out
 *   MPLINOP_SUB    out = (a - shift_n(b)) mod B^out_limbs,  flag = borrow out = (a < shift_n(b)) when both fit
 *                  in out_limbs: subtraction with the borrow scan and the less-than test (:331-335, :343-440)
 *   MPLINOP_NEG    out = B^shift - a (a < B^shift <= B^out_limbs), the B^L - P of PowDiff (:117, :329); flag = carry
 *   MPLINOP_SHIFT  out = shift_n(a) truncated to out_limbs (n = shift, either sign)    (:204)
 *   MPLINOP_PREC   flag = prec(a) = number of significant limbs (:135);  out = a
 *   MPLINOP_ANY    flag = 1 when a limb of a at index >= shift is non-zero (the comparison with B^h, :329); out = a
 */
enum { MPLINOP_ADD = 0, MPLINOP_SUB = 1, MPLINOP_NEG = 2, MPLINOP_SHIFT = 3, MPLINOP_PREC = 4, MPLINOP_ANY = 5 };
int mplinop_batch(int op, const uint32_t *a, int a_limbs, const uint32_t *b, int b_limbs, int shift,
                  uint32_t *out, int out_limbs, uint32_t *flag, int batch, mpdiv_stream_t stream);

/*
 * Host-buffer form of mpdiv_batch for end-to-end use: u, v, q, r are HOST pointers (pinned memory
 * recommended; pageable memory works but serialises the copies); `workspace` is a caller-owned DEVICE
 * buffer of at least mpdiv_host_workspace_bytes(u_limbs, v_limbs, batch) bytes.  The batch is cut into
 * up to 16 chunks of about one division per SM; the H2D copy of chunk i+1 and the D2H copy of chunk i-1
 * overlap the division of chunk i, and the chunk kernels rotate over four streams so that consecutive
 * chunks share the SMs as the blocks of one launch would (six library-owned helper streams, created on
 * first use, never destroyed).  Everything is ordered after the work already enqueued on `stream`, and `stream`
 * completes only after the last D2H copy: the caller synchronises `stream` and reads q, r.
 * The helper streams and events belong to the current device; calls from several host threads are serialised
 * by a lock around the enqueue.  When an error is returned part of the batch may have been enqueued: the call
 * waits for that work before it returns, so the buffers are free again.
 */
size_t mpdiv_host_workspace_bytes(int u_limbs, int v_limbs, int batch);
int mpdiv_batch_host(const uint32_t *u_host, int u_limbs, const uint32_t *v_host, int v_limbs,
                     uint32_t *q_host, uint32_t *r_host, int batch,
                     void *workspace, size_t workspace_bytes, mpdiv_stream_t stream);

/*
 * Integer-multiply roofline probe: every thread of a full-occupancy grid runs
 * `iters` rounds of independent 32x32+64 multiply-accumulate chains (kind 0: IMAD.WIDE with carry
 * chain, the instruction the multiplier uses; kind 1: plain mad.lo 32-bit), no memory traffic.
 * Writes one checksum word per thread to `sink` (device, >= mpdiv_imad_probe_threads() words) and
 * stores the number of limb products issued per launch in *products (host).  Time it with events.
 */
int mpdiv_imad_probe_threads(void);
int mpdiv_imad_probe(uint32_t *sink, int kind, int iters, unsigned long long *products,
                     mpdiv_stream_t stream);

/*
 * Tensor-core issue-rate probe and int8 roofline probe: one 128-thread block per SM in which
 * `issuers` warps (1 or 2) each issue `iters` steps of four tcgen05.mma.kind::i8 (M = 128, K = 32, N = n_cols,
 * 16 <= n_cols <= 128, multiple of 16) into their own accumulator columns, the way the multiplier issues them.
 * form 0: the A operand in tensor memory (the pure rate of the pipe); form 1: A read from shared memory through
 * the overlapped Toeplitz descriptor of csrc/mp_mma.cuh (what the multiplier issues: 32 cycles of shared-memory
 * bandwidth per instruction, so max(32 + n_cols/4, n_cols/2) cycles).
 * cycles (DEVICE pointer, 2 words): SM cycles block 0's warp w needed for its 4 * iters instructions, 0 if a
 * bounded wait gave up.  The tensor core needs n_cols / 2 cycles per instruction; what a single warp measures
 * above that is its own issue path.  One launch executes  SMs x issuers x iters x 4 x 128 x n_cols x 32
 * u8 x u8 multiply-accumulates (mpdiv_mma_probe_macs); timed with events at n_cols = 128 and two issuers it
 * gives the measured peak of the tensor pipe for this data type.  Asynchronous on `stream`.
 */
unsigned long long mpdiv_mma_probe_macs(int n_cols, int issuers, int iters);
int mpdiv_mma_probe(int n_cols, int issuers, int iters, int form, unsigned long long *cycles, mpdiv_stream_t stream);

/*
 * Status word of the current device: sticky bits set by the kernels since the last reset.  Synchronises
 * `stream`, stores the bits in *flags, clears them when `reset` is non-zero.  0 = every result delivered so
 * far is exact.
 *   MPDIV_STATUS_MMA_WAIT    a bounded wait of the tensor-core pipeline gave up; the block recomputed that
 *                            product on the IMAD engine and stopped using the tensor core (results are still
 *                            exact, the bit reports a protocol or scheduling fault)
 *   MPDIV_STATUS_CORR_BOUND  a correction loop of Div hit its bound of 64 steps: that q, r is NOT exact
 *   MPDIV_STATUS_REM_RANGE   clipped variant: the remainder estimate u - v*q0' left the range the
 *                            mod-B^(k+3) arithmetic assumes (its top limb is neither 0 nor all ones): NOT exact
 *   MPDIV_STATUS_V_ZERO      a divisor was zero (undefined): q = all ones, r = low limbs of u
 *   MPDIV_STATUS_IO_WAIT     a bounded wait for a bulk copy of an operand row gave up: NOT exact
 */
#define MPDIV_STATUS_MMA_WAIT 1u
#define MPDIV_STATUS_CORR_BOUND 2u
#define MPDIV_STATUS_REM_RANGE 4u
#define MPDIV_STATUS_V_ZERO 8u
#define MPDIV_STATUS_IO_WAIT 16u
int mpdiv_status(mpdiv_stream_t stream, unsigned int *flags, int reset);

/*
 * Debug counters accumulated by every mpdiv_batch / shinv_batch launch since the last reset
 * (a few device-side atomics per division on a library-owned buffer; reading them synchronises `stream`):
 *   out[0] instances with exactly one delta = -1 correction (u < v*q0)
 *   out[1] instances with exactly one delta = +1 correction
 *   out[2] instances needing more than one +1 step (printed variant: outside Theorem 2, expected 0;
 *          clipped variant: allowed, the clipped quotient estimate may be one lower)
 *   out[3] one-limb divisors      out[4] u < v early exits      out[5] v = 0 instances
 *   out[6] Newton steps that took the negative branch of PowDiff (sign = 0)
 *   out[7] divisors that are an exact power of B (Alg. 1 line 9)
 *   out[8] 8x8-limb tile products executed (x 64 = limb products issued, tile padding included)
 *   out[9] instances needing more than one -1 step      out[10] instances whose correction loops hit
 *          their bound of 64 (result not exact; expected 0)      out[11] Newton steps that ran clipped
 *   out[12] range products that ran on the tensor core (mp_mma.cuh)      out[13] bit mask of tensor-core
 *          pipeline waits that gave up (expected 0)
 *   out[14] add-back steps of the seed's long division (Knuth D6)      out[15] Shinv calls that started
 *          Refine from the 17-digit seed (mpdiv_seed_batch)
 *   out[16] tensor-core work: sum over range products of (MMA steps x accumulator columns); x 16384 = the
 *          u8 x u8 multiply-accumulates the tensor pipe executed (4 instructions of M = 128, K = 32 per step)
 *   out[17] divisions that ran on a thread-block cluster      out[18] quotient windows of the chunked form (dividends above MPDIV_MAX_OPERAND_LIMBS
 *          limbs)      out[19] cycles the tensor unit is occupied by the issued tcgen05.mma (operand fetch from shared
 *          memory included: max(32 + N/4, N/2) per instruction of N columns), summed over blocks      out[20..23] reserved (0)
 */
#define MPDIV_NUM_COUNTERS 24
int mpdiv_debug_counters(unsigned long long out[MPDIV_NUM_COUNTERS], int reset, mpdiv_stream_t stream);

/*
 * The seed of Refine (clipped variant, csrc/mp_div.cuh warp_seed): for each divisor v >= B,
 *      w[i] = floor(B^38 / D),  D = floor(v * B^19 / B^k),  k = prec(v) - 1
 * i.e. the exact quotient of B^38 by the top 20 limbs of v, which stands in for the first four Refine
 * iterations (Alg. 1 lines 19-25, l = 2 -> 17) when h - k >= 17.  One warp per divisor,
 * schoolbook long division with one limb per lane.  Exposed so that the tests can pin the routine on its own.
 *   v   device, batch x v_limbs limbs, little endian          w   device, batch x 24 limbs (20 significant)
 * A divisor with fewer than two significant limbs yields 24 zero limbs.
 */
int mpdiv_seed_batch(const uint32_t *v, int v_limbs, uint32_t *w, int batch, mpdiv_stream_t stream);

/*
 * Kernels one mpdiv_batch_ex call of this shape launches: 1, or 2 when the head of Refine runs in its own
 * kernel (clipped variant, u_limbs >= 512, more divisions than the latency-oriented kernel takes: the seed
 * and the Refine iterations up to l = 129 then run one warp per division ahead of the division kernel and
 * hand their iterate over in a stream-ordered workspace from a library-owned memory pool).  0 on bad arguments.
 */
int mpdiv_batch_launches(int u_limbs, int batch, int flags);

/* "mpdiv <version> sm_100a ..." */
const char *mpdiv_version(void);
const char *mpdiv_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* MPDIV_H */
