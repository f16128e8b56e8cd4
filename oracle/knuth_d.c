/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code with the CUDA library
 * (paper_2606_06386_b200/csrc): no headers, helpers, tables or constants in common.
 *
 * What the hot path of arxiv/paper_2606_06386 computes, as plain definitions:
 *
 *   orc_divmod   (q, r) with u = q*v + r, 0 <= r < v      PAPER.md:131-133 (Alg. 3 output)
 *   orc_shinv    floor(B^h / v)                            PAPER.md:61-66 (Definition 1, shinv_h)
 *   orc_mul      (a*b) mod B^cn                            PAPER.md:105-106 (MULT / MULTMOD)
 *
 * with B = 2^32 and little-endian limbs.  Division is Knuth's
 * Algorithm D (knuth_d_impl.h); shinv is that same routine applied to u = B^h;
 * multiplication is the schoolbook double loop.  Everything is exact integer
 * arithmetic: parity with the CUDA path is bit-for-bit.
 *
 * Pins (tests/test_oracle_pins.py): the paper's Examples 1-2,
 * shinv_15(27183) and shinv_3(8), exhaustive brute force at a
 * test-only base 16 against native C division, CPython's divmod on random big
 * integers, the invariants q*v + r = u and r < v, and closed forms
 * (u < v, u = v*k, v = B^k, v = B^k - 1, v = 1, u = v).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define LB 32
#define FN(name) orc32_##name
#include "knuth_d_impl.h"
#undef LB
#undef FN

#define LB 4
#define FN(name) orc4_##name
#include "knuth_d_impl.h"
#undef LB
#undef FN

/* (q, r) = (floor(u/v), u mod v), base 2^32.  Status: 0 ok, 1 v == 0, 2 overflow of q/r, 3 no memory. */
int orc_divmod(const uint32_t *u, int un, const uint32_t *v, int vn,
               uint32_t *q, int qn, uint32_t *r, int rn)
{
    return orc32_divmod(u, un, v, vn, q, qn, r, rn);
}

/* Same routine at the test-only base 16 (one 4-bit limb per uint32_t). */
int orc_divmod_base16(const uint32_t *u, int un, const uint32_t *v, int vn,
                      uint32_t *q, int qn, uint32_t *r, int rn)
{
    return orc4_divmod(u, un, v, vn, q, qn, r, rn);
}

/* Batch form: instance i uses u + i*un, v + i*vn, q + i*qn, r + i*rn.  Returns the first non-zero status. */
int orc_divmod_batch(const uint32_t *u, int un, const uint32_t *v, int vn,
                     uint32_t *q, int qn, uint32_t *r, int rn, int batch)
{
    int i, st = 0;
    for (i = 0; i < batch; i++) {
        int s = orc32_divmod(u + (size_t)i * un, un, v + (size_t)i * vn, vn,
                             q + (size_t)i * qn, qn, r + (size_t)i * rn, rn);
        if (s != 0 && st == 0) st = s;
    }
    return st;
}

/* c[0..cn) = (a*b) mod B^cn -- schoolbook double loop. */
int orc_mul(const uint32_t *a, int an, const uint32_t *b, int bn, uint32_t *c, int cn)
{
    int i, j;
    for (i = 0; i < cn; i++) c[i] = 0;
    for (i = 0; i < an && i < cn; i++) {
        uint64_t carry = 0;
        uint64_t ai = a[i];
        for (j = 0; j < bn && i + j < cn; j++) {
            uint64_t t = ai * b[j] + c[i + j] + carry;
            c[i + j] = (uint32_t)t;
            carry = t >> 32;
        }
        for (j = i + bn; carry != 0 && j < cn; j++) {
            uint64_t t = (uint64_t)c[j] + carry;
            c[j] = (uint32_t)t;
            carry = t >> 32;
        }
    }
    return 0;
}

int orc_mul_batch(const uint32_t *a, int an, const uint32_t *b, int bn, uint32_t *c, int cn, int batch)
{
    int i;
    for (i = 0; i < batch; i++)
        orc_mul(a + (size_t)i * an, an, b + (size_t)i * bn, bn, c + (size_t)i * cn, cn);
    return 0;
}

/* w[0..wn) = floor(B^h / v) (Definition 1): Algorithm D applied to u = B^h. */
int orc_shinv(const uint32_t *v, int vn, int h, uint32_t *w, int wn)
{
    uint32_t *pw = (uint32_t *)calloc((size_t)h + 1, sizeof(uint32_t));
    uint32_t *rem = (uint32_t *)calloc((size_t)vn, sizeof(uint32_t));
    int st;
    if (!pw || !rem) { free(pw); free(rem); return 3; }
    pw[h] = 1;
    st = orc32_divmod(pw, h + 1, v, vn, w, wn, rem, vn);
    free(pw);
    free(rem);
    return st;
}

int orc_shinv_batch(const uint32_t *v, int vn, int h, uint32_t *w, int wn, int batch)
{
    int i, st = 0;
    for (i = 0; i < batch; i++) {
        int s = orc_shinv(v + (size_t)i * vn, vn, h, w + (size_t)i * wn, wn);
        if (s != 0 && st == 0) st = s;
    }
    return st;
}
