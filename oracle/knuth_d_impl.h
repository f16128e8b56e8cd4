/*
 * ORACLE (test infrastructure only) -- body of the long-division routine,
 * written once and instantiated for two limb widths by knuth_d.c:
 *
 *   LB = 32 : the real oracle, base B = 2^32 (the limb size BASELINE.json fixes);
 *   LB = 4  : a test-only small base B = 16 so that exhaustive brute force over
 *             tiny operands reaches the rare branches of Algorithm D (qhat
 *             correction, add-back), which at B = 2^32 fire with probability ~2/B.
 *
 * What it computes (Alg. 3 "Output: (q, r) with u = q*v + r,
 * r < v"): the Euclidean quotient and remainder of unsigned integers.  The method
 * of the paper reaches exactly this value (Theorem 2 + the corrections of Alg. 3,
 * PAPER.md:141-148, :156-162), so the oracle is the plain definition, computed by
 * textbook long division (Knuth, TAOCP vol. 2, 4.3.1, Algorithm D), NOT by the
 * paper's Newton / shifted-inverse method.  Nothing here is shared with the CUDA path.
 *
 * Limbs are little-endian (index 0 least significant) and are stored
 * one per uint32_t whatever LB is; a limb value is < 2^LB.
 *
 * The includer defines LB and FN(name).
 */

/* number of significant limbs ("prec") */
static int FN(prec)(const uint32_t *a, int n)
{
    while (n > 0 && a[n - 1] == 0) n--;
    return n;
}

/*
 * q[0..qn) = floor(u / v), r[0..rn) = u mod v, both zero padded.
 * Returns 0 on success, 1 if v == 0, 2 if q or r does not fit, 3 on malloc failure.
 */
static int FN(divmod)(const uint32_t *u, int un, const uint32_t *v, int vn,
                      uint32_t *q, int qn, uint32_t *r, int rn)
{
    const uint64_t BASE = (uint64_t)1 << LB;
    const uint64_t MASK = BASE - 1;
    int m = FN(prec)(u, un);   /* significant limbs of the dividend */
    int n = FN(prec)(v, vn);   /* significant limbs of the divisor  */
    int i, j;

    if (n == 0) return 1;
    for (i = 0; i < qn; i++) q[i] = 0;
    for (i = 0; i < rn; i++) r[i] = 0;

    if (m < n) {                       /* u < v: q = 0, r = u */
        if (m > rn) return 2;
        for (i = 0; i < m; i++) r[i] = u[i];
        return 0;
    }
    if (n == 1) {                      /* short division by one limb */
        uint64_t rem = 0, d = v[0];
        for (i = m - 1; i >= 0; i--) {
            uint64_t cur = (rem << LB) | u[i];
            uint64_t qd = cur / d;
            rem = cur % d;
            if (qd != 0 && i >= qn) return 2;
            if (i < qn) q[i] = (uint32_t)qd;
        }
        if (rem != 0 && rn < 1) return 2;
        if (rn >= 1) r[0] = (uint32_t)rem;
        return 0;
    }

    /* D1: normalise so that the top divisor limb has its high bit set */
    {
        uint32_t *un_ = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(m + 1));
        uint32_t *vn_ = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)n);
        int s = 0, status = 0;
        if (!un_ || !vn_) { free(un_); free(vn_); return 3; }
        while ((((uint64_t)v[n - 1] << s) & (BASE >> 1)) == 0) s++;

        for (i = n - 1; i > 0; i--)
            vn_[i] = (uint32_t)((((uint64_t)v[i] << s) | ((uint64_t)v[i - 1] >> (LB - s))) & MASK);
        vn_[0] = (uint32_t)(((uint64_t)v[0] << s) & MASK);

        un_[m] = (uint32_t)((uint64_t)u[m - 1] >> (LB - s));   /* s == 0 gives 0 since u[m-1] < 2^LB */
        for (i = m - 1; i > 0; i--)
            un_[i] = (uint32_t)((((uint64_t)u[i] << s) | ((uint64_t)u[i - 1] >> (LB - s))) & MASK);
        un_[0] = (uint32_t)(((uint64_t)u[0] << s) & MASK);

        /* D2..D7: one quotient limb per step, most significant first */
        for (j = m - n; j >= 0; j--) {
            /* D3: estimate qhat from the top two dividend limbs over the top divisor limb */
            uint64_t num = ((uint64_t)un_[j + n] << LB) | un_[j + n - 1];
            uint64_t qhat = num / vn_[n - 1];
            uint64_t rhat = num % vn_[n - 1];
            int64_t borrow;
            uint64_t carry;

            while (qhat >= BASE ||
                   qhat * vn_[n - 2] > ((rhat << LB) | un_[j + n - 2])) {
                qhat--;
                rhat += vn_[n - 1];
                if (rhat >= BASE) break;
            }

            /* D4: multiply and subtract  un_[j..j+n] -= qhat * vn_[0..n) */
            borrow = 0;
            carry = 0;
            for (i = 0; i < n; i++) {
                uint64_t p = qhat * vn_[i] + carry;
                int64_t t;
                carry = p >> LB;
                t = (int64_t)un_[i + j] - borrow - (int64_t)(p & MASK);
                un_[i + j] = (uint32_t)((uint64_t)t & MASK);
                borrow = (t < 0) ? 1 : 0;
            }
            {
                int64_t t = (int64_t)un_[j + n] - borrow - (int64_t)carry;
                un_[j + n] = (uint32_t)((uint64_t)t & MASK);
                borrow = (t < 0) ? 1 : 0;
            }

            /* D5/D6: qhat was one too large: add the divisor back */
            if (borrow) {
                uint64_t c = 0;
                qhat--;
                for (i = 0; i < n; i++) {
                    uint64_t t = (uint64_t)un_[i + j] + vn_[i] + c;
                    un_[i + j] = (uint32_t)(t & MASK);
                    c = t >> LB;
                }
                un_[j + n] = (uint32_t)(((uint64_t)un_[j + n] + c) & MASK);
            }

            if (qhat != 0 && j >= qn) { status = 2; break; }
            if (j < qn) q[j] = (uint32_t)qhat;
        }

        /* D8: the remainder is un_[0..n) shifted back right by s */
        if (status == 0) {
            for (i = 0; i < n; i++) {
                uint64_t lo = (uint64_t)un_[i] >> s;
                uint64_t hi = (i + 1 < n) ? (((uint64_t)un_[i + 1] << (LB - s)) & MASK) : 0;
                uint32_t limb = (uint32_t)((s == 0) ? un_[i] : (lo | hi));
                if (limb != 0 && i >= rn) { status = 2; break; }
                if (i < rn) r[i] = limb;
            }
        }
        free(un_);
        free(vn_);
        return status;
    }
}
