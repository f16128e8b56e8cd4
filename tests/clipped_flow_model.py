"""Python-integer replay of the DEFAULT division flow of libmpdiv.so (MPDIV_VARIANT_CLIPPED), step by step.

Why this exists.  Theorem 2 bounds the error of the algorithm AS PRINTED, and its proof is in a
thesis that is not available here.  The default variant goes beyond the printed algorithm (clipped products --
the paper's own future work, PAPER.md:507, :511, :542 --, one trailing Refine iteration instead of two, a 17-digit
seed, 32-limb windows on the tensor-core engine), so its exactness rests on bounds of its own: the shifted inverse
is within one unit (lambda in {-1, 0, 1}), the quotient estimate within a few units, and the remainder estimate
u - v*q0' inside (-B^(k+2), B^(k+2)), the range of the mod-B^(k+3) remainder arithmetic.  This module recomputes
the flow with unbounded Python integers, window for window as csrc/mp_div.cuh and csrc/mpdiv_api.inl code it, and
tests/test_clipped_flow_model.py asserts those bounds over directed inputs and a sweep over (k, h - k).

It is test infrastructure.  It shares nothing with oracle/ (Knuth D, the definition of q and r) or with csrc/: the
only arithmetic below is Python's int.  What it mirrors (file: function):
  mp_div.cuh: refine_iters, head_plan (only to know which iterations may use the tensor-core windows), warp_seed
              (its defining formula floor(B^38 / D)), refine_step, shinv_block
  mp_mul.cuh: mul_low / mul_range (tile diagonals Klo <= K < Khi of 8x8-limb tiles: the omitted part E is the sum of
              the tile products with I + J < Klo)
  mp_mma.cuh: mma_mul_range (output blocks of 32 limbs: the omitted part E is the byte columns t < 128 dlo)
  mpdiv_api.inl: mpdiv_kernel, clipped branch (u*shinv from column h - 9 / block (h-1)/32, v*q0 mod B^rlen, the
              two correction loops)
"""
from __future__ import annotations

B = 1 << 32
TILE = 8
G = 2                      # guard digits (Alg. 1 line 16)
SEED_L, SEED_ITERS, SEED_LIMBS = 17, 4, 20
HEAD_L = 129
CORR_MAX = 64


def ru(x: int, m: int) -> int:
    return (x + m - 1) // m * m


def prec(x: int) -> int:
    """Number of significant limbs."""
    return (x.bit_length() + 31) // 32


def low(x: int, limbs: int) -> int:
    return x & ((1 << (32 * limbs)) - 1) if limbs > 0 else 0


# ------------------------------------------------------------------------------------------------
# the two multiplier engines' range products
# ------------------------------------------------------------------------------------------------
def omitted_tiles(a: int, b: int, klo: int) -> int:
    """E of mul_range: the sum of the 8x8-limb tile products (I, J) with I + J < klo."""
    e = 0
    i = 0
    while i < klo and (a >> (256 * i)):
        a_i = (a >> (256 * i)) & ((1 << 256) - 1)
        e += (a_i * low(b, TILE * (klo - i))) << (256 * i)
        i += 1
    return e


def omitted_byte_columns(a: int, b: int, t0: int) -> int:
    """E of mma_mul_range: the byte columns t = x + y < t0 of the byte convolution of a and b."""
    e = 0
    x = 0
    ab = a.to_bytes((a.bit_length() + 7) // 8 or 1, "little")
    for x, ax in enumerate(ab):
        if x >= t0:
            break
        if ax:
            e += (ax * (b & ((1 << (8 * (t0 - x))) - 1))) << (8 * x)
    return e


def range_imad(a: int, na: int, b: int, nb: int, klo: int, khi: int):
    """mul_range<T>(A, na, B, nb, Klo, Khi): returns (value stored from limb 8*Klo, limbs stored)."""
    Na, Nb = ru(na, TILE) // TILE, ru(nb, TILE) // TILE
    kfull = Na + Nb
    kc = min(khi, kfull)
    val = low(a * b - omitted_tiles(a, b, klo), TILE * kc) >> (32 * TILE * klo)
    return val, TILE * max(kc - klo, 0)


def range_mma(a: int, na: int, b: int, nb: int, dlo: int, dhi: int):
    """mma_mul_range<T>(A, na, B, nb, dlo, dhi): (value stored from limb 32*dlo, limbs stored)."""
    dhi = min(dhi, (na + nb + 31) // 32)
    n = dhi - dlo
    if n <= 0:
        return None
    val = low(a * b - omitted_byte_columns(a, b, 128 * dlo), 32 * dhi) >> (32 * 32 * dlo)
    return val, 32 * n


# ------------------------------------------------------------------------------------------------
# Refine
# ------------------------------------------------------------------------------------------------
def refine_iters(H: int, clip: bool = True) -> int:
    return ((H - 2).bit_length() if H - 1 > 1 else 0) + (1 if clip else 2)


def head_plan(H: int, iters: int):
    if H < SEED_L:
        return 0
    l, it = SEED_L, SEED_ITERS
    while l <= HEAD_L and it + 2 < iters:
        m = min(H + 1 - l, l)
        l += m - 1
        it += 1
    return 0 if it == SEED_ITERS else it


class Trace:
    """What the tests look at: per-step records and the ranges reached."""

    def __init__(self):
        self.steps = []
        self.clipped_steps = 0
        self.mma_products = 0
        self.sign_neg = 0


def refine_step(v: int, k: int, H: int, l: int, wlen: int, wc: int, use_mma, tr: Trace):
    """One iteration of Refine with Step and PowDiff inlined, clipped variant (mp_div.cuh: refine_step)."""
    m = min(H + 1 - l, l)
    s = max(0, k - 2 * l + 1 - G) & ~3
    vp = v >> (32 * s)
    pv = k + 1 - s
    hp = k + l + m - s + G
    hpp = hp - m
    bound = min(wlen, l + G + 2)
    assert wc < (1 << (32 * bound)), "iterate longer than l + g + 2 limbs"
    w = wc
    pw = prec(w)
    d = hp - 2 * m
    L = pv + pw - (l - G) + 1
    c = 0
    if L >= hpp:
        p = vp * w
        positive = (p >> (32 * hpp)) == 0
        x = (1 << (32 * hpp)) - p if positive else p - (1 << (32 * hpp))
    else:
        cx = d + 1 - pw
        klo2 = (cx - 9) // 8 - 1 if cx >= 25 else 0
        if klo2 <= 0:
            p = low(vp * w, L)                                   # close product, exact low L limbs
            positive = (p >> (32 * (L - 1))) != 0
            x = (1 << (32 * L)) - p if positive else p
        else:
            tr.clipped_steps += 1
            dlo = (cx - 1) // 32
            got = range_mma(vp, pv, w, pw, dlo, (L + 31) // 32) if use_mma("vw") else None
            if got is not None:
                c = 32 * dlo
                tr.mma_products += 1
                pval = got[0]
            else:
                c = TILE * klo2
                pval = range_imad(vp, pv, w, pw, klo2, (L + TILE - 1) // TILE)[0]
            xl = L - c
            pval = low(pval, xl)
            positive = (pval >> (32 * (xl - 1))) != 0
            x = (pval ^ ((1 << (32 * xl)) - 1)) if positive else pval      # ~P, no "+ 1": below the window's resolution
    if not positive:
        tr.sign_neg += 1
    xl = prec(x)

    nlen = ru(l + m + G + 2, TILE)
    wsh = low(w, wlen) << (32 * (m - 1))
    if xl == 0:
        wn = low(wsh, nlen)
    else:
        dd = d + 1 - c
        klo1 = (dd - 9) // TILE if dd >= 17 else 0
        exact = klo1 == 0 and c == 0
        got = None
        if dd >= 33 and use_mma("wx"):
            got = range_mma(w, pw, x, xl, (dd - 1) // 32, 1 << 20)
        if got is not None:
            tr.mma_products += 1
            pval, tl = got
            off = dd - 32 * ((dd - 1) // 32)
            exact = False
        elif klo1 == 0:
            pval, tl, off = w * x, ru(pw, TILE) + ru(xl, TILE), dd
        else:
            pval, tl = range_imad(w, pw, x, xl, klo1, 1 << 20)
            off = dd - TILE * klo1
        assert off >= 0
        t = low(pval, tl) >> (32 * off)
        if positive:
            wn = low(wsh + t, nlen)
        else:
            borrow = 1 if (exact and low(pval, min(dd, tl)) != 0) else 0
            wn = low(wsh - t - borrow, nlen)
    tr.steps.append({"l": l, "m": m, "positive": positive, "c": c})
    return wn, l + m - 1, nlen


def shinv(v: int, h: int, use_mma=lambda kind: False, seed=True, seed_delta: int = 0, tr: Trace | None = None) -> int:
    """shinv_block<T>(V, k, h, ..., clip = true): the shifted inverse as the default division computes it.
    v >= B (one-limb divisors are mapped to two-limb ones by the caller).  seed_delta perturbs the seed."""
    tr = tr if tr is not None else Trace()
    k = prec(v) - 1
    assert k >= 1
    low_nz = low(v, k) != 0
    vtop = v >> (32 * k)
    pow_b = vtop == 1 and not low_nz
    if k > h or (k == h and not pow_b):
        return 0
    if not pow_b and k == h - 1 and (vtop > 0x80000000 or (vtop == 0x80000000 and low_nz)):
        return 1
    if pow_b:
        return 1 << (32 * (h - k))
    H = max(h - k, 2)
    iters = refine_iters(H)
    head_end = head_plan(H, iters) if seed else 0
    if seed and H >= SEED_L:
        D = (v >> (32 * (k - 19))) if k >= 19 else (v << (32 * (19 - k)))
        w = (1 << (32 * 38)) // D + seed_delta
        l, wlen, it0 = SEED_L, 24, SEED_ITERS
    else:
        V2 = v >> (32 * (k - 1))
        w = ((1 << 96) // V2) << (32 * G)
        l, wlen, it0 = 2, TILE, 0
    for it in range(it0, iters):
        # the head kernel and the narrow phase run refine_step<32> without the engine
        allow = (lambda kind: use_mma(kind)) if it >= head_end else (lambda kind: False)
        w, l, wlen = refine_step(v, k, H, l, wlen, w, allow, tr)
    sh = G + (H - (h - k))
    res = low(w, wlen) >> (32 * sh)
    return low(low(res, ru(h - k + 2, TILE)), h - k + 1)             # psh = top_prec(WA, nw), nw = h - k + 1


# ------------------------------------------------------------------------------------------------
# Div
# ------------------------------------------------------------------------------------------------
class DivResult:
    __slots__ = ("q", "r", "lam", "q0", "delta", "rem_estimate", "k", "minus", "plus", "rem_top_ok", "trace")


def divide(u: int, v: int, use_mma=lambda kind: False, seed=True, seed_delta: int = 0) -> DivResult:
    """mpdiv_kernel, clipped branch.  Returns the final (q, r) and the intermediate quantities the bounds are about."""
    res = DivResult()
    tr = Trace()
    res.trace = tr
    h, pv = prec(u), prec(v)
    assert v > 0
    if pv > h:
        res.q, res.r, res.lam, res.q0, res.delta, res.rem_estimate = 0, u, 0, 0, 0, u
        res.k, res.minus, res.plus, res.rem_top_ok = pv - 1, 0, 0, True
        return res
    scale = 0
    if pv == 1:                       # one-limb divisor: divide u*B by v*B (same quotient, remainder r*B)
        u, v, h, scale = u << 32, v << 32, h + 1, 1
    k = prec(v) - 1
    w = shinv(v, h, use_mma, seed, seed_delta, tr)
    res.lam = w - (1 << (32 * h)) // v
    psh = prec(w)
    nq = h - k + 1
    qlen = ru(nq + 1, TILE)
    if psh == 0:
        q0 = 0
    else:
        got = range_mma(u, h, w, psh, (h - 1) // 32, 1 << 20) if use_mma("uw") else None
        if got is not None:
            tr.mma_products += 1
            q0 = low(low(got[0], got[1]) >> (32 * (h - 32 * ((h - 1) // 32))), qlen)
        else:
            klo = (h - 9) // TILE if h >= 17 else 0
            pval, pl = range_imad(u, h, w, psh, klo, 1 << 20)
            q0 = low(low(pval, pl) >> (32 * (h - TILE * klo)), qlen)
    q0 = low(q0, nq)                                                  # pq = top_prec(Q, nq)
    res.q0 = q0
    res.k = k
    res.rem_estimate = u - v * q0
    res.delta = u // v - q0
    rlen = ru(k + 3, TILE)
    p = 0
    if q0:
        got = range_mma(v, k + 1, q0, prec(q0), 0, (rlen + 31) // 32) if use_mma("vq") else None
        if got is not None:
            tr.mma_products += 1
            p = low(got[0], min(rlen, got[1]))
        else:
            p = low(low(v * q0, TILE * ((rlen + TILE - 1) // TILE)), min(rlen, ru(k + 1, TILE) + ru(prec(q0), TILE)))
    mod = 1 << (32 * rlen)
    r = (low(u, rlen) - p) % mod
    top = r >> (32 * (rlen - 1))
    res.rem_top_ok = top in (0, 0xFFFFFFFF)
    q = q0
    minus = 0
    while (r >> (32 * (rlen - 1))) != 0 and minus < CORR_MAX:
        minus += 1
        r = (r + v) % mod
        q = (q - 1) % (1 << (32 * qlen))
    plus = 0
    for _ in range(CORR_MAX):
        if r < v:
            break
        r -= v
        q = (q + 1) % (1 << (32 * qlen))
        plus += 1
    res.minus, res.plus = minus, plus
    res.q = q
    res.r = r >> 32 if scale else low(r, k + 1)
    return res
