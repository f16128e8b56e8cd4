"""Seeded synthetic inputs for the division hot path (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only draws random limbs with a
counter-based generator (numpy's Philox, keyed by (seed, config, stream)) and lays them out
as little-endian uint32 limb arrays (index 0 least significant).  Where a
workload needs a structured operand (``u = v*t``) it is built with Python integers.
Neither the oracle nor the CUDA library is imported here.

Workloads (BASELINE.json ``configs``; the paper measures on its own random integers,
PAPER.md:474, not on a public suite, so these synthetic draws ARE the workload):

  config 1..4  u of M limbs, v of M/2 limbs, uniform limbs, top limbs forced non-zero
  config 5     adversarial mix at M = 2048 (see ``config5``)
  directed     the shapes uniform inputs never reach (small top limb, B^k + c, delta = -1 ...)
  paper_shape  prec(u) = M-2, prec(v) uniform in 2..M/2
"""
from __future__ import annotations

import numpy as np

SEED = 20260638
LIMB_BITS = 32
B = 1 << LIMB_BITS

# (batch, u_limbs, v_limbs) of BASELINE.json configs 1..5
CONFIG_SHAPES = {
    1: (32, 1024, 512),
    2: (1184, 2048, 1024),
    3: (1184, 4096, 2048),
    4: (592, 8192, 4096),
    5: (1184, 2048, 2048),
}


def rng_for(config, stream: int = 0, seed: int = SEED) -> np.random.Generator:
    """Counter-based generator keyed by (seed, config id, stream)."""
    key = (int(seed) & 0xFFFFFFFF) | ((int(config) & 0xFFFF) << 32) | ((int(stream) & 0xFFFF) << 48)
    return np.random.Generator(np.random.Philox(key=key))


# ----------------------------------------------------------------------------------------
# limb <-> Python integer marshalling
# ----------------------------------------------------------------------------------------
def to_limbs(x: int, n_limbs: int) -> np.ndarray:
    """Little-endian uint32 limbs of a non-negative integer, zero padded to n_limbs."""
    if x < 0:
        raise ValueError("negative")
    raw = x.to_bytes(4 * n_limbs, "little")  # raises OverflowError if it does not fit
    return np.frombuffer(raw, dtype="<u4").astype(np.uint32)


def from_limbs(a) -> int:
    a = np.ascontiguousarray(a, dtype="<u4")
    return int.from_bytes(a.tobytes(), "little")


def rows_to_ints(a) -> list:
    return [from_limbs(row) for row in np.asarray(a)]


def ints_to_rows(xs, n_limbs: int) -> np.ndarray:
    out = np.zeros((len(xs), n_limbs), dtype=np.uint32)
    for i, x in enumerate(xs):
        out[i] = to_limbs(x, n_limbs)
    return out


def _uniform(rng, batch: int, limbs: int) -> np.ndarray:
    """Uniform random limbs (two limbs per 64-bit draw)."""
    if limbs == 0:
        return np.zeros((batch, 0), dtype=np.uint32)
    words = rng.integers(0, 1 << 64, size=(batch, (limbs + 1) // 2), dtype=np.uint64)
    return words.view(np.uint32).reshape(batch, -1)[:, :limbs].copy()


def _force_top_nonzero(a: np.ndarray) -> None:
    top = a[:, -1]
    top[top == 0] = 1


def uniform_operands(batch: int, u_limbs: int, v_limbs: int, config=0, seed: int = SEED):
    """u (batch, u_limbs), v (batch, v_limbs): uniform limbs, top limb of each forced non-zero."""
    u = _uniform(rng_for(config, 0, seed), batch, u_limbs)
    v = _uniform(rng_for(config, 1, seed), batch, v_limbs)
    _force_top_nonzero(u)
    _force_top_nonzero(v)
    return u, v


def config(idx: int, batch: int | None = None, seed: int = SEED):
    """Inputs of BASELINE.json config ``idx`` (1-based).  ``batch`` overrides the instance count."""
    if idx == 5:
        return config5(batch=batch, seed=seed)
    b, m, n = CONFIG_SHAPES[idx]
    return uniform_operands(b if batch is None else batch, m, n, config=idx, seed=seed)


def _random_int(rng, limbs: int, top_nonzero: bool = True) -> int:
    if limbs <= 0:
        return 0
    a = _uniform(rng, 1, limbs)
    if top_nonzero:
        _force_top_nonzero(a)
    return from_limbs(a[0])


def config5(batch: int | None = None, limbs: int = 2048, seed: int = SEED):
    """Adversarial mix (BASELINE.json config 5): stride ``limbs`` for u and v.

    Per instance: divisor length lv uniform in 1..limbs, then one category draw:
      25 %  v = B^(lv-1) or B^lv - 1 (half each), u uniform
      25 %  u = v*t exactly, t uniform of (limbs - lv) limbs (t = 1 when lv = limbs), v uniform
      15 %  u < v (shorter u, or same length with a smaller top limb)
      10 %  v = top ceil(lv/2) limbs all ones, low limbs uniform; u uniform
      25 %  both uniform
    "Top limb non-zero" refers to the effective top limb.
    """
    batch = CONFIG_SHAPES[5][0] if batch is None else batch
    rng = rng_for(5, 0, seed)
    us, vs = [], []
    for _ in range(batch):
        lv = int(rng.integers(1, limbs + 1))
        cat = float(rng.random())
        if cat < 0.25:
            v = (1 << (32 * (lv - 1))) if rng.random() < 0.5 else (1 << (32 * lv)) - 1
            u = _random_int(rng, limbs)
        elif cat < 0.50:
            v = _random_int(rng, lv)
            t_limbs = limbs - lv
            t = _random_int(rng, t_limbs) if t_limbs > 0 else 1
            u = v * t
        elif cat < 0.65:
            v = _random_int(rng, lv)
            if lv > 1 and rng.random() < 0.5:
                u = _random_int(rng, int(rng.integers(0, lv)))
            else:
                top = v >> (32 * (lv - 1))
                if top > 1:
                    utop = int(rng.integers(1, top))
                    u = (utop << (32 * (lv - 1))) | _random_int(rng, lv - 1, top_nonzero=False)
                else:
                    u = _random_int(rng, lv - 1)
            assert u < v
        elif cat < 0.75:
            ones = (lv + 1) // 2
            low = _random_int(rng, lv - ones, top_nonzero=False)
            v = (((1 << (32 * ones)) - 1) << (32 * (lv - ones))) | low
            u = _random_int(rng, limbs)
        else:
            v = _random_int(rng, lv)
            u = _random_int(rng, limbs)
        us.append(u)
        vs.append(v)
    return ints_to_rows(us, limbs), ints_to_rows(vs, limbs)


def paper_shape(batch: int, m_limbs: int, seed: int = SEED):
    """The paper's own workload: prec(u) = M-2, prec(v) uniform in 2..M/2."""
    rng = rng_for(40 + m_limbs.bit_length(), 0, seed)
    us = [_random_int(rng, m_limbs - 2) for _ in range(batch)]
    vs = [_random_int(rng, int(rng.integers(2, m_limbs // 2 + 1))) for _ in range(batch)]
    return ints_to_rows(us, m_limbs), ints_to_rows(vs, m_limbs // 2)


def directed(u_limbs: int, v_limbs: int, count: int = 256, seed: int = SEED):
    """Correctness-only shapes that uniform inputs do not reach.

    Small-top-limb divisors (v = B^k + c, top limb 1, sparse v) drive the negative branch of
    the close product and the shifted-inverse over-estimate; the ``q*v + (v-1)`` dividends with
    q near the top of its range drive the delta = -1 correction;
    h - k in {0,1,2,3,2^j+1} and 1..3-limb divisors drive the special cases of Alg. 1.
    """
    rng = rng_for(100 + u_limbs.bit_length(), v_limbs & 0xFFFF, seed)
    M, n = u_limbs, v_limbs
    pairs = []

    def add(u, v):
        if v > 0 and u < (1 << (32 * M)) and v < (1 << (32 * n)):
            pairs.append((u, v))

    # fixed corner cases
    add(0, 1)
    add(0, _random_int(rng, n))
    add(314159265358979, 27183)            # PAPER.md:82 Example 1
    add(726319138718412, 27183)            # PAPER.md:84 Example 2
    for lv in (1, 2, 3, min(4, n), n):
        v = _random_int(rng, lv)
        add(v, v)                           # u = v
        add(v - 1, v)                       # u = v - 1
        add(v + 1, v)
        add((1 << (32 * M)) - 1, v)         # u = B^M - 1
        add(_random_int(rng, M), v)
        add(_random_int(rng, M), 1 << (32 * (lv - 1)))
        add(_random_int(rng, M), (1 << (32 * lv)) - 1)
    add(_random_int(rng, M), 1)
    add(_random_int(rng, M), B - 1)
    add(_random_int(rng, M), B)
    add(_random_int(rng, M), B + 1)

    kinds = 8
    while len(pairs) < count:
        kind = len(pairs) % kinds
        lv = int(rng.integers(2, n + 1))
        k = lv - 1
        if kind == 0:      # v = B^k + c, c < 2^40
            v = (1 << (32 * k)) + int(rng.integers(0, 1 << 40)) if k >= 2 else (1 << (32 * k)) + int(rng.integers(1, 1 << 20))
            u = _random_int(rng, int(rng.integers(lv, M + 1)))
        elif kind == 1:    # top limb 1, random rest
            v = (1 << (32 * k)) | _random_int(rng, k, top_nonzero=False)
            u = _random_int(rng, int(rng.integers(lv, M + 1)))
        elif kind == 2:    # sparse divisor: a few set limbs
            v = 1 << (32 * k)
            for _ in range(3):
                v |= int(rng.integers(1, 4)) << (32 * int(rng.integers(0, lv)))
            u = _random_int(rng, int(rng.integers(lv, M + 1)))
        elif kind == 3:    # delta = -1 recipe: v = B^k + c, q ~ floor((B^h - 1)/v), u = q*v + (v-1)
            h = int(rng.integers(lv, M + 1))
            v = (1 << (32 * k)) + int(rng.integers(1, 1 << 33))
            q = ((1 << (32 * h)) - 1) // v - int(rng.integers(0, 3))
            u = q * v + (v - 1)
            if u >= (1 << (32 * h)):
                u -= v
        elif kind == 4:    # h - k in {0, 1, 2, 3}
            d = int(rng.integers(0, 4))
            hu = min(M, k + d)
            if hu < 1:
                hu = 1
            v = _random_int(rng, lv)
            u = _random_int(rng, hu)
        elif kind == 5:    # h - k = 2^j + 1
            j = int(rng.integers(0, max(1, (M - k).bit_length())))
            hu = min(M, k + (1 << j) + 1)
            v = _random_int(rng, lv)
            u = _random_int(rng, hu)
        elif kind == 6:    # exact multiples and near multiples with small-top-limb v
            v = (1 << (32 * k)) | _random_int(rng, k // 2, top_nonzero=False)
            t = _random_int(rng, int(rng.integers(1, M - lv + 1))) if M > lv else 1
            u = v * t + int(rng.integers(0, 2)) * (v - 1)
        else:              # all-ones patterns
            v = (1 << (32 * lv)) - 1 - int(rng.integers(0, 2))
            u = (1 << (32 * int(rng.integers(lv, M + 1)))) - 1 - int(rng.integers(0, 3))
        add(u, v)

    pairs = pairs[:count]
    return ints_to_rows([p[0] for p in pairs], M), ints_to_rows([p[1] for p in pairs], n)
