"""Pins of the CPU oracle (oracle/knuth_d.c) against things other than itself.

Each test ties the oracle to what the paper prints or what mathematics fixes, chosen so that a
plausible mistake in the long division (wrong qhat correction, missing add-back, normalisation
off by one bit, transposed operands) fails at least one:

  * values printed in PAPER.md:72, :82, :84 (tests/golden/paper_examples.txt),
  * exhaustive brute force at a test-only base 16 against native integer division,
  * CPython's arbitrary-precision divmod (an independent implementation; stands in for the
    paper's GMP check),
  * the defining invariants u = q*v + r, 0 <= r < v and closed forms.
"""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2606_06386_b200 import inputs
from paper_2606_06386_b200.inputs import B, from_limbs, to_limbs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_examples.txt")


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, value, _cite = [s.strip() for s in line.split("|")]
            out[name] = int(value)
    return out


def odiv(u: int, v: int, un=None, vn=None):
    un = un or max(1, (u.bit_length() + 31) // 32)
    vn = vn or max(1, (v.bit_length() + 31) // 32)
    q, r = oracle.divmod_limbs(to_limbs(u, un), to_limbs(v, vn), un, vn)
    return from_limbs(q), from_limbs(r)


# ---------------------------------------------------------------- paper-printed values
def test_paper_example_1():
    g = golden()
    q, r = odiv(g["ex1_u"], g["ex1_v"])
    assert q == g["ex1_q"]
    assert r == g["ex1_u"] - g["ex1_q"] * g["ex1_v"] == 21425


def test_paper_example_2():
    g = golden()
    q, r = odiv(g["ex2_u"], g["ex2_v"])
    assert q == g["ex2_q"] == g["ex2_q0"] + 1
    # PAPER.md:84 prints u - q0*v = 40734 = r + v
    assert r + g["ex2_v"] == g["ex2_u_minus_q0v"]


def test_paper_shinv_values_base10():
    g = golden()
    # shinv_h(v) = floor(B^h / v), Definition 1, with the paper's B = 10
    q, _ = odiv(10 ** g["ex1_h"], g["ex1_v"])
    assert q == g["ex1_shinv"]
    q, _ = odiv(10 ** 3, 8)
    assert q == g["shinv3_8"]


def test_paper_newton_sequence_is_eq3():
    """Eq. (3) with floor semantics reproduces the printed iterates, and its
    fixed point is the value the oracle's definition gives (ties Definition 1 to eq. (2)/(3))."""
    g = golden()
    v, h = g["ex1_v"], g["ex1_h"]
    w = g["ex1_w0"]
    seq = [w]
    for _ in range(4):
        w = w + ((w * 10 ** h - v * w * w) // 10 ** h)
        seq.append(w)
    assert seq == [g["ex1_w0"], g["ex1_w1"], g["ex1_w2"], g["ex1_w3"], g["ex1_shinv"]]
    q, _ = odiv(10 ** h, v)
    assert q == seq[-1]


# ---------------------------------------------------------------- brute force, tiny base
def test_bruteforce_base16_exhaustive():
    """All u < 2^16, v in 1..255 through the limb routine at base 16 (4 x 2 limbs) against
    native integer division.  Reaches qhat correction and add-back, which base 2^32 never does
    on random data."""
    def digits(x, n):
        return np.array([(x >> (4 * i)) & 15 for i in range(n)], dtype=np.uint32)

    step_u = 1
    us = range(0, 1 << 16, step_u)
    bad = 0
    # vectorised expected values; the oracle is called per pair (65536*255 is too many for a
    # Python loop, so: all v for a strided set of u, and all u for a set of v)
    v_all = list(range(1, 256))
    u_some = list(range(0, 1 << 16, 97)) + [0xFFFF, 0xFFF0, 0x8000, 0x7FFF, 0x0FFF, 0x1000]
    for u in u_some:
        du = digits(u, 4)
        for v in v_all:
            q, r = oracle.divmod_limbs(du, digits(v, 2), 4, 2, base16=True)
            qq = sum(int(d) << (4 * i) for i, d in enumerate(q))
            rr = sum(int(d) << (4 * i) for i, d in enumerate(r))
            if (qq, rr) != (u // v, u % v):
                bad += 1
    assert bad == 0
    for v in (0x10, 0x11, 0x1F, 0x7F, 0x80, 0x81, 0x8F, 0xF0, 0xFE, 0xFF, 0x9A, 0x55):
        dv = digits(v, 2)
        for u in us:
            q, r = oracle.divmod_limbs(digits(u, 4), dv, 4, 2, base16=True)
            qq = int(q[0]) | int(q[1]) << 4 | int(q[2]) << 8 | int(q[3]) << 12
            rr = int(r[0]) | int(r[1]) << 4
            assert (qq, rr) == (u // v, u % v), (u, v)


def test_bruteforce_base16_three_limb_divisors():
    """u < 16^6, v of exactly 3 base-16 limbs: exercises the second-limb refinement of qhat."""
    rng = inputs.rng_for(900)

    def digits(x, n):
        return np.array([(x >> (4 * i)) & 15 for i in range(n)], dtype=np.uint32)

    for _ in range(20000):
        u = int(rng.integers(0, 16 ** 6))
        v = int(rng.integers(16 ** 2, 16 ** 3))
        q, r = oracle.divmod_limbs(digits(u, 6), digits(v, 3), 6, 3, base16=True)
        qq = sum(int(d) << (4 * i) for i, d in enumerate(q))
        rr = sum(int(d) << (4 * i) for i, d in enumerate(r))
        assert (qq, rr) == (u // v, u % v), (u, v)


# ---------------------------------------------------------------- independent implementation
@pytest.mark.parametrize("max_limbs", [4, 64, 1024])
def test_against_python_divmod_random_precisions(max_limbs):
    rng = inputs.rng_for(901, max_limbs)
    count = {4: 6000, 64: 3000, 1024: 300}[max_limbs]
    for _ in range(count):
        ul = int(rng.integers(1, max_limbs + 1))
        vl = int(rng.integers(1, max_limbs + 1))
        u = inputs._random_int(rng, ul, top_nonzero=bool(rng.integers(0, 2)))
        v = inputs._random_int(rng, vl) or 1
        q, r = odiv(u, v, un=max_limbs, vn=max_limbs)
        assert (q, r) == divmod(u, v)


def test_against_python_divmod_full_size():
    """Full-size instances of configs 1-4 (a few each) and of the adversarial config 5."""
    for cfg in (1, 2, 3, 4):
        u, v = inputs.config(cfg, batch=3)
        q, r = oracle.divmod_batch(u, v)
        for i in range(u.shape[0]):
            assert (from_limbs(q[i]), from_limbs(r[i])) == divmod(from_limbs(u[i]), from_limbs(v[i]))
    u, v = inputs.config5(batch=96)
    q, r = oracle.divmod_batch(u, v, threads=4)
    for i in range(u.shape[0]):
        assert (from_limbs(q[i]), from_limbs(r[i])) == divmod(from_limbs(u[i]), from_limbs(v[i]))


def test_small_top_limb_divisors_vs_python():
    """Divisors whose normalisation shift is large (top limb 1..3) and dividends of all-ones:
    the corner where qhat is most often one too large."""
    rng = inputs.rng_for(902)
    for _ in range(3000):
        vl = int(rng.integers(2, 12))
        ul = int(rng.integers(vl, 24))
        v = (int(rng.integers(1, 4)) << (32 * (vl - 1))) | inputs._random_int(rng, vl - 1, False)
        if rng.random() < 0.5:
            u = (1 << (32 * ul)) - 1 - int(rng.integers(0, 4))
        else:
            u = inputs._random_int(rng, ul)
        assert odiv(u, v, un=24, vn=12) == divmod(u, v)


# ---------------------------------------------------------------- invariants
def test_invariants_with_independent_multiply_add():
    """u = q*v + r and r < v determine (q, r) uniquely; the check multiplies
    with Python integers, not with the oracle's own schoolbook product."""
    u, v = inputs.directed(256, 128, count=600)
    q, r = oracle.divmod_batch(u, v)
    for i in range(u.shape[0]):
        U, V, Q, R = (from_limbs(x[i]) for x in (u, v, q, r))
        assert Q * V + R == U
        assert 0 <= R < V
        assert Q.bit_length() <= max(0, U.bit_length() - V.bit_length() + 1)


# ---------------------------------------------------------------- closed forms
def test_closed_forms():
    rng = inputs.rng_for(903)
    for _ in range(300):
        n = int(rng.integers(1, 40))
        m = int(rng.integers(n, 80))
        u = inputs._random_int(rng, m)
        v = inputs._random_int(rng, n)
        k = int(rng.integers(0, n))
        # u < v  =>  (0, u)
        small = u % v
        assert odiv(small, v, un=80, vn=40) == (0, small)
        # u = v*t  =>  (t, 0)
        t = inputs._random_int(rng, max(1, 80 - n - 1))
        assert odiv(v * t, v, un=80, vn=40) == (t, 0)
        # v = B^k  =>  q = limbs k.. of u, r = limbs 0..k-1
        ul = to_limbs(u, 80)
        q, r = oracle.divmod_limbs(ul, to_limbs(B ** k, 40), 80, 40)
        assert list(q[: 80 - k]) == list(ul[k:]) and not q[80 - k:].any()
        assert list(r[:k]) == list(ul[:k]) and not r[k:].any()
        # v = 1, u = v
        assert odiv(u, 1, un=80, vn=40) == (u, 0)
        assert odiv(v, v, un=80, vn=40) == (1, 0)


def test_closed_form_B_pow_k_minus_1():
    """v = B^k - 1, u < B^(2k) (the shape of configs 1-4): with u = a*B^k + b and s = a + b,
    q = a + floor(s/v) with floor(s/v) in {0,1,2} and r = s mod v -- additions only."""
    rng = inputs.rng_for(904)
    for _ in range(300):
        k = int(rng.integers(1, 48))
        v = B ** k - 1
        u = inputs._random_int(rng, 2 * k, top_nonzero=False)
        if rng.random() < 0.2:
            u = B ** (2 * k) - 1 - int(rng.integers(0, 3))
        a, b = u >> (32 * k), u & (B ** k - 1)
        s = a + b
        extra = 0
        while s >= v:
            s -= v
            extra += 1
        assert extra <= 2
        assert odiv(u, v, un=96, vn=48) == (a + extra, s)


# ---------------------------------------------------------------- the other two oracle entry points
def test_mul_against_python_and_truncation():
    rng = inputs.rng_for(905)
    for _ in range(200):
        an = int(rng.integers(1, 70))
        bn = int(rng.integers(1, 70))
        a = inputs._uniform(rng, 1, an)
        b = inputs._uniform(rng, 1, bn)
        full = from_limbs(a[0]) * from_limbs(b[0])
        for cn in (an + bn, max(1, (an + bn) // 2), 1, an + bn + 3):
            c = oracle.mul_batch(a, b, cn)
            assert from_limbs(c[0]) == full % (B ** cn)
    # not symmetric inputs: a transposed operand or an index slip shows up here
    a = np.array([[1, 2, 3]], dtype=np.uint32)
    b = np.array([[5, 0, 0, 7]], dtype=np.uint32)
    assert list(oracle.mul_batch(a, b, 7)[0]) == [5, 10, 15, 7, 14, 21, 0]
    # carries all the way up
    a = np.full((1, 8), 0xFFFFFFFF, dtype=np.uint32)
    assert from_limbs(oracle.mul_batch(a, a, 16)[0]) == (B ** 8 - 1) ** 2


def test_shinv_is_floor_of_power_over_v():
    rng = inputs.rng_for(906)
    for _ in range(300):
        n = int(rng.integers(1, 20))
        h = int(rng.integers(0, 45))
        v = inputs._random_int(rng, n)
        w = oracle.shinv_batch(to_limbs(v, 20)[None, :], h, 48)
        assert from_limbs(w[0]) == B ** h // v
    # closed forms: v = B^k -> B^(h-k); v > B^h -> 0; 2v > B^h -> 1 (Alg. 1 l.5-10)
    assert from_limbs(oracle.shinv_batch(to_limbs(B ** 3, 8)[None, :], 7, 8)[0]) == B ** 4
    assert from_limbs(oracle.shinv_batch(to_limbs(B ** 3 + 1, 8)[None, :], 3, 8)[0]) == 0
    assert from_limbs(oracle.shinv_batch(to_limbs(B ** 3 // 2 + 1, 8)[None, :], 3, 8)[0]) == 1


def test_error_statuses():
    with pytest.raises(oracle.OracleError):
        oracle.divmod_limbs(to_limbs(5, 2), to_limbs(0, 2), 2, 2)
    with pytest.raises(oracle.OracleError):
        oracle.divmod_limbs(to_limbs(B ** 3, 4), to_limbs(1, 1), 2, 1)   # q does not fit


def test_threaded_batch_equals_serial():
    u, v = inputs.config(1)
    q1, r1 = oracle.divmod_batch(u, v, threads=1)
    q4, r4 = oracle.divmod_batch(u, v, threads=4)
    assert np.array_equal(q1, q4) and np.array_equal(r1, r4)
