"""The bounds the default (clipped) division rests on, checked on a Python-integer replay of the shipped flow.

Theorem 2 (lambda in {0,1}, then delta in {-1,0,1}) is stated for the algorithm as printed and
proved in a thesis that is not available; the paper leaves clipped products as future work.
tests/clipped_flow_model.py replays exactly what csrc/ computes for MPDIV_VARIANT_CLIPPED -- the 8-limb tile
windows of the IMAD engine and the 32-limb windows of the tensor-core engine (c_x, Klo2, Klo1, dlo as coded in
mp_div.cuh refine_step), the "+1" Refine loop, the 17-digit seed, the head split, u*shinv from column h - 9, and
the remainder arithmetic mod B^(k+3) -- and these tests assert, over the directed inputs and a sweep over
(k, h - k) and divisor families:

  * lambda = shinv - floor(B^h / v) in {-1, 0, 1}
  * pre-correction delta = floor(u / v) - q0' in {-1, 0, 1, 2}  (far inside the 64 steps of the correction loops)
  * |u - v*q0'| < B^(k+2), i.e. the top limb of the mod-B^(k+3) remainder estimate is 0 or all ones
  * the final (q, r) equals Python's divmod
  * every iterate stays below B^(l+g+2) (the window the kernel reads)

and the same with the seed perturbed by +-1 and +-2 units.  CPU only; nothing here touches oracle/ or the library
(tests/test_gpu_parity.py::test_shinv_matches_the_flow_model ties the replay to the kernels bit for bit).
"""
import random

import pytest

import clipped_flow_model as model
from paper_2606_06386_b200 import inputs

B = 1 << 32

POLICIES = {
    "imad": lambda rnd: (lambda kind: False),              # 8-limb tile windows everywhere (small sizes, latency kernels)
    "tensor": lambda rnd: (lambda kind: True),             # 32-limb windows wherever the kernel may choose them
    "mixed": lambda rnd: (lambda kind: rnd.random() < 0.5),  # any per-product decision of mma_plan
}


class Ranges:
    def __init__(self):
        self.lam, self.delta, self.minus, self.plus = set(), set(), 0, 0
        self.cases = self.clipped = self.mma = self.sign_neg = 0

    def add(self, u, v, res):
        assert (res.q, res.r) == divmod(u, v), "model result is not the quotient and remainder"
        assert res.rem_top_ok, "remainder estimate left the range of the mod-B^(k+3) arithmetic"
        if res.trace.steps or res.q0:
            assert abs(res.rem_estimate) < 1 << (32 * (res.k + 2))
        self.lam.add(res.lam)
        self.delta.add(res.delta)
        self.minus = max(self.minus, res.minus)
        self.plus = max(self.plus, res.plus)
        self.cases += 1
        self.clipped += res.trace.clipped_steps
        self.mma += res.trace.mma_products
        self.sign_neg += res.trace.sign_neg

    def check(self):
        assert self.lam <= {-1, 0, 1}, "lambda range %s" % sorted(self.lam)
        assert self.delta <= {-1, 0, 1, 2}, "delta range %s" % sorted(self.delta)
        assert self.minus <= 2 and self.plus <= 3


@pytest.mark.parametrize("policy", sorted(POLICIES))
@pytest.mark.parametrize("M,n,count", [(8, 4, 200), (64, 32, 400), (128, 64, 400), (256, 128, 300), (512, 256, 160),
                                       (300, 300, 160), (1024, 512, 120)])
def test_bounds_on_the_directed_set(M, n, count, policy):
    rnd = random.Random(M * 131 + n)
    u, v = inputs.directed(M, n, count=count)
    rg = Ranges()
    for i in range(count):
        ui, vi = inputs.from_limbs(u[i]), inputs.from_limbs(v[i])
        rg.add(ui, vi, model.divide(ui, vi, POLICIES[policy](rnd)))
    rg.check()
    print(M, n, policy, "lambda", sorted(rg.lam), "delta", sorted(rg.delta), "clipped steps", rg.clipped, "tensor windows", rg.mma)
    if M >= 128:
        assert rg.clipped > 0                         # long enough for the windows to clip something
        if policy != "imad":
            assert rg.mma > 0
    if M >= 64 and count >= 160:
        assert rg.sign_neg > 0 and 1 in rg.lam        # the directed set reaches the over-estimate and the negative branch


def _divisor(rnd, family, k):
    """v with prec(v) = k + 1 from one of the families of SURVEY 8(c) (small top limbs reach the rare branches)."""
    if family == "uniform":
        return (rnd.randrange(1, B) << (32 * k)) | rnd.getrandbits(32 * k)
    if family == "pow_plus_c":
        return (1 << (32 * k)) + rnd.randrange(1, 1 << 40)
    if family == "top_one":
        return (1 << (32 * k)) | rnd.getrandbits(32 * k)
    if family == "top_ones":
        ones = (k + 2) // 2
        return (((1 << (32 * ones)) - 1) << (32 * (k + 1 - ones))) | rnd.getrandbits(32 * (k + 1 - ones))
    v = 1 << (32 * k)                                  # sparse
    for _ in range(3):
        v |= rnd.randrange(1, 4) << (32 * rnd.randrange(0, k + 1))
    return v


def _dividends(rnd, v, h):
    top = 1 << (32 * h)
    yield (rnd.randrange(1, B) << (32 * (h - 1))) | rnd.getrandbits(32 * (h - 1))          # uniform, h limbs
    yield top - 1                                                                         # B^h - 1
    q = (top - 1) // v - rnd.randrange(0, 3)                                              # the delta = -1 recipe
    if q > 0:
        u = q * v + v - 1
        yield u if u < top else u - v


KS = (1, 2, 3, 7, 16, 18, 19, 20, 21, 40, 64, 65, 130, 260)
HKS = (0, 1, 2, 3, 4, 5, 9, 16, 17, 18, 32, 33, 34, 64, 65, 66, 129, 130, 131, 257, 258)
FAMILIES = ("uniform", "pow_plus_c", "top_one", "top_ones", "sparse")


@pytest.mark.parametrize("policy", sorted(POLICIES))
def test_bounds_on_a_sweep_over_k_and_h_minus_k(policy):
    """Every (k, h - k) pair around the thresholds of the flow: the seed (H >= 17), the window conditions
    (c_x >= 25, dd >= 17, dd >= 33), the head split (l <= 129), powers of two plus one."""
    rnd = random.Random(20260638)
    rg = Ranges()
    for k in KS:
        for hk in HKS:
            if k + hk > 400 or k + hk < 1:
                continue
            for fam in FAMILIES:
                v = _divisor(rnd, fam, k)
                for u in _dividends(rnd, v, k + hk):
                    rg.add(u, v, model.divide(u, v, POLICIES[policy](rnd)))
    rg.check()
    print(policy, rg.cases, "cases: lambda", sorted(rg.lam), "delta", sorted(rg.delta), "max -1 steps", rg.minus,
          "max +1 steps", rg.plus, "clipped steps", rg.clipped, "tensor windows", rg.mma)
    assert rg.cases > 2500 and rg.clipped > 1000


@pytest.mark.parametrize("seed_delta", [-2, -1, 1, 2])
def test_bounds_with_a_perturbed_seed(seed_delta):
    """The seed floor(B^38 / D) is within one unit of B^(k+19)/v; the flow must absorb more than that."""
    rnd = random.Random(77 + seed_delta)
    rg = Ranges()
    for k in (18, 19, 20, 40, 130):
        for hk in (17, 18, 33, 65, 130, 258):
            for fam in FAMILIES:
                v = _divisor(rnd, fam, k)
                for u in _dividends(rnd, v, k + hk):
                    rg.add(u, v, model.divide(u, v, POLICIES["mixed"](rnd), seed=True, seed_delta=seed_delta))
    rg.check()
    assert rg.cases > 400


def test_seedless_flow_and_one_limb_divisors():
    """MPDIV_FLAG_NO_SEED (Refine from l = 2 as printed) and the one-limb mapping u*B / v*B."""
    rnd = random.Random(5)
    rg = Ranges()
    for k in (1, 2, 19, 64):
        for hk in (1, 2, 17, 40, 129):
            v = _divisor(rnd, "top_one", k)
            for u in _dividends(rnd, v, k + hk):
                rg.add(u, v, model.divide(u, v, POLICIES["mixed"](rnd), seed=False))
    for h in (1, 2, 5, 40, 200):
        for v in (1, 2, 3, B - 1, rnd.randrange(1, B)):
            u = rnd.getrandbits(32 * h) | (1 << (32 * h - 1))
            rg.add(u, v, model.divide(u, v))
    rg.check()


def test_the_model_of_the_windows_against_their_definition():
    """The omitted parts E of the two engines are what mp_mul.cuh / mp_mma.cuh promise: 0 <= E < B^(8 Klo + 9) for the
    tile windows (their comment's bound) and 0 <= E < B^(32 dlo + 1) for the byte-column windows, and a window
    that omits nothing is the exact product."""
    rnd = random.Random(9)
    for _ in range(200):
        na, nb = rnd.randrange(1, 90), rnd.randrange(1, 90)
        a, b = rnd.getrandbits(32 * na), rnd.getrandbits(32 * nb)
        klo = rnd.randrange(0, (na + nb) // 8 + 1)
        e = model.omitted_tiles(a, b, klo)
        assert 0 <= e < 1 << (32 * (8 * klo + 9)) or klo == 0 and e == 0
        val, limbs = model.range_imad(a, na, b, nb, klo, 1 << 20)
        assert (val << (256 * klo)) + e == a * b and limbs >= na + nb - 8 * klo
        dlo = rnd.randrange(0, (na + nb) // 32 + 1)
        e = model.omitted_byte_columns(a, b, 128 * dlo)
        assert 0 <= e < 1 << (32 * (32 * dlo + 1)) or dlo == 0 and e == 0
        got = model.range_mma(a, na, b, nb, dlo, 1 << 20)
        if got is not None:
            assert (got[0] << (1024 * dlo)) + e == a * b
    assert model.refine_iters(1025) == 11 and model.refine_iters(1025, clip=False) == 12     # "+1" against the printed "+2"
    assert model.head_plan(1025, 11) == 8 and model.head_plan(16, 5) == 0
