"""The 17-digit seed of Refine (csrc/mp_div.cuh warp_seed, include/mpdiv.h mpdiv_seed_batch) against its
definition, floor(B^38 / D) with D the top 20 limbs of v, evaluated with CPython integers; and Shinv / Div with
and without the seed give the same exact results (the seed replaces Alg. 1's first four iterations,
PAPER.md:92 lines 19-25)."""
import numpy as np
import pytest

from paper_2606_06386_b200 import inputs

pytestmark = pytest.mark.gpu

B = 1 << 32
SPECIAL = np.array([0, 1, 2, 0x7FFFFFFF, 0x80000000, 0x80000001, 0xFFFFFFFE, 0xFFFFFFFF], dtype=np.uint64)


def _expected(row):
    x = inputs.from_limbs(row)
    k = (x.bit_length() + 31) // 32 - 1
    if k < 1:
        return 0
    d = (x << (32 * 19)) >> (32 * k)
    return (1 << (32 * 38)) // d


def _run(v):
    import torch

    from paper_2606_06386_b200 import binding

    dv = torch.from_numpy(v.view(np.int32)).cuda()
    w = binding.seed_batch(dv)
    torch.cuda.synchronize()
    return w.cpu().numpy().view(np.uint32)


def _check(v):
    w = _run(v)
    assert w.shape == (v.shape[0], 24)
    for i in range(v.shape[0]):
        assert inputs.from_limbs(w[i]) == _expected(v[i]), (i, [hex(int(t)) for t in v[i][-6:]])


@pytest.mark.parametrize("limbs", [4, 8, 20, 24, 64, 1024])
def test_seed_uniform(limbs):
    rng = np.random.Generator(np.random.Philox(inputs.SEED + limbs))
    v = rng.integers(0, B, size=(257, limbs), dtype=np.uint64).astype(np.uint32)
    v[:, -1] |= 1                                   # top limb non-zero
    _check(v)


@pytest.mark.parametrize("limbs", [4, 20, 24, 40])
def test_seed_special_limbs(limbs):
    """Limbs drawn from {0, 1, 2, B/2-1, B/2, B/2+1, B-2, B-1}: quotient digits of B-1, the two-digit test of
    Knuth D3 and the add-back of D6 all occur (the add-back counter must move)."""
    import torch

    from paper_2606_06386_b200 import binding

    rng = np.random.Generator(np.random.Philox(inputs.SEED + 77 + limbs))
    v = SPECIAL[rng.integers(0, len(SPECIAL), size=(4096, limbs))].astype(np.uint32)
    v[:, -1] = np.where(v[:, -1] == 0, 1, v[:, -1])
    binding.debug_counters(reset=True)
    _check(v)
    torch.cuda.synchronize()
    if limbs >= 20:
        assert binding.debug_counters()["seed_addbacks"] > 0


def test_seed_precision_sweep():
    """prec(v) from 1 to 48 limbs inside a 48-limb row: one-limb and zero divisors give zeros, short divisors are
    extended with zero limbs below (D = v B^(19-k))."""
    rng = np.random.Generator(np.random.Philox(inputs.SEED + 5))
    rows = []
    for p in range(0, 49):
        for _ in range(4):
            r = np.zeros(48, dtype=np.uint32)
            if p:
                r[:p] = rng.integers(0, B, size=p, dtype=np.uint64).astype(np.uint32)
                r[p - 1] |= 1
            rows.append(r)
    _check(np.stack(rows))


def test_seed_extremes():
    rows = []
    for top in (1, 2, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF):
        for fill in (0, 1, 0xFFFFFFFF):
            r = np.full(32, fill, dtype=np.uint32)
            r[-1] = top
            rows.append(r)
            r2 = r.copy()
            r2[0] = 0                                # below the 20 limbs the seed reads: no effect
            r2[11] ^= 1
            rows.append(r2)
            r3 = r.copy()
            r3[12] ^= 1                              # the lowest limb the seed reads
            rows.append(r3)
    _check(np.stack(rows))


@pytest.mark.parametrize("cfg", [1, 2, 5])
def test_division_same_with_and_without_seed(cfg):
    """MPDIV_FLAG_NO_SEED starts Refine at l = 2 as printed; q and r must not change (both are exact), and the
    shifted inverse may differ by its lambda only."""
    import torch

    from paper_2606_06386_b200 import binding

    u, v = inputs.config(cfg, batch=64)
    du = torch.from_numpy(u.view(np.int32)).cuda()
    dv = torch.from_numpy(v.view(np.int32)).cuda()
    binding.debug_counters(reset=True)
    q1, r1 = binding.mpdiv_batch(du, dv)
    torch.cuda.synchronize()
    assert binding.debug_counters()["seeds"] > 0
    binding.debug_counters(reset=True)
    q0, r0 = binding.mpdiv_batch(du, dv, variant=binding.VARIANT_CLIPPED | binding.FLAG_NO_SEED)
    torch.cuda.synchronize()
    assert binding.debug_counters()["seeds"] == 0
    assert torch.equal(q0, q1) and torch.equal(r0, r1)


# ---- the head of Refine in its own kernel (csrc/mp_div.cuh "Head of Refine") ------------------------------

def _div(u, v, flags=None):
    import torch

    from paper_2606_06386_b200 import binding

    du = torch.from_numpy(u.view(np.int32)).cuda()
    dv = torch.from_numpy(v.view(np.int32)).cuda()
    binding.status(reset=True)
    q, r = binding.mpdiv_batch(du, dv, variant=flags)
    assert binding.status(reset=True) == 0
    return q.cpu().numpy().view(np.uint32), r.cpu().numpy().view(np.uint32)


def test_batch_launches_reports_the_head_kernel():
    from paper_2606_06386_b200 import binding

    assert binding.batch_launches(2048, 1184) == 2            # config 2: head + division
    assert binding.batch_launches(8192, 592) == 2
    assert binding.batch_launches(2048, 32) == 1              # latency-oriented kernel keeps Refine in the block
    assert binding.batch_launches(256, 100000) == 1           # below 512 limbs
    assert binding.batch_launches(2048, 1184, binding.VARIANT_PRINTED) == 1
    assert binding.batch_launches(0, 5) == 0


@pytest.mark.parametrize("M,count", [(512, 1500), (1024, 900), (2048, 700), (4096, 400)])
def test_head_kernel_random_precisions(M, count):
    """Batches large enough for the head kernel, random effective precisions of u and v: every H = h - k from
    below the seed's threshold (17) through every split point of head_plan occurs.  q and r against the oracle,
    and identical with the head switched off."""
    from oracle import oracle
    from paper_2606_06386_b200 import binding

    assert binding.batch_launches(M, count) == 2
    rng = inputs.rng_for(410, M % 65536)
    us, vs = [], []
    for i in range(count):
        lv = int(rng.integers(1, M + 1))
        if i % 4 == 0:
            lu = min(M, lv + int(rng.integers(0, 300)))       # H around the thresholds 17, 33, 65, 129, 257
        else:
            lu = int(rng.integers(0, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    u, v = inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, M)
    binding.debug_counters(reset=True)
    q1, r1 = _div(u, v)
    cnt = binding.debug_counters(reset=True)
    assert cnt["seeds"] > 0 and cnt["delta_out_of_range"] == 0
    qo, ro = oracle.divmod_batch(u, v)
    assert (q1 == qo).all() and (r1 == ro).all()
    q0, r0 = _div(u, v, binding.VARIANT_CLIPPED | binding.FLAG_NO_HEAD)
    assert (q0 == q1).all() and (r0 == r1).all()


@pytest.mark.parametrize("M,n", [(1024, 512), (2048, 1024), (2048, 2048)])
def test_head_kernel_directed(M, n):
    """The directed corner-case set at head-kernel batch sizes (powers of B, v = B^k + c, sparse divisors,
    delta = -1 dividends, h - k in {0, 1, 2, 3, 2^j + 1})."""
    from oracle import oracle

    u, v = inputs.directed(M, n, count=1024, seed=inputs.SEED + 3)
    q, r = _div(u, v)
    qo, ro = oracle.divmod_batch(u, v)
    assert (q == qo).all() and (r == ro).all()
