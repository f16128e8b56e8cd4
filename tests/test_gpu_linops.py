"""Unit tests of the linear-cost building blocks (mplinop_batch, include/mpdiv.h) against Python integers:
addition and subtraction with the block carry / borrow scan, the less-than test that
falls out of the borrow (:331-335), B^L - P (:117, :329), whole-limb shifts (Definition 1, :61-70; the
paper's own examples shift_1([1,2,3]) = [0,1,2], shift_{-1}([1,2,3]) = [2,3,0], :70), prec (:135) and the
comparison with a power of B (:329).  Every test needs a B200."""
import numpy as np
import pytest
import torch

from paper_2606_06386_b200 import binding, inputs
from paper_2606_06386_b200.inputs import from_limbs, ints_to_rows

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def run(op, a, b, shift, out_limbs):
    out, flag = binding.mplinop_batch(op, dev(a), dev(b), shift, out_limbs)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint32), flag.cpu().numpy().view(np.uint32)


def operands(an, bn, batch, seed):
    rng = inputs.rng_for(600, seed % 65536)
    a = inputs._uniform(rng, batch, an)
    b = inputs._uniform(rng, batch, bn)
    a[0, :] = 0xFFFFFFFF          # longest carry chains
    b[0, :] = 0
    b[0, 0] = 1
    a[1, :] = 0
    b[1, :] = 0
    b[1, 0] = 1                   # 0 - 1: borrow through every limb
    a[2] = 0
    a[2, -1] = 1
    b[2] = 0
    b[2, 0] = 1                   # B^(an-1) - 1: borrow through all but one
    if batch > 3:
        b[3, :] = a[3, :bn] if bn <= an else 0      # equal low parts
    return a, b


SHAPES = [(8, 8, 0, 8), (8, 4, 1, 12), (64, 64, 0, 64), (100, 36, 7, 108), (1024, 1024, 0, 1028), (1028, 520, -3, 1032),
          (2048, 1024, 1024, 2052), (4096, 4096, 0, 4096), (8192, 8192, 0, 8196), (8192, 4, 8190, 8196)]


@pytest.mark.parametrize("an,bn,shift,on", SHAPES)
def test_add_with_carry_scan(an, bn, shift, on):
    a, b = operands(an, bn, 9, an + bn)
    out, flag = run(binding.LINOP_ADD, a, b, shift, on)
    mod = 1 << (32 * on)
    for i in range(a.shape[0]):
        sb = from_limbs(b[i]) << (32 * shift) if shift >= 0 else from_limbs(b[i]) >> (32 * -shift)
        # operands are read as zero beyond out_limbs too: the block adds limb-wise over out_limbs
        total = (from_limbs(a[i]) % mod) + (sb % mod)
        assert from_limbs(out[i]) == total % mod, i
        assert int(flag[i]) == total // mod, i


@pytest.mark.parametrize("an,bn,shift,on", SHAPES)
def test_sub_with_borrow_scan_and_less_than(an, bn, shift, on):
    a, b = operands(an, bn, 9, an * 3 + bn)
    out, flag = run(binding.LINOP_SUB, a, b, shift, on)
    mod = 1 << (32 * on)
    for i in range(a.shape[0]):
        sb = from_limbs(b[i]) << (32 * shift) if shift >= 0 else from_limbs(b[i]) >> (32 * -shift)
        x, y = from_limbs(a[i]) % mod, sb % mod
        assert from_limbs(out[i]) == (x - y) % mod, i
        assert int(flag[i]) == (1 if x < y else 0), i        # the borrow IS the less-than test


@pytest.mark.parametrize("an,L,on", [(8, 8, 8), (8, 5, 8), (64, 64, 68), (1028, 1000, 1028), (4096, 4096, 4100), (8, 12, 16)])
def test_power_of_B_minus(an, L, on):
    rng = inputs.rng_for(601, an + L)
    vals = [inputs._random_int(rng, min(an, L), top_nonzero=False) for _ in range(6)] + [0, 1, (1 << (32 * min(an, L))) - 1]
    a = ints_to_rows(vals, an)
    out, _ = run(binding.LINOP_NEG, a, a, L, on)
    for i, x in enumerate(vals):
        assert from_limbs(out[i]) == ((1 << (32 * L)) - x) % (1 << (32 * on)), i


def test_shift_paper_examples():
    """shift_1([1,2,3]) = [0,1,2] and shift_{-1}([1,2,3]) = [2,3,0] (index 0 least significant)."""
    a = np.array([[1, 2, 3, 0]], dtype=np.uint32)
    out, _ = run(binding.LINOP_SHIFT, a, a, 1, 4)
    assert list(out[0][:3]) == [0, 1, 2]
    out, _ = run(binding.LINOP_SHIFT, a, a, -1, 4)
    assert list(out[0][:3]) == [2, 3, 0]


@pytest.mark.parametrize("an,shift,on", [(8, 3, 12), (8, -3, 8), (1024, 517, 2048), (1024, -1000, 1024), (4096, 0, 4096),
                                         (64, 100, 64), (64, -100, 64)])
def test_shift_whole_limbs(an, shift, on):
    rng = inputs.rng_for(602, an)
    a = inputs._uniform(rng, 5, an)
    out, _ = run(binding.LINOP_SHIFT, a, a, shift, on)
    for i in range(5):
        x = from_limbs(a[i])
        want = (x << (32 * shift)) if shift >= 0 else (x >> (32 * -shift))
        assert from_limbs(out[i]) == want % (1 << (32 * on)), i


@pytest.mark.parametrize("an", [4, 8, 100, 1024, 8192])
def test_prec_and_compare_with_power_of_B(an):
    rng = inputs.rng_for(603, an)
    lens = [0, 1, 2, an // 2, an - 1, an, int(rng.integers(0, an + 1)), int(rng.integers(0, an + 1))]
    vals = [inputs._random_int(rng, l) for l in lens]
    a = ints_to_rows(vals, an)
    out, flag = run(binding.LINOP_PREC, a, a, 0, an)
    assert [int(f) for f in flag] == lens
    assert (out == a).all()
    for h in (0, 1, an // 2, an - 1):
        _, flag = run(binding.LINOP_ANY, a, a, h, an)
        assert [int(f) for f in flag] == [1 if x >= (1 << (32 * h)) else 0 for x in vals], h


@pytest.mark.gpu
def test_mma_probe_rates():
    """mpdiv_mma_probe: every bounded wait completes, and the measured cycles per tcgen05.mma are never below the
    tensor core's N / 2 (two issuing warps share one tensor core) nor absurdly above it."""
    from paper_2606_06386_b200 import binding
    for n in (16, 64, 128):
        one = binding.mma_probe(n, 1, iters=500)
        two = binding.mma_probe(n, 2, iters=500)
        assert one[0] > 0 and min(two) > 0, "a bounded wait gave up"
        assert one[0] >= n / 2.0 * 0.98 and max(two) / 2.0 >= n / 2.0 * 0.98
        assert one[0] < 400 and max(two) < 800
    with pytest.raises(binding.MpdivError):
        binding.mma_probe(24, 1)
