"""2^19-bit dividends (the paper stops at 2^18 bits for lack of shared memory): the
chunked form of mpdiv_batch (include/mpdiv.h, csrc/mpdiv_api.inl mpdiv_kernel<.., BIG>) against the oracle, bit exact.

The dividend stays in HBM and the quotient is produced window by window, so the cases here are the ones a window
boundary can break: quotients of exactly t, t + 1, 2t limbs, dividends whose top window is one limb long, running
remainders of v - 1, one-limb divisors (u*B / v*B re-basing across windows), u < v and v = 0 (rows copied HBM to HBM).
"""
import os

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_06386_b200 import binding, inputs

pytestmark = pytest.mark.gpu

NCPU = max(1, os.cpu_count() or 1)
T = 2048     # the chunk at v_limbs <= 8192 on a B200 (227 KB of shared memory)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host(t):
    return t.cpu().numpy().view(np.uint32)


def check(u, v, what, flags=None, allow=0):
    binding.status(reset=True)
    q, r = binding.mpdiv_batch(dev(u), dev(v), variant=flags)
    st = binding.status(reset=True)
    assert st & ~allow == 0, "mpdiv_status = %#x" % st
    q, r = host(q), host(r)
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    bad = np.nonzero((q != qo).any(axis=1) | (r != ro).any(axis=1))[0]
    assert bad.size == 0, "%s: %d of %d instances differ, first %d" % (what, bad.size, u.shape[0], bad[0])


def test_config_shape_2p19():
    """The configs' shape one size up: 2^19-bit by 2^18-bit, uniform limbs, top limbs non-zero."""
    binding.debug_counters(reset=True)
    u, v = inputs.uniform_operands(40, 16384, 8192, config=19)
    check(u, v, "uniform 16384/8192")
    cnt = binding.debug_counters(reset=True)
    print("counters", cnt)
    assert cnt["chunks"] == 40 * 5           # D = 8193 quotient limbs = 4 windows of 2048 + a top window of 1
    assert cnt["delta_out_of_range"] == 0 and cnt["mma_wait_failures"] == 0
    assert cnt["mma_products"] > 0, "the tensor-core range products never ran"


@pytest.mark.parametrize("M,n,count", [(16384, 8192, 96), (16384, 4096, 64), (12288, 8192, 48), (8196, 2048, 64),
                                       (16384, 64, 48)])
def test_directed_2p19(M, n, count):
    binding.debug_counters(reset=True)
    u, v = inputs.directed(M, n, count=count)
    check(u, v, "directed %d/%d" % (M, n))
    cnt = binding.debug_counters(reset=True)
    print("counters", cnt)
    assert cnt["delta_out_of_range"] == 0
    assert cnt["one_limb"] > 0 and cnt["u_lt_v"] > 0 and cnt["pow_b"] > 0


def test_paper_shape_2p19():
    """prec u = M - 2, prec v uniform in 2..M/2: long quotients, up to eight windows."""
    u, v = inputs.paper_shape(48, 16384)
    check(u, v, "paper shape 16384")


def test_head_kernel_on_and_off_2p19():
    """The head of Refine runs in its own kernel for the chunked form too (the inverse all windows share has t + 2 limbs:
    the head must plan for H = t + 1, not for h - k); with MPDIV_FLAG_NO_HEAD everything stays in the block."""
    assert binding.batch_launches(16384, 592) == 2
    assert binding.batch_launches(16384, 592, binding.VARIANT_CLIPPED | binding.FLAG_NO_HEAD) == 1
    u, v = inputs.directed(16384, 8192, count=64, seed=inputs.SEED + 5)
    check(u, v, "directed 16384/8192, head in the block", flags=binding.VARIANT_CLIPPED | binding.FLAG_NO_HEAD)
    check(u, v, "directed 16384/8192, no seed", flags=binding.VARIANT_CLIPPED | binding.FLAG_NO_SEED)
    q = torch.empty((u.shape[0], 16384), dtype=torch.int32, device="cuda")
    r = torch.empty((u.shape[0], 8192), dtype=torch.int32, device="cuda")
    binding.mpdiv_batch_noalloc(dev(u), dev(v), q, r)                 # the static scratch serves the chunked form as well
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    assert (host(q) == qo).all() and (host(r) == ro).all() and binding.status(reset=True) == 0


def test_no_tensor_engine_2p19():
    u, v = inputs.uniform_operands(8, 16384, 8192, config=20)
    check(u, v, "uniform 16384/8192, IMAD only", flags=binding.VARIANT_CLIPPED | binding.FLAG_NO_MMA)


def test_window_boundaries():
    """Quotient lengths around multiples of the chunk, and running remainders of v - 1."""
    rng = inputs.rng_for(77, 3)
    M, n = 16384, 8192
    B = inputs.B
    us, vs = [], []

    def rnd(limbs):
        return inputs.from_limbs(rng.integers(0, 1 << 32, size=limbs, dtype=np.uint64).astype(np.uint32)) | (1 << (32 * limbs - 1))

    for lv in (8192, 5000, 2, 3, 2049):
        for D in (1, 2, T - 1, T, T + 1, 2 * T, 2 * T + 1, 3 * T - 1):
            h = lv - 1 + D                       # prec(u)
            if h > M or h < lv:
                continue
            v = rnd(lv)
            us.append(rnd(h)); vs.append(v)
            # u = q*v + (v - 1) with q = B^j - 1 patterns: every window's remainder is v - 1 or close to it
            q = (1 << (32 * (h - lv))) - 1
            us.append(q * v + (v - 1)); vs.append(v)
            # exact multiple whose low windows are all zero
            us.append((v << (32 * (h - lv))) if h - lv > 0 else v); vs.append(v)
    # one-limb divisors with dividends that fill every window
    for d in (1, 2, B - 1, 0x80000000, 12345):
        us.append(rnd(M)); vs.append(d)
        us.append((1 << (32 * M)) - 1); vs.append(d)
    keep = [(a, b) for a, b in zip(us, vs) if a < (1 << (32 * M)) and b < (1 << (32 * n))]
    u = inputs.ints_to_rows([a for a, _ in keep], M)
    v = inputs.ints_to_rows([b for _, b in keep], n)
    check(u, v, "window boundaries")


def test_zero_divisor_and_u_lt_v_2p19():
    u, v = inputs.uniform_operands(4, 16384, 8192, config=21)
    v[0, :] = 0                                   # v = 0: q = all ones, r = low limbs of u
    u[1, 8000:] = 0                               # u < v
    u[2, :] = 0                                   # u = 0
    binding.status(reset=True)
    q, r = binding.mpdiv_batch(dev(u), dev(v))
    assert binding.status(reset=True) == binding.STATUS_V_ZERO
    q, r = host(q), host(r)
    assert (q[0] == 0xFFFFFFFF).all() and (r[0] == u[0, :8192]).all()
    qo, ro = oracle.divmod_batch(u[1:], v[1:], threads=NCPU)
    assert (q[1:] == qo).all() and (r[1:] == ro).all()


def test_limits_2p19():
    z = torch.zeros((1, 16384), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.MpdivError) as e:                       # divisor stride above 8192
        binding.mpdiv_batch(z, torch.ones((1, 8196), dtype=torch.int32, device="cuda"))
    assert e.value.code == binding.ERR_UNSUPPORTED
    with pytest.raises(binding.MpdivError) as e:                       # the printed variant needs the operands on chip
        binding.mpdiv_batch(z, torch.ones((1, 4096), dtype=torch.int32, device="cuda"), variant=binding.VARIANT_PRINTED)
    assert e.value.code == binding.ERR_UNSUPPORTED
