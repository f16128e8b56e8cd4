"""Randomised sweep over every mapping of mpdiv_batch in one place: the chunked form for 2^19-bit dividends, a
thread-block cluster per division, one warp per division, and the resident tensor-core path -- directed sets and random
effective precisions drawn with a few seeds, bit exact against the oracle, status word clean."""
import os

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_06386_b200 import binding, inputs

pytestmark = pytest.mark.gpu

NCPU = max(1, os.cpu_count() or 1)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host(t):
    return t.cpu().numpy().view(np.uint32)


def check(u, v, flags, what, per_call=None):
    binding.status(reset=True)
    per = per_call or u.shape[0]
    qs, rs = [], []
    for lo in range(0, u.shape[0], per):
        q, r = binding.mpdiv_batch(dev(u[lo:lo + per]), dev(v[lo:lo + per]), variant=flags)
        qs.append(host(q))
        rs.append(host(r))
    st = binding.status(reset=True)
    assert st & ~binding.STATUS_V_ZERO == 0, "%s: mpdiv_status = %#x" % (what, st)
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    bad = np.nonzero((np.concatenate(qs) != qo).any(axis=1) | (np.concatenate(rs) != ro).any(axis=1))[0]
    assert bad.size == 0, "%s: %d of %d instances differ, first %d" % (what, bad.size, u.shape[0], bad[0])


def random_precisions(rng, count, M, n):
    us, vs = [], []
    for _ in range(count):
        us.append(inputs._random_int(rng, int(rng.integers(0, M + 1))))
        vs.append(inputs._random_int(rng, int(rng.integers(1, n + 1))))
    return inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, n)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_every_mapping(seed):
    rng = inputs.rng_for(900 + seed, 7)
    s = inputs.SEED + 1000 + seed
    for M, n, c in [(16384, 8192, 24), (16384, 2048, 24), (9000, 8192, 24), (12288, 4100, 24)]:       # chunked form
        check(*inputs.directed(M, n, count=c, seed=s), None, "chunked, directed %d/%d" % (M, n))
        check(*random_precisions(rng, c, M, n), None, "chunked, random precisions %d/%d" % (M, n))
    for M, n in [(1024, 512), (2048, 1024), (1500, 700)]:                                              # clusters
        check(*inputs.directed(M, n, count=144, seed=s), None, "clusters, directed %d/%d" % (M, n), per_call=24)
        u, v = random_precisions(rng, 96, M, n)
        check(u, v, binding.VARIANT_CLIPPED | binding.flag_cluster(2), "2-CTA clusters %d/%d" % (M, n), per_call=48)
        check(u, v, binding.VARIANT_CLIPPED | binding.flag_cluster(8), "8-CTA clusters %d/%d" % (M, n), per_call=16)
    for M, n in [(32, 16), (128, 128), (256, 100), (512, 256), (1024, 512)]:                           # warp per division
        check(*random_precisions(rng, 2500, M, n), None, "warp mapping, random precisions %d/%d" % (M, n))
        check(*inputs.directed(M, n, count=600, seed=s), binding.VARIANT_CLIPPED | binding.flag_threads(32),
              "32 threads, directed %d/%d" % (M, n))
    for M, n, c in [(2048, 1024, 1300), (4096, 2048, 400), (8192, 4096, 160)]:                        # resident tensor path
        check(*inputs.directed(M, n, count=c, seed=s), None, "directed %d/%d" % (M, n))
        check(*random_precisions(rng, c // 2, M, n), None, "random precisions %d/%d" % (M, n))
