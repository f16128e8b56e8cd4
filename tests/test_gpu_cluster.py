"""A thread-block cluster per division: batches far smaller than the GPU run
every division on 2, 4 or 8 CTAs that share the tile diagonals of each product through distributed shared memory
(csrc/mp_mul.cuh "cluster").  Bit exact against the oracle; a counter proves the cluster path ran."""
import os

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_06386_b200 import binding, inputs

pytestmark = pytest.mark.gpu

NCPU = max(1, os.cpu_count() or 1)
PRINTED, CLIPPED = binding.VARIANT_PRINTED, binding.VARIANT_CLIPPED


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host(t):
    return t.cpu().numpy().view(np.uint32)


def run_small_batches(u, v, flags, per_call):
    """The rows `per_call` at a time (each call is its own small batch); returns q, r and the counters."""
    binding.status(reset=True)
    binding.debug_counters(reset=True)
    qs, rs = [], []
    for lo in range(0, u.shape[0], per_call):
        q, r = binding.mpdiv_batch(dev(u[lo:lo + per_call]), dev(v[lo:lo + per_call]), variant=flags)
        qs.append(host(q))
        rs.append(host(r))
    assert binding.status(reset=True) == 0
    return np.concatenate(qs), np.concatenate(rs), binding.debug_counters(reset=True)


def check(u, v, flags, per_call, what, expect_cluster=True):
    q, r, cnt = run_small_batches(u, v, flags, per_call)
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    bad = np.nonzero((q != qo).any(axis=1) | (r != ro).any(axis=1))[0]
    assert bad.size == 0, "%s: %d of %d instances differ, first %d" % (what, bad.size, u.shape[0], bad[0])
    assert cnt["delta_out_of_range"] == 0
    return cnt


def test_config1_runs_on_clusters():
    """BASELINE config 1 (32 divisions of 2^15 bits) through plain mpdiv_batch: every division on a cluster."""
    u, v = inputs.config(1)
    binding.status(reset=True)
    binding.debug_counters(reset=True)
    q, r = binding.mpdiv_batch(dev(u), dev(v))
    assert binding.status(reset=True) == 0
    cnt = binding.debug_counters(reset=True)
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    assert (host(q) == qo).all() and (host(r) == ro).all()
    assert cnt["cluster_divs"] == u.shape[0], cnt
    assert cnt["seeds"] == u.shape[0], "counters must count a division once, not once per CTA"


@pytest.mark.parametrize("variant", [pytest.param(CLIPPED, id="clipped"), pytest.param(PRINTED, id="printed")])
@pytest.mark.parametrize("cs", [2, 4, 8])
@pytest.mark.parametrize("M,n", [(1024, 512), (2048, 1024), (512, 512), (260, 132)])
def test_directed_on_clusters(M, n, cs, variant):
    u, v = inputs.directed(M, n, count=144)
    per_call = 148 // cs - 2
    cnt = check(u, v, variant | binding.flag_cluster(cs), per_call, "directed %d/%d cluster %d" % (M, n, cs))
    nontrivial = u.shape[0] - cnt["u_lt_v"] - cnt["v_zero"]
    assert cnt["cluster_divs"] == nontrivial, cnt


def test_cluster_off_switch_and_larger_batches():
    u, v = inputs.directed(1024, 512, count=96)
    cnt = check(u, v, CLIPPED | binding.FLAG_NO_CLUSTER, 16, "no-cluster flag")
    assert cnt["cluster_divs"] == 0
    cnt = check(u, v, CLIPPED, 96, "a batch that does not fit clusters")      # 96 x 2 CTAs > 148 SMs
    assert cnt["cluster_divs"] == 0


def test_random_precisions_on_clusters():
    rng = inputs.rng_for(403)
    M = 1024
    us, vs = [], []
    for _ in range(180):
        lv = int(rng.integers(1, M + 1))
        lu = int(rng.integers(0, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    check(inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, M), CLIPPED, 18, "random precisions on clusters")
