"""mpdiv_batch_noalloc (include/mpdiv.h): the division entry point that allocates nothing -- its scratch (the rows
through which the head-of-Refine kernel hands its iterates to the division kernel) is a static device array
inside the library instead of a stream-ordered pool allocation.

Collected last on purpose (the suite runs with pytest -x).  The result must equal the existing path's
(mpdiv_batch) limb for limb -- q and r are unique, so the tolerance is zero, as everywhere in this suite -- on two
calls in a row that share the scratch, the second on other inputs so that anything it wrongly kept from the first
would show.  Passes alone in a fresh process and after the other tests (it touches no state of theirs).
"""
import numpy as np
import pytest
import torch

from paper_2606_06386_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def test_noalloc_matches_mpdiv_batch_on_two_calls_in_a_row():
    # config 2's shape (a throughput batch: the head kernel and with it the scratch are really used) and the
    # adversarial mix of config 5 (special cases that never read their scratch row sit between rows that do)
    assert binding.batch_launches(2048, 1184) == 2
    batches = [inputs.config(2), inputs.config(5), inputs.config(2, seed=inputs.SEED + 9)]
    binding.status(reset=True)
    for u, v in batches:
        du, dv = dev(u), dev(v)
        q_ref, r_ref = binding.mpdiv_batch(du, dv)                       # the existing path (pool allocation)
        q = torch.full_like(du, 0x5A5A5A5A)
        r = torch.full_like(dv, 0x5A5A5A5A)
        binding.mpdiv_batch_noalloc(du, dv, q, r)
        torch.cuda.synchronize()
        assert torch.equal(q, q_ref) and torch.equal(r, r_ref)
    assert binding.status(reset=True) == 0


def test_noalloc_small_and_latency_batches():
    """Batches that run without the head kernel (no scratch used at all) go through the same entry point."""
    for u, v in (inputs.config(1), inputs.directed(64, 32, count=256)):
        du, dv = dev(u), dev(v)
        q_ref, r_ref = binding.mpdiv_batch(du, dv)
        q, r = torch.empty_like(du), torch.empty_like(dv)
        binding.mpdiv_batch_noalloc(du, dv, q, r)
        torch.cuda.synchronize()
        assert torch.equal(q, q_ref) and torch.equal(r, r_ref)


def test_noalloc_rejects_batches_beyond_its_static_scratch():
    n = binding.NOALLOC_MAX_BATCH + 1
    u = torch.ones((n, 8), dtype=torch.int32, device="cuda")
    v = torch.ones((n, 4), dtype=torch.int32, device="cuda")
    q, r = torch.empty_like(u), torch.empty_like(v)
    with pytest.raises(binding.MpdivError) as e:
        binding.mpdiv_batch_noalloc(u, v, q, r)
    assert e.value.code == binding.ERR_TOO_LARGE and "MPDIV_NOALLOC_MAX_BATCH" in str(e.value)
    binding.mpdiv_batch_noalloc(u[:-1], v[:-1], q[:-1], r[:-1])          # the maximum itself is accepted
    torch.cuda.synchronize()
    assert bool((q[:-1, 0] == 1).all()) and not bool(r[:-1].any())     # 1 / 1 = 1 remainder 0
