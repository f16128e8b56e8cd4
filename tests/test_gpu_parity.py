"""Parity of the CUDA path (libmpdiv.so through the C ABI) with the CPU oracle -- bit exact.

Every test here needs a B200 (``-m gpu``).  Inputs come from the seeded generators of
``paper_2606_06386_b200.inputs``; expected values come from ``oracle/`` only.  q and r are
unique, so every limb including the zero padding must match.  For shinv_batch the
two admissible values floor(B^h/v) + {0, 1} (Theorem 2) are both accepted; the clipped
variant behind shinv_batch_ex may also return floor(B^h/v) - 1.
"""
import os

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_06386_b200 import binding, inputs

pytestmark = pytest.mark.gpu

NCPU = max(1, os.cpu_count() or 1)


def dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


PRINTED, CLIPPED = binding.VARIANT_PRINTED, binding.VARIANT_CLIPPED
VARIANTS = [pytest.param(CLIPPED, id="clipped"), pytest.param(PRINTED, id="printed")]


def gpu_div(u, v, variant=None, allow=0):
    """One batch through the C ABI; afterwards the sticky status word must be clean (mpdiv_status: no pipeline
    wait gave up, no correction loop hit its bound, the clipped remainder stayed in range), except for the
    bits in `allow` (a test that feeds v = 0 allows STATUS_V_ZERO)."""
    binding.status(reset=True)
    q, r = binding.mpdiv_batch(dev(u), dev(v), variant=variant)
    st = binding.status(reset=True)
    assert st & ~allow == 0, "mpdiv_status = %#x after the batch" % st
    return host(q), host(r)


def check_div(u, v, what="", variant=None):
    q, r = gpu_div(u, v, variant)
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    bad = np.nonzero((q != qo).any(axis=1) | (r != ro).any(axis=1))[0]
    assert bad.size == 0, "%s: %d of %d instances differ, first %d" % (what, bad.size, u.shape[0], bad[0])


# ------------------------------------------------------------------ multiplication
@pytest.mark.parametrize("an,bn,cn", [
    (4, 4, 8), (8, 8, 16), (12, 20, 32), (64, 64, 128), (512, 512, 1024), (516, 260, 776),
    (1024, 1024, 2048), (2048, 1024, 3072), (4096, 4096, 8192), (8192, 4096, 12288),
    (1024, 1024, 1024), (1024, 1024, 516), (2048, 2048, 1028), (4096, 4096, 4096), (520, 516, 524),
    (64, 64, 4), (8192, 8192, 16384), (8192, 8192, 8192),
])
def test_mul_parity(an, bn, cn):
    batch = 12
    rng = inputs.rng_for(200, an % 65536)
    a = inputs._uniform(rng, batch, an)
    b = inputs._uniform(rng, batch, bn)
    # ragged effective precisions, all-ones (worst carries) and zero operands
    a[1, an // 2:] = 0
    b[2, max(1, bn // 3):] = 0
    a[3, :] = 0xFFFFFFFF
    b[3, :] = 0xFFFFFFFF
    a[4, :] = 0
    b[5, :] = 0
    a[6, 1:] = 0
    b[7, 1:] = 0
    a[8, :] = 0xFFFFFFFF
    b[8, :] = 0
    b[8, 0] = 1
    c = host(binding.mpmul_batch(dev(a), dev(b), cn))
    co = oracle.mul_batch(a, b, cn)
    bad = np.nonzero((c != co).any(axis=1))[0]
    assert bad.size == 0, "instances %s differ" % bad[:8]


@pytest.mark.parametrize("an,bn,cn", [
    (1024, 1024, 2048), (2048, 2048, 4096), (4096, 4096, 8192), (4096, 4096, 4096), (8192, 4096, 4132),
    (32, 32, 64), (100, 36, 136), (36, 1000, 1036), (4096, 4100, 8196), (2052, 2080, 4132), (8192, 4096, 8192),
])
def test_mul_tensor_engine_parity(an, bn, cn):
    """The int8 tcgen05 engine (csrc/mp_mma.cuh) must give the same limbs as the schoolbook oracle."""
    batch = 10
    rng = inputs.rng_for(210, an % 65536)
    a = inputs._uniform(rng, batch, an)
    b = inputs._uniform(rng, batch, bn)
    a[1, an // 2:] = 0
    b[2, max(1, bn // 3):] = 0
    a[3, :] = 0xFFFFFFFF                      # largest byte-column sums and longest carry chains
    b[3, :] = 0xFFFFFFFF
    a[4, :] = 0
    b[5, 1:] = 0
    a[6, :] = 0xFFFFFFFF
    b[6, :] = 0
    b[6, 0] = 1
    binding.debug_counters(reset=True)
    c = host(binding.mpmul_batch(dev(a), dev(b), cn, engine=binding.ENGINE_TENSOR))
    co = oracle.mul_batch(a, b, cn)
    bad = np.nonzero((c != co).any(axis=1))[0]
    assert bad.size == 0, "instances %s differ" % bad[:8]
    assert binding.debug_counters(reset=True)["mma_wait_failures"] == 0


def test_mul_tensor_engine_refuses_what_does_not_fit():
    a = torch.zeros((1, 8192), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.MpdivError) as e:
        binding.mpmul_batch(a, a, 16384, engine=binding.ENGINE_TENSOR)     # 512 blocks fit TMEM, not shared memory
    assert e.value.code == binding.ERR_UNSUPPORTED


def test_div_uses_tensor_engine_at_2_18_bits():
    """Config 4 must really run its large range products on the tensor core (and get the oracle's answer:
    test_div_config_full_size checks that)."""
    u, v = inputs.config(4, batch=8)
    binding.debug_counters(reset=True)
    gpu_div(u, v)
    cnt = binding.debug_counters(reset=True)
    assert cnt["mma_products"] >= 2 * 8 and cnt["mma_wait_failures"] == 0


# ------------------------------------------------------------------ shifted inverse
@pytest.mark.parametrize("vn,h", [(4, 7), (8, 16), (16, 17), (64, 128), (512, 1024), (1024, 2048),
                                  (260, 777), (2048, 4096), (4096, 8192), (512, 512), (512, 300)])
@pytest.mark.parametrize("variant", [pytest.param(None, id="plain"), pytest.param(CLIPPED, id="clipped-ex"),
                                     pytest.param(PRINTED, id="printed-ex")])
def test_shinv_parity(vn, h, variant):
    """shinv_batch (no flags) is Theorem 2's value: lambda in {0, 1} ONLY."""
    batch = 24
    wn = (h + 1 + 3) // 4 * 4
    _, v = inputs.directed(max(vn, 8), vn, count=batch, seed=inputs.SEED + h)
    v2 = inputs._uniform(inputs.rng_for(201, h % 65536), 8, vn)
    inputs._force_top_nonzero(v2)
    v = np.concatenate([v, v2])
    binding.status(reset=True)
    w = host(binding.shinv_batch(dev(v), h, wn, variant=variant))
    assert binding.status(reset=True) & ~binding.STATUS_V_ZERO == 0
    wo = oracle.shinv_batch(v, h, wn)
    allowed = (-1, 0, 1) if variant == CLIPPED else (0, 1)      # Theorem 2; one more unit when clipped
    lam_hist = {-1: 0, 0: 0, 1: 0}
    for i in range(v.shape[0]):
        if not v[i].any():
            continue                                            # v = 0: undefined (all ones, status bit)
        lam = inputs.from_limbs(w[i]) - inputs.from_limbs(wo[i])
        assert lam in allowed, "instance %d: lambda = %d (allowed %s)" % (i, lam, allowed)
        lam_hist[lam] += 1
    print("lambda histogram", lam_hist)


@pytest.mark.parametrize("vn,h", [(8, 16), (32, 64), (64, 128), (128, 256), (256, 512), (260, 400), (512, 1024), (512, 530)])
def test_shinv_matches_the_flow_model(vn, h):
    """tests/clipped_flow_model.py claims to replay the shipped clipped flow window for window.  Tie it to the
    kernels: shinv_batch_ex(MPDIV_VARIANT_CLIPPED) (IMAD engine: shinv_kernel carries no tensor-core code) must
    return the model's value LIMB FOR LIMB -- not just something within one unit of floor(B^h / v) -- on directed
    and uniform divisors, with and without the 17-digit seed."""
    import clipped_flow_model as model

    wn = (h + 1 + 3) // 4 * 4
    _, v = inputs.directed(max(vn, 8), vn, count=96, seed=inputs.SEED + 5 * h)
    v2 = inputs._uniform(inputs.rng_for(202, h % 65536), 16, vn)
    inputs._force_top_nonzero(v2)
    v = np.concatenate([v, v2])
    for flags, seed in ((CLIPPED, True), (CLIPPED | binding.FLAG_NO_SEED, False)):
        w = host(binding.shinv_batch(dev(v), h, wn, variant=flags))
        for i in range(v.shape[0]):
            vi = inputs.from_limbs(v[i])
            if vi == 0:
                continue
            if vi < (1 << 32):                      # one-limb divisor: Shinv(v*B, h+1)
                want = model.shinv(vi << 32, h + 1, seed=seed)
            else:
                want = model.shinv(vi, h, seed=seed)
            assert inputs.from_limbs(w[i]) == want, "instance %d (seed %s): kernel and model differ" % (i, seed)


# ------------------------------------------------------------------ division: the five configs
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_div_config_full_size(cfg, variant):
    """BASELINE.json configs at full size, in the launch configuration bench.py times.

    Configs 1-2 and 5 are checked on every instance; 3 and 4 (oracle: tens of ms per division)
    on a seeded sample of instances, each compared limb by limb."""
    u, v = inputs.config(cfg)
    q, r = gpu_div(u, v, variant)
    batch = u.shape[0]
    if cfg in (3, 4):
        pick = np.sort(inputs.rng_for(300 + cfg).choice(batch, size=96 if cfg == 3 else 48, replace=False))
    else:
        pick = np.arange(batch)
    qo, ro = oracle.divmod_batch(u[pick], v[pick], threads=NCPU)
    bad = np.nonzero((q[pick] != qo).any(axis=1) | (r[pick] != ro).any(axis=1))[0]
    assert bad.size == 0, "config %d: %d of %d checked instances differ (first: %d)" % (
        cfg, bad.size, pick.size, pick[bad[0]])


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("cfg", [3, 4])
def test_div_config_invariants_all_instances(cfg, variant):
    """Properties that hold at any size, on EVERY instance of the big configs:
    r < v limb-wise compare and u = q*v + r checked with Python integers (independent of both sides)."""
    u, v = inputs.config(cfg)
    q, r = gpu_div(u, v, variant)
    step = 1 if cfg == 3 else 1
    for i in range(0, u.shape[0], step):
        ui, vi = inputs.from_limbs(u[i]), inputs.from_limbs(v[i])
        qi, ri = inputs.from_limbs(q[i]), inputs.from_limbs(r[i])
        assert ri < vi and qi * vi + ri == ui, "instance %d" % i


# ------------------------------------------------------------------ division: directed and ragged
@pytest.mark.parametrize("M,n,count", [(8, 4, 256), (16, 8, 512), (32, 32, 512), (64, 32, 512),
                                       (128, 64, 512), (1024, 512, 768), (2048, 1024, 384),
                                       (2048, 2048, 384), (4096, 2048, 128), (8192, 4096, 48),
                                       (8192, 8192, 32), (1028, 516, 256), (100, 52, 256)])
@pytest.mark.parametrize("variant", VARIANTS)
def test_div_directed(M, n, count, variant):
    if variant == PRINTED and M + n > 12288:
        with pytest.raises(binding.MpdivError) as e:     # the 2M-limb product does not fit on chip
            gpu_div(*inputs.directed(M, n, count=2), variant)
        assert e.value.code == binding.ERR_UNSUPPORTED
        return
    binding.debug_counters(reset=True)
    u, v = inputs.directed(M, n, count=count)
    check_div(u, v, "directed M=%d n=%d" % (M, n), variant)
    cnt = binding.debug_counters()
    print("counters", cnt)
    assert cnt["delta_out_of_range"] == 0
    if variant == PRINTED:
        assert cnt["delta_multi"] == 0, "a quotient needed more than one +1 step (Theorem 2 violated)"
        assert cnt["delta_neg_multi"] == 0 and cnt["clipped_steps"] == 0


@pytest.mark.parametrize("M,n,count", [(1024, 512, 4096), (2048, 1024, 4096), (2048, 2048, 2048), (4096, 2048, 2048),
                                       (8192, 4096, 512)])
def test_div_directed_large_sets(M, n, count):
    """The directed set at the size SURVEY 8(d) asks for (thousands per size) on the default variant: the clipped
    products, the "+1" Refine loop and the tensor-core range products must leave every quotient within reach of
    the correction loops."""
    binding.debug_counters(reset=True)
    u, v = inputs.directed(M, n, count=count, seed=inputs.SEED + 17)
    check_div(u, v, "directed (large set) M=%d n=%d" % (M, n))
    cnt = binding.debug_counters(reset=True)
    print("counters", cnt)
    assert cnt["delta_out_of_range"] == 0 and cnt["mma_wait_failures"] == 0


@pytest.mark.parametrize("variant", VARIANTS)
def test_directed_reaches_corner_paths(variant):
    """The directed set must actually drive the rare branches: delta = -1, delta = +1,
    the negative PowDiff sign, powers of B and one-limb divisors."""
    binding.debug_counters(reset=True)
    u, v = inputs.directed(64, 32, count=2048)
    check_div(u, v, "directed 64/32", variant)
    u, v = inputs.directed(512, 256, count=1024)       # long enough for the clipped windows to bite
    check_div(u, v, "directed 512/256", variant)
    cnt = binding.debug_counters(reset=True)
    print("counters", cnt)
    for key in ("delta_neg", "delta_pos", "sign_neg", "pow_b", "one_limb", "u_lt_v", "tiles"):
        assert cnt[key] > 0, "%s never fired" % key
    assert cnt["delta_out_of_range"] == 0
    if variant == PRINTED:
        assert cnt["delta_multi"] == 0 and cnt["clipped_steps"] == 0
    else:
        assert cnt["clipped_steps"] > 0


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("M", [64, 1024, 2048, 8192])
def test_div_paper_shape(M, variant):
    """The paper's own workload shape: prec(u) = M-2, prec(v) uniform in 2..M/2."""
    u, v = inputs.paper_shape(256 if M < 8192 else 48, M)
    check_div(u, v, "paper shape M=%d" % M, variant)


@pytest.mark.parametrize("variant", VARIANTS)
def test_div_random_effective_precisions(variant):
    """1000 randomised instances with random values and random effective precisions."""
    rng = inputs.rng_for(400)
    M = 256
    us, vs = [], []
    for _ in range(1000):
        lu = int(rng.integers(0, M + 1))
        lv = int(rng.integers(1, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    check_div(inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, M), "random precisions", variant)


@pytest.mark.parametrize("variant", VARIANTS)
def test_div_random_effective_precisions_large(variant):
    """Random effective precisions at the 2^16-bit stride: every clipping window position occurs."""
    rng = inputs.rng_for(401)
    M = 2048
    us, vs = [], []
    for _ in range(400):
        lv = int(rng.integers(1, M + 1))
        lu = int(rng.integers(0, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    check_div(inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, M), "random precisions 2048", variant)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("M,n,threads", [(8, 4, 32), (32, 32, 32), (64, 32, 32), (128, 64, 32), (256, 128, 32), (512, 256, 32),
                                         (1024, 512, 32), (1024, 512, 64), (512, 512, 64), (100, 52, 32)])
def test_div_one_warp_per_division(M, n, threads, variant):
    """small numbers in large batches get one warp (32-thread blocks) or two per division instead of a
    128-thread block.  Forced here through MPDIV_FLAG_THREADS on the directed set; every primitive runs
    in its warp form."""
    u, v = inputs.directed(M, n, count=768)
    check_div(u, v, "directed M=%d n=%d T=%d" % (M, n, threads), variant | binding.flag_threads(threads))


@pytest.mark.parametrize("M,n,batch", [(64, 32, 4736), (256, 128, 4736), (512, 256, 2400), (1024, 512, 1200)])
def test_div_small_numbers_large_batches_default_mapping(M, n, batch):
    """The mapping mpdiv_batch picks by itself for batches of at least 16 (8) divisions per SM: random effective
    precisions, default variant."""
    rng = inputs.rng_for(402, M)
    us, vs = [], []
    for i in range(batch):
        lv = int(rng.integers(1, n + 1))
        lu = int(rng.integers(0, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    check_div(inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, n), "random precisions %d/%d x %d" % (M, n, batch))


def test_div_uses_tensor_engine_at_2_16_bits_in_throughput_batches_only():
    """128-thread blocks: a throughput batch of config 2's shape runs its large range products on the tensor core
    (warp 0 produces and issues, mp_mma.cuh); the latency kernel of a small batch is compiled without the engine.
    Both must give the oracle's answer."""
    u, v = inputs.config(2, batch=592)                  # more than two blocks per SM: throughput kernel
    binding.debug_counters(reset=True)
    check_div(u, v, "config 2 shape, throughput batch")
    cnt = binding.debug_counters(reset=True)
    assert cnt["mma_products"] >= 2 * 592 and cnt["mma_wait_failures"] == 0
    check_div(u[:64], v[:64], "config 2 shape, latency batch")
    cnt = binding.debug_counters(reset=True)
    assert cnt["mma_products"] == 0


@pytest.mark.parametrize("M,count", [(2048, 600), (4096, 240), (8192, 96)])
def test_div_random_effective_precisions_tensor_sizes(M, count):
    """Random effective precisions at the strides whose kernels carry the tensor-core engine: every shape of
    range product (and every decision of mma_plan) occurs, including operands far from 32-limb multiples."""
    rng = inputs.rng_for(402, M % 65536)
    us, vs = [], []
    for i in range(count):
        if i % 3 == 0:          # balanced: the shapes that do reach the tensor core
            lu = int(rng.integers(M - 600, M + 1))
            lv = int(rng.integers(lu // 2 - 300, lu // 2 + 300))
        else:
            lv = int(rng.integers(1, M + 1))
            lu = int(rng.integers(0, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, max(1, lv)))
    binding.debug_counters(reset=True)
    check_div(inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, M), "random precisions %d" % M)
    cnt = binding.debug_counters(reset=True)
    print("counters", cnt)
    assert cnt["mma_products"] > 0 and cnt["mma_wait_failures"] == 0 and cnt["delta_out_of_range"] == 0


def test_div_zero_divisor_does_not_trap():
    binding.debug_counters(reset=True)
    u, v = inputs.uniform_operands(8, 64, 32, config=77)
    v[3] = 0
    binding.status(reset=True)
    binding.mpdiv_batch(dev(u), dev(v))
    assert binding.status(reset=True) == binding.STATUS_V_ZERO      # undefined input is reported, not hidden
    q, r = gpu_div(u, v, allow=binding.STATUS_V_ZERO)
    assert (q[3] == 0xFFFFFFFF).all() and (r[3] == u[3, :32]).all()
    keep = [0, 1, 2, 4, 5, 6, 7]
    qo, ro = oracle.divmod_batch(u[keep], v[keep])
    assert (q[keep] == qo).all() and (r[keep] == ro).all()
    assert binding.debug_counters(reset=True)["v_zero"] == 2         # the batch ran twice


@pytest.mark.parametrize("M,n", [(8, 16), (64, 128), (512, 1024), (2048, 4096), (1024, 8192)])
def test_div_divisor_stride_longer_than_dividend(M, n):
    """v_limbs > u_limbs is allowed: a divisor that is really longer gives (0, u); one whose
    effective precision fits inside u's stride divides as usual.  r has the divisor's stride."""
    rng = inputs.rng_for(420, n % 65536)
    us, vs = [], []
    for i in range(96):
        lu = int(rng.integers(0, M + 1))
        lv = int(rng.integers(1, n + 1)) if i % 2 else int(rng.integers(1, M + 1))
        us.append(inputs._random_int(rng, lu))
        vs.append(inputs._random_int(rng, lv))
    u, v = inputs.ints_to_rows(us, M), inputs.ints_to_rows(vs, n)
    q, r = gpu_div(u, v)
    assert q.shape == (96, M) and r.shape == (96, n)
    for i in range(96):
        qi, ri = divmod(us[i], vs[i])          # Python integers: the strides differ, so the limb oracle is
        assert inputs.from_limbs(q[i]) == qi and inputs.from_limbs(r[i]) == ri, i   # called below on the padded u
    up = np.zeros((96, n), dtype=np.uint32)
    up[:, :M] = u
    qo, ro = oracle.divmod_batch(up, v, threads=NCPU)
    assert (qo[:, :M] == q).all() and not qo[:, M:].any() and (ro == r).all()


def test_host_buffer_form_matches():
    u, v = inputs.config(1)
    ut = torch.from_numpy(u.view(np.int32)).pin_memory()
    vt = torch.from_numpy(v.view(np.int32)).pin_memory()
    qt = torch.empty_like(ut).pin_memory()
    rt = torch.empty_like(vt).pin_memory()
    ws = torch.empty(binding.host_workspace_bytes(u.shape[1], v.shape[1], u.shape[0]), dtype=torch.uint8, device="cuda")
    binding.mpdiv_batch_host(ut, vt, qt, rt, ws)
    torch.cuda.synchronize()
    qo, ro = oracle.divmod_batch(u, v, threads=NCPU)
    assert (qt.numpy().view(np.uint32) == qo).all() and (rt.numpy().view(np.uint32) == ro).all()


def test_bad_arguments_are_rejected():
    u, v = inputs.uniform_operands(2, 8, 4, config=78)
    du, dv = dev(u), dev(v)
    with pytest.raises(binding.MpdivError) as e:
        binding.mpdiv_batch(du[:, :6].contiguous(), dv)           # stride not a multiple of 4
    assert e.value.code == binding.ERR_BAD_ARG
    big = torch.zeros((1, 16388), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.MpdivError) as e:
        binding.mpdiv_batch(big, dv[:1])
    assert e.value.code == binding.ERR_UNSUPPORTED
