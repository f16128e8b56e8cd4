#!/usr/bin/env python
"""bench.py -- divisions/sec of mpdiv_batch on B200, with the integer-multiply roofline, the
division/multiplication cost ratios and the CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference] [--brief]

A "step" is one pass of the whole hot path (load, Shinv/Refine, quotient, back-multiply, correction,
store: SURVEY.md 8(a) rows a1-a12 = one mpdiv_batch call) over one batch of the workload.  The
default workload is BASELINE.json configs[1]: 1184 divisions of a 2^16-bit by a 2^15-bit number.
Rank 0 prints ONE JSON line.  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "divisions/sec at 2^15..2^18 bits; % int-multiply roofline; div/mul cost ratio"
UNIT = "divisions/s"

# Algorithmic work per division W(M): limb products (32x32->64) of the method as printed (Alg. 1-3 with
# exact operand sizes, truncated products counted truncated), u = M limbs, v = M/2 limbs.
# SURVEY.md 8(d) / DESIGN.md "Roofline"; fixed constants, not measured.
W_LIMB_PRODUCTS = {1024: 1898264, 2048: 7553425, 4096: 30136284, 8192: 120394683}

# Nominal 32-bit integer multiply-add issue rate: 4 SMSPs x 16 lanes per clock
# per SM (IMAD on the fma pipe, reciprocal throughput 2 cycles per warp instruction per SMSP).
IMAD_PER_CLK_PER_SM = 64
FLUSH_BYTES = 256 << 20   # > 126 MB of L2

# ncu-derived figures (DRAM traffic per launch, kernel share of a step, pipe activity) are NOT measured by this
# script: they are read from a committed summary that names the commit and the command it was captured with
# (profiles/ncu_summary.json, written from the .ncu-rep files by hand-run ncu exports), or reported as null.
NCU_SUMMARY = os.path.join(ROOT, "profiles", "ncu_summary.json")


def ncu_summary(cfg: int):
    try:
        with open(NCU_SUMMARY) as f:
            doc = json.load(f)
        row = doc.get("configs", {}).get(str(cfg))
        if row is None:
            return None
        return dict(row, commit=doc.get("commit"), source="profiles/ncu_summary.json (captured at that commit; "
                    "per-launch times under ncu are cold-cache and serialised: compare shares, not absolutes)")
    except (OSError, ValueError):
        return None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=25)      # the paper's run count
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config 1..5 (default 2 = configs[1])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--brief", action="store_true", help="skip the per-config table and the CPU baseline")
    return ap.parse_args()


def workload_name(cfg: int) -> str:
    from paper_2606_06386_b200 import inputs

    b, m, n = inputs.CONFIG_SHAPES[cfg]
    kind = "adversarial mix" if cfg == 5 else "uniform limbs"
    return "config %d: %d divisions, u %d limbs (2^%d bits) / v %d limbs, %s, seed %d" % (
        cfg, b, m, (32 * m).bit_length() - 1, n, kind, inputs.SEED)


# ----------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            parts = [p.strip() for p in r.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                smax = float(parts[1])
            except ValueError:
                continue
            for name, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------------------------
# device timing helpers
# ----------------------------------------------------------------------------------------------
def time_steps(fn, steps: int, warmup: int, flush):
    """Run `fn` warmup + steps times on the current stream; each timed call is bracketed by its own
    pair of CUDA events on that stream and preceded by an L2 flush (outside the events).
    Returns the list of per-step milliseconds."""
    import torch

    for _ in range(warmup):
        flush()
        fn()
    torch.cuda.synchronize()
    evs = []
    for _ in range(steps):
        flush()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    return [e0.elapsed_time(e1) for e0, e1 in evs]


def to_dev(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def measure_imad_peak(binding, iters: int = 4000):
    """Limb products/s of the multiplier's own inner tile with no memory traffic (kind 0) and plain
    32-bit IMADs/s (kind 1), best of 5, on the current device."""
    import torch

    out = {}
    for kind, name in ((0, "imad_wide_chain"), (1, "imad_lo32")):
        best = None
        sink = None
        for _ in range(6):
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            prods, sink = binding.imad_probe(kind, iters, sink)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None or ms < best else best
        out[name] = prods / (best * 1e-3)
    return out


def measure_tensor_peak(binding, iters: int = 20000):
    """u8 x u8 multiply-accumulates per second of the tensor pipe, measured: two warps of one block per SM issue
    tcgen05.mma.kind::i8 (M = 128, N = 128, K = 32) back to back into disjoint accumulators (mpdiv_mma_probe);
    best of 5 launches timed with events.  Nominal: 8192 MAC per clock per SM."""
    import torch

    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    macs = binding.mma_probe_macs(128, 2, iters)
    best = None
    for _ in range(6):
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        binding.mma_probe_launch(128, 2, iters, out)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None or ms < best else best
    assert int(out.min().item()) > 0, "mpdiv_mma_probe: a bounded wait gave up"
    return macs / (best * 1e-3)


def measure_mma_issue(binding):
    """Cycles per tcgen05.mma (M = 128, K = 32, u8) seen by one issuing warp and by two (mpdiv_mma_probe): the
    tensor core needs N / 2; the rest is the issue path."""
    out = {}
    for n in (16, 48, 64, 96, 128):
        one = binding.mma_probe(n, 1)
        two = binding.mma_probe(n, 2)
        ss = binding.mma_probe(n, 1, form=1)
        out["N=%d" % n] = {"one_warp_cycles_per_mma": one[0], "two_warps_cycles_per_mma_together": max(two) / 2.0,
                           "toeplitz_descriptor_form_cycles_per_mma": ss[0], "shared_memory_model_cycles": max(32 + n / 4.0, n / 2.0),
                           "tensor_core_cycles_per_mma": n / 2.0}
    return out


def cpu_baseline(cfg: int, target_core_seconds: float = 16.0):
    """The oracle as it stands (Knuth D, one instance per call, batch split over host threads), timed on a
    bounded sample of the same workload: whole passes over the first instances of the batch until about
    `target_core_seconds` of CPU work have been spent."""
    from oracle import oracle
    from paper_2606_06386_b200 import inputs

    cores = max(1, os.cpu_count() or 1)
    b, m, n = inputs.CONFIG_SHAPES[cfg]
    u, v = inputs.config(cfg)
    probe = min(b, 4 * cores)
    t0 = time.perf_counter()
    oracle.divmod_batch(u[:probe], v[:probe], threads=cores)
    per = (time.perf_counter() - t0) / probe            # wall seconds per division with all cores busy
    wall = target_core_seconds / cores
    count = int(max(cores, min(b, wall / max(per, 1e-9))))
    passes = 0
    t0 = time.perf_counter()
    while True:                                         # whole passes until the core-second budget is spent
        oracle.divmod_batch(u[:count], v[:count], threads=cores)
        passes += 1
        dt = time.perf_counter() - t0
        if dt >= wall or passes >= 200:
            break
    return {"value": passes * count / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d passes over the first %d of %d instances of config %d, Knuth Algorithm D (oracle/knuth_d.c), "
                      "%d host threads, %.2f s wall (%.1f core-seconds)" % (passes, count, b, cfg, cores, dt, dt * cores)}


# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
MAC_PER_COLSTEP = 4 * 128 * 32      # one MMA step = 4 instructions of M = 128, K = 32 per accumulator column


def executed_work(binding, du, dv, q, r, variant=None):
    """What ONE launch really executes, counted by the kernels themselves (mpdiv_debug_counters): limb products on
    the IMAD pipe (8x8 tiles x 64, tile padding included) and u8 x u8 multiply-accumulates on the tensor pipe
    (MMA steps x accumulator columns x 16384, column padding included)."""
    import torch

    binding.debug_counters(reset=True)
    binding.mpdiv_batch(du, dv, q, r, variant=variant)
    torch.cuda.synchronize()
    c = binding.debug_counters(reset=True)
    return 64 * c["tiles"], MAC_PER_COLSTEP * c["mma_colsteps"], c


def pipe_fractions(imad_products, tensor_macs, ms, peaks):
    """Executed work / time / measured peak of each pipe, and which one is the (nearer) bound."""
    t = ms * 1e-3
    f_imad = imad_products / t / peaks["imad_wide_chain"]
    f_tc = tensor_macs / t / peaks["tensor_u8_mac"]
    return f_imad, f_tc, ("tensor" if f_tc >= f_imad else "alu")


def config_row(binding, cfg, flush, peaks):
    """divisions/s, both pipe fractions, the printed variant's work-conserving fraction and the cost ratios of
    SURVEY.md G12 for one config (25 timed runs each, the paper's count PAPER.md:476; median)."""
    import torch

    from paper_2606_06386_b200 import inputs

    b, m, n = inputs.CONFIG_SHAPES[cfg]
    u, v = inputs.config(cfg)
    du, dv = to_dev(u), to_dev(v)
    q = torch.empty_like(du)
    r = torch.empty_like(dv)
    med = lambda fn: float(np.median(time_steps(fn, 25, 3, flush)))   # noqa: E731
    t_div = med(lambda: binding.mpdiv_batch(du, dv, q, r))
    t_div_printed = med(lambda: binding.mpdiv_batch(du, dv, q, r, variant=binding.VARIANT_PRINTED))
    ex_imad, ex_tc, cnt_row = executed_work(binding, du, dv, q, r)
    exp_imad, exp_tc, _ = executed_work(binding, du, dv, q, r, variant=binding.VARIANT_PRINTED)
    f_imad, f_tc, bound = pipe_fractions(ex_imad, ex_tc, t_div, peaks)
    # R1 unit: M x M -> low M limbs (the paper's "full multiplication", M^2/2 limb products);
    # R2 unit: n x n -> 2n limbs; each on both engines
    a1 = to_dev(inputs._uniform(inputs.rng_for(500 + cfg, 0), b, m))
    b1 = to_dev(inputs._uniform(inputs.rng_for(500 + cfg, 1), b, m))
    c1 = torch.empty((b, m), dtype=torch.int32, device="cuda")
    nn = max(n if cfg != 5 else m // 2, 4)
    a2 = a1[:, :nn].contiguous()
    b2 = b1[:, :nn].contiguous()
    c2 = torch.empty((b, 2 * nn), dtype=torch.int32, device="cuda")
    t_m1 = med(lambda: binding.mpmul_batch(a1, b1, m, c1))
    t_m2 = med(lambda: binding.mpmul_batch(a2, b2, 2 * nn, c2))
    t_m1_tc = t_m2_tc = None
    try:
        t_m1_tc = med(lambda: binding.mpmul_batch(a1, b1, m, c1, engine=binding.ENGINE_TENSOR))
        t_m2_tc = med(lambda: binding.mpmul_batch(a2, b2, 2 * nn, c2, engine=binding.ENGINE_TENSOR))
    except binding.MpdivError:
        pass
    wl = (m + 1 + 3) // 4 * 4
    w = torch.empty((b, wl), dtype=torch.int32, device="cuda")
    t_sh = med(lambda: binding.shinv_batch(dv, m, wl, w))                                       # Theorem 2's value
    t_sh_clip = med(lambda: binding.shinv_batch(dv, m, wl, w, variant=binding.VARIANT_CLIPPED))  # what Div runs
    assert binding.status(reset=True) == 0, "mpdiv_status reported a fault during the per-config runs"
    row = {
        "batch": b, "u_limbs": m, "v_limbs": n, "bits": 32 * m,
        "div_ms": t_div, "div_per_s": b / (t_div * 1e-3), "us_per_div_latency": t_div * 1e3 if b <= 148 else None,
        "frac_imad_pipe": f_imad, "frac_tensor_pipe": f_tc, "bound": bound, "frac": max(f_imad, f_tc),
        "executed_limb_products_per_div": ex_imad / b, "executed_tensor_macs_per_div": ex_tc / b,
        "tensor_unit_occupancy": cnt_row["mma_unit_cycles"] / (peaks["sm_count"] * t_div * 1e-3 * peaks["sm_hz"]),
        "printed_div_per_s": b / (t_div_printed * 1e-3),
        "frac_printed": exp_imad / (t_div_printed * 1e-3) / peaks["imad_wide_chain"],
        "mul_MxM_lowM_ms": {"imad": t_m1, "tensor": t_m1_tc}, "mul_nxn_full_ms": {"imad": t_m2, "tensor": t_m2_tc},
        "shinv_ms": {"printed": t_sh, "clipped": t_sh_clip},
        # R1 = T(div) / T(M x M -> low M); the default division against BOTH multiplication engines, and the
        # printed division against the IMAD engine (the paper-comparable pairing: same engine on both sides)
        "R1": {"printed_div_over_imad_mul": t_div_printed / t_m1, "div_over_imad_mul": t_div / t_m1,
               "div_over_tensor_mul": (t_div / t_m1_tc) if t_m1_tc else None},
        "R2": {"printed_div_over_imad_mul": t_div_printed / t_m2, "div_over_imad_mul": t_div / t_m2,
               "div_over_tensor_mul": (t_div / t_m2_tc) if t_m2_tc else None},
        "shinv_over_mul_MxM_lowM": {"printed_over_imad": t_sh / t_m1,
                                    "clipped_over_tensor": (t_sh_clip / t_m1_tc) if t_m1_tc else None},
        "mul_imad_products_per_s": b * nn * nn / (t_m2 * 1e-3),
        "mul_tensor_products_per_s": (b * nn * nn / (t_m2_tc * 1e-3)) if t_m2_tc else None,
        "hbm_GBps_div_io": b * 4 * (2 * m + 2 * n) / (t_div * 1e-3) / 1e9,
    }
    if cfg != 5:
        row["W_limb_products"] = W_LIMB_PRODUCTS[m]
        row["speedup_vs_printed_work"] = row["div_per_s"] * W_LIMB_PRODUCTS[m] / peaks["imad_wide_chain"]
    return row


# The paper's own workload shape: prec(u) = M - 2, prec(v) uniform in 2..M/2, with the
# divisions/s derived from its Table 1 (A100, 64-bit digits) as context, not as the target.
PAPER_A100_DIV_PER_S = {2048: 165671, 4096: 46636, 8192: 11674}


def paper_shape_table(binding, flush):
    import torch

    from paper_2606_06386_b200 import inputs

    table = {}
    for m, b in ((2048, 2368), (4096, 1184), (8192, 592)):
        u, v = inputs.paper_shape(b, m)
        du, dv = to_dev(u), to_dev(v)
        q = torch.empty_like(du)
        r = torch.empty_like(dv)
        t = float(np.median(time_steps(lambda: binding.mpdiv_batch(du, dv, q, r), 25, 3, flush)))
        table["2^%d bits" % ((32 * m).bit_length() - 1)] = {
            "batch": b, "u_limbs": m, "v_stride": m // 2, "div_ms": t, "div_per_s": b / (t * 1e-3),
            "paper_A100_div_per_s_context": PAPER_A100_DIV_PER_S[m],
            "note": "prec(u) = M-2, prec(v) uniform in 2..M/2 (PAPER.md:474); the A100 figure is derived from the "
                    "paper's Table 1 (64-bit digits, other hardware): context only"}
        del du, dv, q, r
    return table


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2606_06386_b200 import binding, inputs, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = args.config
    b, m, n = inputs.CONFIG_SHAPES[cfg]
    # weak scaling: every rank divides its own batch of the config's size (independent problems,
    # no data-path collective); rank r draws with seed SEED + r.
    u, v = inputs.config(cfg, seed=shard.rank_seed(inputs.SEED, rank))
    du, dv = to_dev(u), to_dev(v)
    q = torch.empty_like(du)
    r = torch.empty_like(dv)
    flush_buf = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(rank & 0xFF)   # noqa: E731  (writes 256 MiB > L2)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    hu = torch.from_numpy(u.view(np.int32)).pin_memory()
    hv = torch.from_numpy(v.view(np.int32)).pin_memory()
    hq = torch.empty_like(hu).pin_memory()
    hr = torch.empty_like(hv).pin_memory()
    ws = torch.empty(binding.host_workspace_bytes(m, n, b), dtype=torch.uint8, device="cuda")
    binding.status(reset=True)

    # ---- device-resident throughput, then end to end (host buffers through mpdiv_batch_host: H2D + division +
    # D2H inside the timing); the clock sampler runs over both timed regions
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t0 = time.time()
    ms = time_steps(lambda: binding.mpdiv_batch(du, dv, q, r), args.steps, args.warmup, flush)
    barrier()
    ms_e = time_steps(lambda: binding.mpdiv_batch_host(hu, hv, hq, hr, ws), args.steps, args.warmup, flush)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    total_ms = shard.max_over_ranks(float(sum(ms)), device="cuda")
    ms_per_step = total_ms / args.steps
    value = shard.aggregate_rate(b, world, ms_per_step)
    e_total = shard.max_over_ranks(float(sum(ms_e)), device="cuda")
    e2e_value = shard.aggregate_rate(b, world, e_total / args.steps)
    io_bytes = b * 4 * (m + n)
    # the device-timed result and the host round trip must agree bit for bit (cheap self-consistency)
    same = bool((hq.cuda() == q).all().item() and (hr.cuda() == r).all().item())
    status = binding.status(reset=True)

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- roofline: what the timed step EXECUTED on each pipe, against peaks measured in this run -----------
    peaks = measure_imad_peak(binding)
    peaks["tensor_u8_mac"] = measure_tensor_peak(binding)
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    peaks["sm_count"] = sm_count
    peaks["sm_hz"] = (clocks.get("sm_mhz") or 1965.0) * 1e6
    kernel_ms = float(np.mean(ms))
    ex_imad, ex_tc, counters = executed_work(binding, du, dv, q, r)
    f_imad, f_tc, bound = pipe_fractions(ex_imad, ex_tc, kernel_ms, peaks)
    launches = binding.batch_launches(m, b)
    ncu = ncu_summary(cfg)
    if bound == "tensor":
        achieved, peak, unit = ex_tc / (kernel_ms * 1e-3) / 1e12, peaks["tensor_u8_mac"] / 1e12, "T u8-MAC/s"
    else:
        achieved, peak, unit = ex_imad / (kernel_ms * 1e-3) / 1e9, peaks["imad_wide_chain"] / 1e9, "G limb-products/s"
    roofline = {
        "bound": bound, "achieved": achieved, "peak": peak, "unit": unit, "frac": max(f_imad, f_tc),
        "definition": "frac = max over the two arithmetic pipes of (work the timed step EXECUTED on that pipe, counted "
                      "by the kernels) / (step time) / (that pipe's peak measured in this run); recompute it from the "
                      "executed_* and peak_* fields of this dict and ms_per_step",
        "frac_imad_pipe": f_imad, "frac_tensor_pipe": f_tc,
        "executed_limb_products_per_launch": ex_imad, "executed_tensor_macs_per_launch": ex_tc,
        "peak_imad_limb_products_per_s": peaks["imad_wide_chain"], "peak_tensor_u8_macs_per_s": peaks["tensor_u8_mac"],
        # how long the tensor unit is OCCUPIED (not how much arithmetic it does): the Toeplitz operand is read from
        # shared memory, so an instruction of N columns holds the unit max(32 + N/4, N/2) cycles (mpdiv_mma_probe form
        # 1), N/2 of them multiplying; counted per issued instruction by the engine, over all SMs at the clock seen
        "tensor_unit_occupancy": counters["mma_unit_cycles"] / (sm_count * kernel_ms * 1e-3 * peaks["sm_hz"]),
        "peak_source": "measured in this run: mpdiv_imad_probe kind 0 (carry-chained IMAD.WIDE.U32 tile, no memory; "
                       "nominal 32/clk/SM) and mpdiv_mma_probe (tcgen05.mma.kind::i8 M=128 N=128 K=32 from two warps, "
                       "events; nominal 8192 MAC/clk/SM)",
        "nominal_peaks": {"imad_limb_products_per_s": sm_count * 32 * 1965e6, "tensor_u8_macs_per_s": sm_count * 8192 * 1965e6,
                          "imad_lo32_per_s_measured": peaks["imad_lo32"]},
        "kernel": "mpdiv_kernel", "kernels_per_step": launches,
        "timed_region": "CUDA events around the whole step on the launch stream (shinv_head_kernel + mpdiv_kernel when "
                        "kernels_per_step = 2): achieved and frac charge the head kernel's time to the step",
        "traffic": (ncu or {}).get("dram_bytes_per_launch"), "ncu": ncu,
        "algorithmic_bytes_per_launch": b * 4 * (2 * m + 2 * n),
        "hbm_GBps_io": b * 4 * (2 * m + 2 * n) / (kernel_ms * 1e-3) / 1e9,
    }
    if cfg != 5:
        roofline["work_per_division_as_printed"] = W_LIMB_PRODUCTS[m]
        roofline["speedup_vs_printed_work"] = b * W_LIMB_PRODUCTS[m] / (kernel_ms * 1e-3) / peaks["imad_wide_chain"]
        roofline["speedup_vs_printed_work_note"] = (
            "divisions/s x W(M) / IMAD peak, W(M) = limb products of the method AS PRINTED (SURVEY 8(d)): how much "
            "faster than an IMAD-roofline implementation of the printed algorithm; NOT a utilisation (the default "
            "variant clips products, PAPER.md:507, :542, and runs the large ones on the tensor core)")
    if not args.brief:
        # one compact row per config INSIDE the roofline dict: div/s, both pipe fractions, the printed variant's
        # work-conserving fraction, R1 against both multiplication engines
        roofline["per_config"] = {"config%d" % c: config_row(binding, c, flush, peaks) for c in (1, 2, 3, 4, 5)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "batch_per_gpu": b, "u_limbs": m, "v_limbs": n,
                   "l2": "256 MiB buffer written between timed steps (L2 flush); inputs 14.5 MB",
                   "timing": "CUDA events per step on the launch stream, summed; max over ranks"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                "api": "mpdiv_batch_host (pinned host buffers)", "matches_device_run": same},
        "gpu_launches": args.steps * launches,
        "clocks": clocks,
        "roofline": roofline,
        "mpdiv_status": status,
        "step_ms_min_median_max": [float(np.min(ms)), float(np.median(ms)), float(np.max(ms))],
        "counters_one_step": {k: counters[k] for k in ("tiles", "mma_colsteps", "mma_products", "clipped_steps",
                                                       "chunks", "delta_pos", "delta_neg")},
        "version": binding.version(),
    }
    if not args.brief:
        out["paper_shape"] = paper_shape_table(binding, flush)
        # config 1 has 32 instances (latency bound on 148 SMs); the same shape with 32 x 148 instances gives the
        # THROUGHPUT point of the metric at 2^15 bits
        u15, v15 = inputs.uniform_operands(32 * 148, 1024, 512, config=11)
        d15u, d15v = to_dev(u15), to_dev(v15)
        q15, r15 = torch.empty_like(d15u), torch.empty_like(d15v)
        t15 = float(np.median(time_steps(lambda: binding.mpdiv_batch(d15u, d15v, q15, r15), 25, 3, flush)))
        e15, c15, _ = executed_work(binding, d15u, d15v, q15, r15)
        f15 = pipe_fractions(e15, c15, t15, peaks)
        out["throughput_2^15_bits"] = {"batch": 32 * 148, "u_limbs": 1024, "v_limbs": 512, "div_ms": t15,
                                       "div_per_s": 32 * 148 / (t15 * 1e-3), "frac_imad_pipe": f15[0],
                                       "frac_tensor_pipe": f15[1],
                                       "speedup_vs_printed_work": 32 * 148 / (t15 * 1e-3) * W_LIMB_PRODUCTS[1024] / peaks["imad_wide_chain"]}
        del d15u, d15v, q15, r15
        # 2^19-bit dividends (above the paper's shared-memory ceiling): the chunked form,
        # the dividend streamed from HBM window by window
        u19, v19 = inputs.uniform_operands(4 * 148, 16384, 8192, config=19)
        d19u, d19v = to_dev(u19), to_dev(v19)
        q19, r19 = torch.empty_like(d19u), torch.empty_like(d19v)
        t19 = float(np.median(time_steps(lambda: binding.mpdiv_batch(d19u, d19v, q19, r19), 10, 3, flush)))
        e19, c19, cnt19 = executed_work(binding, d19u, d19v, q19, r19)
        f19 = pipe_fractions(e19, c19, t19, peaks)
        out["range_extension_2^19_bits"] = {"batch": 4 * 148, "u_limbs": 16384, "v_limbs": 8192, "div_ms": t19,
                                            "div_per_s": 4 * 148 / (t19 * 1e-3), "frac_imad_pipe": f19[0],
                                            "frac_tensor_pipe": f19[1], "windows_per_division": cnt19["chunks"] / (4 * 148),
                                            "note": "dividend not resident: quotient in windows of 2048 limbs, one "
                                                    "shifted inverse of 2050 limbs for all windows (include/mpdiv.h)"}
        del d19u, d19v, q19, r19
        # small numbers in large batches -- one warp per division (32-thread blocks) against the
        # 128-thread block per division that larger numbers use (forced with MPDIV_FLAG_THREADS)
        small = {}
        for ms_, ns_, bs_ in ((32, 16, 64 * 148), (128, 64, 64 * 148), (256, 128, 64 * 148), (512, 256, 32 * 148)):
            us_, vs_ = inputs.uniform_operands(bs_, ms_, ns_, config=12)
            dsu, dsv = to_dev(us_), to_dev(vs_)
            qs, rs = torch.empty_like(dsu), torch.empty_like(dsv)
            t_def = float(np.median(time_steps(lambda: binding.mpdiv_batch(dsu, dsv, qs, rs), 10, 3, flush)))
            fl = binding.VARIANT_DEFAULT | binding.flag_threads(128)
            t_blk = float(np.median(time_steps(lambda: binding.mpdiv_batch(dsu, dsv, qs, rs, variant=fl), 10, 3, flush)))
            small["2^%d bits" % ((32 * ms_).bit_length() - 1)] = {
                "batch": bs_, "u_limbs": ms_, "v_limbs": ns_, "div_per_s": bs_ / (t_def * 1e-3),
                "div_per_s_128_thread_block_per_division": bs_ / (t_blk * 1e-3)}
            del dsu, dsv, qs, rs
        out["small_numbers_one_warp_per_division"] = small
        # the same shapes at 8 times the batch: more waves per SM, so the head kernel amortises and the resident blocks of
        # an SM drift out of lock step
        big = {}
        for cfg_, mult in ((2, 8), (3, 8), (4, 8)):
            bb, mm, nn_ = inputs.CONFIG_SHAPES[cfg_]
            ub, vb = inputs.uniform_operands(bb * mult, mm, nn_, config=30 + cfg_)
            dbu, dbv = to_dev(ub), to_dev(vb)
            qb, rb = torch.empty_like(dbu), torch.empty_like(dbv)
            tb = float(np.median(time_steps(lambda: binding.mpdiv_batch(dbu, dbv, qb, rb), 5, 3, flush)))
            big["config%d_shape_x%d" % (cfg_, mult)] = {"batch": bb * mult, "u_limbs": mm, "v_limbs": nn_, "div_ms": tb,
                                                      "div_per_s": bb * mult / (tb * 1e-3)}
            del dbu, dbv, qb, rb
        out["larger_batches"] = big
        out["tensor_issue_probe"] = measure_mma_issue(binding)
        out["cpu_baseline"] = cpu_baseline(cfg)
        out["paper_context"] = "A100, 64-bit digits (PAPER.md:481-484): div/mul 6.77x/6.66x/6.94x/9.73x at 2^18..2^15 bits; model 5-7"
    print(json.dumps(out))


# ----------------------------------------------------------------------------------------------
# reference arm: the CPU oracle (there is no reference implementation to install for this paper)
# ----------------------------------------------------------------------------------------------
def run_reference(args):
    """Times oracle/knuth_d.c, as it stands, on the host cores: each step is a bounded sample of the
    same workload.  Rank 0 only; other ranks exit 0 without work."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import oracle
    from paper_2606_06386_b200 import inputs

    cfg = args.config
    cores = max(1, os.cpu_count() or 1)
    b, m, n = inputs.CONFIG_SHAPES[cfg]
    u, v = inputs.config(cfg)
    # bound the whole run to about a minute: estimate the per-division cost on a few instances
    probe = min(b, 2 * cores)
    t0 = time.perf_counter()
    oracle.divmod_batch(u[:probe], v[:probe], threads=cores)
    per = (time.perf_counter() - t0) / probe
    budget = 60.0 / max(1, args.steps + args.warmup)
    count = int(max(cores, min(b, budget / max(per, 1e-9))))
    us, vs = u[:count], v[:count]
    for _ in range(args.warmup):
        oracle.divmod_batch(us, vs, threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.divmod_batch(us, vs, threads=cores)
    dt = time.perf_counter() - t0
    value = count * args.steps / dt
    sample = "first %d of %d instances of config %d per step, Knuth Algorithm D (oracle/knuth_d.c), %d host threads" % (
        count, b, cfg, cores)
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "batch_per_gpu": b, "u_limbs": m, "v_limbs": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as plain `python bench.py --gpus N`: launch the N ranks ourselves (one process per GPU, NCCL
        # used for the barrier and the max-over-ranks time only) and pass their exit code on
        from paper_2606_06386_b200 import shard

        raise SystemExit(subprocess.call(shard.torchrun_argv(args.gpus, os.path.abspath(__file__), sys.argv[1:])))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
