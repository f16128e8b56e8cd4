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

# DRAM bytes per launch of the division kernel from the committed ncu captures (profiles/r1_tensor_2p16.md)
NCU_DRAM_BYTES_PER_LAUNCH = {2: 24250368 + 7540480, 3: 39329536 + 24618240, 4: 38618880 + 23916800}
# share of the division kernel in a device-resident step (the rest is the head kernel), same captures
# (head kernel of configs 3 and 4 as captured in profiles/r1_final.md: it has not changed since)
NCU_DIV_KERNEL_SHARE = {2: 284.7 / (284.7 + 42.3), 3: 679.7 / (679.7 + 43.6), 4: 849.8 / (849.8 + 40.3)}
# pipe activity of the division kernel in the same captures, % of elapsed cycles:
# (sm__pipe_tensor_cycles_active, sm__pipe_fmaheavy_cycles_active, smsp__issue_active)
NCU_PIPES = {2: (13.75, 17.31, 44.75), 3: (18.91, 14.92, 37.62), 4: (25.86, 17.35, 34.65)}


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
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
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


def measure_mma_issue(binding):
    """Cycles per tcgen05.mma (M = 128, K = 32, u8) seen by one issuing warp and by two (mpdiv_mma_probe): the
    tensor core needs N / 2; the rest is the issue path."""
    out = {}
    for n in (16, 64, 128):
        one = binding.mma_probe(n, 1)
        two = binding.mma_probe(n, 2)
        out["N=%d" % n] = {"one_warp_cycles_per_mma": one[0], "two_warps_cycles_per_mma_together": max(two) / 2.0,
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
def per_config_table(binding, flush, peak_products: float):
    """divisions/s, shinv and multiplication times and the cost ratios of SURVEY.md G12 for configs 1-5
    (25 timed runs each, the paper's count; median)."""
    import torch

    from paper_2606_06386_b200 import inputs

    table = {}
    for cfg in (1, 2, 3, 4, 5):
        b, m, n = inputs.CONFIG_SHAPES[cfg]
        u, v = inputs.config(cfg)
        du, dv = to_dev(u), to_dev(v)
        q = torch.empty_like(du)
        r = torch.empty_like(dv)
        t_div = float(np.median(time_steps(lambda: binding.mpdiv_batch(du, dv, q, r), 25, 3, flush)))
        t_div_printed = float(np.median(time_steps(
            lambda: binding.mpdiv_batch(du, dv, q, r, variant=binding.VARIANT_PRINTED), 25, 3, flush)))
        executed = executed_products(binding, du, dv, q, r)
        # R1 unit: M x M -> low M limbs (the paper's "full multiplication", M^2/2 limb products)
        a1 = to_dev(inputs._uniform(inputs.rng_for(500 + cfg, 0), b, m))
        b1 = to_dev(inputs._uniform(inputs.rng_for(500 + cfg, 1), b, m))
        c1 = torch.empty((b, m), dtype=torch.int32, device="cuda")
        t_m1 = float(np.median(time_steps(lambda: binding.mpmul_batch(a1, b1, m, c1), 25, 3, flush)))
        # R2 unit: n x n -> 2n limbs, the full product of two divisor-sized numbers (M^2/4 limb products)
        nn = max(n if cfg != 5 else m // 2, 4)
        a2 = a1[:, :nn].contiguous()
        b2 = b1[:, :nn].contiguous()
        c2 = torch.empty((b, 2 * nn), dtype=torch.int32, device="cuda")
        t_m2 = float(np.median(time_steps(lambda: binding.mpmul_batch(a2, b2, 2 * nn, c2), 25, 3, flush)))
        # the same two products on the tensor-core engine (int8 tcgen05), where it fits
        t_m1_tc = t_m2_tc = None
        try:
            t_m1_tc = float(np.median(time_steps(
                lambda: binding.mpmul_batch(a1, b1, m, c1, engine=binding.ENGINE_TENSOR), 25, 3, flush)))
        except binding.MpdivError:
            pass
        try:
            t_m2_tc = float(np.median(time_steps(
                lambda: binding.mpmul_batch(a2, b2, 2 * nn, c2, engine=binding.ENGINE_TENSOR), 25, 3, flush)))
        except binding.MpdivError:
            pass
        wl = (m + 1 + 3) // 4 * 4
        w = torch.empty((b, wl), dtype=torch.int32, device="cuda")
        t_sh = float(np.median(time_steps(lambda: binding.shinv_batch(dv, m, wl, w), 25, 3, flush)))
        row = {
            "batch": b, "u_limbs": m, "v_limbs": n,
            "div_ms": t_div, "div_per_s": b / (t_div * 1e-3), "us_per_div_latency": t_div * 1e3 if cfg == 1 else None,
            "mul_MxM_lowM_ms": t_m1, "mul_nxn_full_ms": t_m2, "shinv_ms": t_sh,
            "R1_div_over_mul_MxM_lowM": t_div / t_m1, "R2_div_over_mul_nxn_full": t_div / t_m2,
            "shinv_over_mul_MxM_lowM": t_sh / t_m1,
            "mul_MxM_lowM_products_per_s": b * (m * (m + 1) / 2) / (t_m1 * 1e-3),
            "mul_nxn_full_products_per_s": b * nn * nn / (t_m2 * 1e-3),
            "hbm_GBps_div_io": b * 4 * (2 * m + 2 * n) / (t_div * 1e-3) / 1e9,
            "mul_MxM_lowM_tensor_ms": t_m1_tc, "mul_nxn_full_tensor_ms": t_m2_tc,
            "mul_nxn_full_tensor_products_per_s": (b * nn * nn / (t_m2_tc * 1e-3)) if t_m2_tc else None,
            "tensor_over_imad_speedup_nxn_full": (t_m2 / t_m2_tc) if t_m2_tc else None,
            "printed_variant_div_ms": t_div_printed, "printed_variant_div_per_s": b / (t_div_printed * 1e-3),
            "printed_variant_R1": t_div_printed / t_m1,
            "executed_limb_products_per_division": executed / b,
            "pipe_frac_executed": executed / (t_div * 1e-3) / peak_products,
        }
        if cfg != 5:
            row["W_limb_products"] = W_LIMB_PRODUCTS[m]
            row["roofline_frac"] = row["div_per_s"] * W_LIMB_PRODUCTS[m] / peak_products
            row["printed_variant_roofline_frac"] = row["printed_variant_div_per_s"] * W_LIMB_PRODUCTS[m] / peak_products
        table["config%d" % cfg] = row
        del du, dv, q, r, a1, b1, c1, a2, b2, c2, w
    return table


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


def executed_products(binding, du, dv, q, r, variant=None) -> int:
    """Limb products one launch really issues (8x8 tiles counted by the kernel x 64, tile padding included)."""
    import torch

    binding.debug_counters(reset=True)
    binding.mpdiv_batch(du, dv, q, r, variant=variant)
    torch.cuda.synchronize()
    return 64 * binding.debug_counters(reset=True)["tiles"]


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

    # ---- device-resident throughput ------------------------------------------------------------
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t0 = time.time()
    ms = time_steps(lambda: binding.mpdiv_batch(du, dv, q, r), args.steps, args.warmup, flush)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    total_ms = shard.max_over_ranks(float(sum(ms)), device="cuda")
    ms_per_step = total_ms / args.steps
    value = shard.aggregate_rate(b, world, ms_per_step)

    # ---- end to end: host buffers through mpdiv_batch_host (H2D + division + D2H inside the timing) ----
    hu = torch.from_numpy(u.view(np.int32)).pin_memory()
    hv = torch.from_numpy(v.view(np.int32)).pin_memory()
    hq = torch.empty_like(hu).pin_memory()
    hr = torch.empty_like(hv).pin_memory()
    ws = torch.empty(binding.host_workspace_bytes(m, n, b), dtype=torch.uint8, device="cuda")
    barrier()
    ms_e = time_steps(lambda: binding.mpdiv_batch_host(hu, hv, hq, hr, ws), args.steps, args.warmup, flush)
    barrier()
    e_total = shard.max_over_ranks(float(sum(ms_e)), device="cuda")
    e2e_value = shard.aggregate_rate(b, world, e_total / args.steps)
    io_bytes = b * 4 * (m + n)
    # the device-timed result and the host round trip must agree bit for bit (cheap self-consistency)
    same = bool((hq.cuda() == q).all().item() and (hr.cuda() == r).all().item())

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- roofline of the dominant kernel (a step = the head kernel + the division kernel, timed together) ---
    peaks = measure_imad_peak(binding)
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    nominal_peak = sm_count * IMAD_PER_CLK_PER_SM * 1965e6          # 32-bit IMAD/s at the max SM clock
    peak_products = peaks["imad_wide_chain"]
    kernel_ms = float(np.mean(ms))
    roofline = None
    if cfg != 5:
        achieved = b * W_LIMB_PRODUCTS[m] / (kernel_ms * 1e-3)
        executed = executed_products(binding, du, dv, q, r)
        ms_printed = float(np.mean(time_steps(
            lambda: binding.mpdiv_batch(du, dv, q, r, variant=binding.VARIANT_PRINTED), args.steps, args.warmup, flush)))
        roofline = {
            "note": "achieved = W(M) x batch / t with W(M) the limb products of the method AS PRINTED (SURVEY 8(d)); the "
                    "default (clipped) variant skips the low part of w*x and u*shinv, the low and high parts of v'w and the "
                    "high part of v*q (PAPER.md:507, :542), so frac may exceed 1; pipe_frac counts the limb products that "
                    "really ran on the IMAD pipe (the products that ran on the tensor cores are not in it)",
            "executed_limb_products_per_launch": executed,
            "pipe_frac": executed / (kernel_ms * 1e-3) / peak_products,
            "tensor_engine": "range products with enough work (u*shinv, v*q and the last Refine steps) run as int8 "
                             "tcgen05 GEMMs (csrc/mp_mma.cuh) in throughput batches from 2^16 bits up; per_config times "
                             "both engines on the same products",
            "printed_variant": {"ms": ms_printed, "divisions_per_s": b / (ms_printed * 1e-3),
                                "frac": b * W_LIMB_PRODUCTS[m] / (ms_printed * 1e-3) / peak_products},
            "ncu_pipes_pct": (dict(zip(("tensor", "fmaheavy", "issue_active"), NCU_PIPES[cfg]),
                                   source="profiles/r1_tensor_2p16.md: neither pipe is the limit, the kernel is bound by "
                                          "the latency of the phases inside a block") if cfg in NCU_PIPES else None),
            "bound": "alu", "kernel": "mpdiv_kernel",
            "kernels_per_step": binding.batch_launches(m, b),
            "kernel_share_of_step": NCU_DIV_KERNEL_SHARE.get(cfg) if binding.batch_launches(m, b) == 2 else 1.0,
            "timed_region": "CUDA events around the whole step (shinv_head_kernel + mpdiv_kernel on the launch stream): "
                            "achieved and frac are per step, i.e. they charge the head kernel's time to the division",
            "achieved": achieved / 1e9, "peak": peak_products / 1e9, "unit": "G limb-products/s",
            "frac": achieved / peak_products, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(cfg),
            "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture per launch "
                              "(profiles/r1_tensor_2p16.md); algorithmic bytes per launch = %d" % (b * 4 * (2 * m + 2 * n)),
            "peak_source": "measured in this run: mpdiv_imad_probe kind 0 (carry-chained IMAD.WIDE.U32 tile, no memory)",
            "nominal_imad32_peak": nominal_peak / 1e9,
            "measured_imad_lo32_peak": peaks["imad_lo32"] / 1e9,
            "frac_of_nominal_imad32": achieved / nominal_peak,
            "work_per_division": W_LIMB_PRODUCTS[m],
            "hbm_GBps_io": b * 4 * (2 * m + 2 * n) / (kernel_ms * 1e-3) / 1e9,
        }

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "batch_per_gpu": b, "u_limbs": m, "v_limbs": n,
                   "l2": "256 MiB buffer written between timed steps (L2 flush); inputs 14.5 MB",
                   "timing": "CUDA events per step on the launch stream, summed; max over ranks"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                "api": "mpdiv_batch_host (pinned host buffers)", "matches_device_run": same},
        "gpu_launches": args.steps * binding.batch_launches(m, b),
        "clocks": clocks,
        "roofline": roofline,
        "step_ms_min_median_max": [float(np.min(ms)), float(np.median(ms)), float(np.max(ms))],
        "version": binding.version(),
    }
    if not args.brief:
        out["per_config"] = per_config_table(binding, flush, peak_products)
        out["paper_shape"] = paper_shape_table(binding, flush)
        # config 1 has 32 instances (latency bound on 148 SMs); the same shape with 32 x 148 instances gives the
        # THROUGHPUT point of the metric at 2^15 bits
        u15, v15 = inputs.uniform_operands(32 * 148, 1024, 512, config=11)
        d15u, d15v = to_dev(u15), to_dev(v15)
        q15, r15 = torch.empty_like(d15u), torch.empty_like(d15v)
        t15 = float(np.median(time_steps(lambda: binding.mpdiv_batch(d15u, d15v, q15, r15), 25, 3, flush)))
        out["throughput_2^15_bits"] = {"batch": 32 * 148, "u_limbs": 1024, "v_limbs": 512, "div_ms": t15,
                                       "div_per_s": 32 * 148 / (t15 * 1e-3),
                                       "roofline_frac": 32 * 148 / (t15 * 1e-3) * W_LIMB_PRODUCTS[1024] / peak_products}
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
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
