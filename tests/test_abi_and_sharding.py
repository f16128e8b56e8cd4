"""CPU-side checks: the C-ABI library builds, loads and exports every symbol include/mpdiv.h declares
(no compute calls without a GPU); the batch-sharding host logic under a world_size-2 gloo group."""
import ctypes
import os
import re
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_06386_b200 import binding, build, shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    lib = ctypes.CDLL(path)
    header = open(os.path.join(ROOT, "include", "mpdiv.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b((?:mpdiv|mpmul|mplinop|shinv)_\w+)\s*\(", header))
    assert {"mpdiv_batch", "mpmul_batch", "shinv_batch"} <= declared
    for name in declared:
        assert hasattr(lib, name), "libmpdiv.so does not export %s" % name
    assert declared == set(binding.EXPORTS)
    # host-only entry points are callable without a GPU
    lib.mpdiv_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.mpdiv_version()
    lib.mpdiv_strerror.restype = ctypes.c_char_p
    lib.mpdiv_strerror.argtypes = [ctypes.c_int]
    assert lib.mpdiv_strerror(0) == b"ok"
    lib.mpdiv_host_workspace_bytes.restype = ctypes.c_size_t
    assert lib.mpdiv_host_workspace_bytes(2048, 1024, 1184) == 1184 * 2 * (2048 + 1024) * 4


def test_bad_arguments_rejected_before_any_cuda_call():
    lib = binding.lib()
    null = ctypes.c_void_p(0)
    buf = ctypes.create_string_buffer(64 * 4 + 16)
    p = (ctypes.addressof(buf) + 15) & ~15
    assert lib.mpdiv_batch(null, 8, p, 4, p, p, 1, null) == binding.ERR_BAD_ARG
    assert lib.mpdiv_batch(p, 6, p, 4, p, p, 1, null) == binding.ERR_BAD_ARG          # stride % 4
    assert lib.mpdiv_batch(p, 8, p, 4, p, p, 0, null) == binding.ERR_BAD_ARG          # empty batch
    assert lib.mpdiv_batch(p + 4, 8, p, 4, p, p, 1, null) == binding.ERR_BAD_ARG      # misaligned
    assert lib.mpdiv_batch_ex(p, 8, p, 4, p, p, 1, 7, null) == binding.ERR_BAD_ARG    # unknown variant
    assert lib.mpdiv_batch_ex(p, 8, p, 4, p, p, 1, 0x4000, null) == binding.ERR_BAD_ARG   # unknown flag bit
    assert lib.mpdiv_batch(p, 8, p, 8196, p, p, 1, null) == binding.ERR_UNSUPPORTED    # v stride above the maximum
    assert lib.mpdiv_batch(p, 16388, p, 4, p, p, 1, null) == binding.ERR_UNSUPPORTED   # u stride above the maximum
    assert lib.mpmul_batch(p, 8, p, 8, p, 20, 1, null) == binding.ERR_BAD_ARG         # c_limbs > a+b
    assert lib.shinv_batch(p, 8, 16, p, 16, 1, null) == binding.ERR_BAD_ARG           # w_limbs < h+1


def test_binding_refuses_cpu_tensors():
    t = torch.zeros((1, 8), dtype=torch.int32)
    with pytest.raises(ValueError):
        binding.mpdiv_batch(t, t)


def test_shard_bounds_tile_the_batch():
    for batch in (0, 1, 7, 592, 1184, 1185):
        for world in (1, 2, 3, 8):
            cuts = [shard.shard_bounds(batch, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == batch
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_bounds(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard.shard_bounds(1185, rank, world)
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi))
    ms = shard.max_over_ranks(10.0 + 5.0 * rank)
    dist.barrier()
    if rank == 0:
        out.put((gathered, ms, shard.aggregate_rate(1184, world, ms), shard.rank_seed(7, 1)))
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_max_time():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    gathered, ms, rate, seed = out.get()
    assert gathered == [(0, 593), (593, 1185)]
    assert ms == 15.0                       # the slower rank's time
    assert abs(rate - 2 * 1184 / 15e-3) < 1e-6
    assert seed == 8


def test_bench_spawns_its_own_ranks_with_torchrun():
    """`python bench.py --gpus N` without WORLD_SIZE re-executes itself under torchrun (shard.torchrun_argv); the
    same command line is run here on a CPU probe with the gloo backend and world size 2."""
    import json
    import subprocess
    import sys

    argv = shard.torchrun_argv(2, os.path.join(ROOT, "tests", "dist_probe.py"), ["--gpus", "2", "--steps", "3"])
    assert argv[:3] == [sys.executable, "-m", "torch.distributed.run"] and "127.0.0.1" in argv
    assert argv[argv.index("--nproc-per-node") + 1] == "2"
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    proc = subprocess.run(argv, capture_output=True, text=True, timeout=240, env=env)
    assert proc.returncode == 0, proc.stderr[-2000:]
    line = [ln for ln in proc.stdout.splitlines() if ln.startswith("{")][-1]
    out = json.loads(line)
    assert out["n_gpus"] == 2 and out["ms"] == 11.0 and out["first"] == [0, 592]
    assert out["args"] == ["--gpus", "2", "--steps", "3"] and out["master"] == "127.0.0.1"
    with pytest.raises(ValueError):
        shard.torchrun_argv(0, "x.py", [])


def test_bench_main_takes_the_spawn_path_only_without_world_size(monkeypatch):
    """bench.main() spawns ranks iff --gpus > 1 and it is not already a rank (WORLD_SIZE unset)."""
    import importlib
    import subprocess
    import sys

    sys.path.insert(0, ROOT)
    bench = importlib.import_module("bench")
    calls = []
    monkeypatch.setattr(subprocess, "call", lambda argv: calls.append(argv) or 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2", "--warmup", "1"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0 and len(calls) == 1
    assert calls[0][calls[0].index("--nproc-per-node") + 1] == "4" and calls[0][-6:] == ["--gpus", "4", "--steps", "2", "--warmup", "1"]
