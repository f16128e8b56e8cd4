"""ORACLE -- TEST INFRASTRUCTURE ONLY (not the product path).

Thin numpy/ctypes front end of ``oracle/knuth_d.c``: the plain CPU definition of what the
hot path of arxiv/paper_2606_06386 computes (Euclidean quotient and remainder,
PAPER.md:131-133; whole shifted inverse floor(B^h / v); product mod B^d,
PAPER.md:105-106), on little-endian uint32 limbs.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_2606_06386_b200`` and shares no code with the CUDA library.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "knuth_d.c")
_HDR = os.path.join(_HERE, "knuth_d_impl.h")
_LIB = os.path.join(_HERE, "libknuthd.so")

_lib = None
_U32P = ctypes.POINTER(ctypes.c_uint32)


def build(force: bool = False) -> str:
    """Compile knuth_d.c with gcc into oracle/libknuthd.so (rebuilt when a source is newer)."""
    stale = (
        force
        or not os.path.exists(_LIB)
        or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    )
    if stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i = ctypes.c_int
        lib.orc_divmod.argtypes = [_U32P, i, _U32P, i, _U32P, i, _U32P, i]
        lib.orc_divmod_base16.argtypes = [_U32P, i, _U32P, i, _U32P, i, _U32P, i]
        lib.orc_divmod_batch.argtypes = [_U32P, i, _U32P, i, _U32P, i, _U32P, i, i]
        lib.orc_mul.argtypes = [_U32P, i, _U32P, i, _U32P, i]
        lib.orc_mul_batch.argtypes = [_U32P, i, _U32P, i, _U32P, i, i]
        lib.orc_shinv.argtypes = [_U32P, i, i, _U32P, i]
        lib.orc_shinv_batch.argtypes = [_U32P, i, i, _U32P, i, i]
        for name in ("orc_divmod", "orc_divmod_base16", "orc_divmod_batch", "orc_mul",
                     "orc_mul_batch", "orc_shinv", "orc_shinv_batch"):
            getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(_U32P)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.uint32)


class OracleError(RuntimeError):
    pass


_STATUS = {1: "divisor is zero", 2: "quotient or remainder does not fit", 3: "out of memory"}


def _check(st: int):
    if st != 0:
        raise OracleError(_STATUS.get(st, "status %d" % st))


def divmod_limbs(u, v, q_limbs: int, r_limbs: int, base16: bool = False):
    """(q, r) of one instance; u, v are 1-D limb arrays (little endian)."""
    lib = _load()
    u = _c(u)
    v = _c(v)
    q = np.zeros(q_limbs, dtype=np.uint32)
    r = np.zeros(r_limbs, dtype=np.uint32)
    fn = lib.orc_divmod_base16 if base16 else lib.orc_divmod
    _check(fn(_p(u), u.size, _p(v), v.size, _p(q), q_limbs, _p(r), r_limbs))
    return q, r


def divmod_batch(u, v, q_limbs: int | None = None, r_limbs: int | None = None, threads: int = 1):
    """Batched (q, r): u is (batch, u_limbs), v is (batch, v_limbs).

    q stride defaults to u_limbs and r stride to v_limbs (the layout of include/mpdiv.h).
    ``threads`` > 1 splits the batch over host threads (ctypes releases the GIL); the C
    routine itself is the same single-threaded loop.
    """
    lib = _load()
    u = _c(u)
    v = _c(v)
    batch, un = u.shape
    vn = v.shape[1]
    assert v.shape[0] == batch
    qn = un if q_limbs is None else q_limbs
    rn = vn if r_limbs is None else r_limbs
    q = np.zeros((batch, qn), dtype=np.uint32)
    r = np.zeros((batch, rn), dtype=np.uint32)

    def run(lo, hi):
        if hi <= lo:
            return 0
        return lib.orc_divmod_batch(_p(u[lo:hi]), un, _p(v[lo:hi]), vn,
                                    _p(q[lo:hi]), qn, _p(r[lo:hi]), rn, hi - lo)

    threads = max(1, min(threads, batch))
    if threads == 1:
        _check(run(0, batch))
    else:
        cuts = [batch * t // threads for t in range(threads + 1)]
        with ThreadPoolExecutor(max_workers=threads) as ex:
            for st in ex.map(lambda ab: run(*ab), zip(cuts[:-1], cuts[1:])):
                _check(st)
    return q, r


def mul_batch(a, b, c_limbs: int):
    """c = (a*b) mod B^c_limbs per instance; a is (batch, a_limbs), b is (batch, b_limbs)."""
    lib = _load()
    a = _c(a)
    b = _c(b)
    batch = a.shape[0]
    c = np.zeros((batch, c_limbs), dtype=np.uint32)
    _check(lib.orc_mul_batch(_p(a), a.shape[1], _p(b), b.shape[1], _p(c), c_limbs, batch))
    return c


def shinv_batch(v, h: int, w_limbs: int):
    """w = floor(B^h / v) per instance (Definition 1); v is (batch, v_limbs)."""
    lib = _load()
    v = _c(v)
    batch = v.shape[0]
    w = np.zeros((batch, w_limbs), dtype=np.uint32)
    _check(lib.orc_shinv_batch(_p(v), v.shape[1], h, _p(w), w_limbs, batch))
    return w
