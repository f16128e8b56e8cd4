"""Python binding of libmpdiv.so (include/mpdiv.h): argument marshalling only.

Every function takes torch CUDA tensors (dtype int32 or uint32, contiguous, batch x limbs,
little-endian limbs) that the CALLER allocates, passes their ``data_ptr()`` and the current
CUDA stream to the C ABI, and returns the output tensors.  No arithmetic happens here and
there is no CPU fallback: if the library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

_LIB = None
_VOIDP = ctypes.c_void_p

OK, ERR_BAD_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_TOO_LARGE = 0, 1, 2, 3, 4
NOALLOC_MAX_BATCH = 4096
VARIANT_PRINTED, VARIANT_CLIPPED = 0, 1
VARIANT_DEFAULT = VARIANT_CLIPPED
# tuning switches OR-ed into the `flags` of the *_ex calls (include/mpdiv.h)
FLAG_NO_SEED, FLAG_NO_HEAD, FLAG_NO_MMA, FLAG_NO_CLUSTER = 0x10, 0x20, 0x40, 0x80
STATUS_MMA_WAIT, STATUS_CORR_BOUND, STATUS_REM_RANGE, STATUS_V_ZERO, STATUS_IO_WAIT = 1, 2, 4, 8, 16
NUM_COUNTERS = 24


def flag_threads(n: int) -> int:
    """MPDIV_FLAG_THREADS(n): block size override."""
    return {32: 0x500, 64: 0x100, 128: 0x200, 256: 0x300, 512: 0x400}[int(n)]

def flag_cluster(n: int) -> int:
    """MPDIV_FLAG_CLUSTER(n): at most n CTAs per division in the cluster form."""
    return {2: 0x1000, 4: 0x2000, 8: 0x3000}[int(n)]


ENGINE_IMAD, ENGINE_TENSOR = 0, 1
LINOP_ADD, LINOP_SUB, LINOP_NEG, LINOP_SHIFT, LINOP_PREC, LINOP_ANY = range(6)
MAX_LIMBS = 16384          # u_limbs of mpdiv_batch (default variant)
MAX_OPERAND_LIMBS = 8192   # every other stride


class MpdivError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__("%s: status %d (%s)" % (what, code, strerror(code)))
        self.code = code


def lib() -> ctypes.CDLL:
    """Load libmpdiv.so (must have been built: ``python -m paper_2606_06386_b200.build``)."""
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(
                "libmpdiv.so is not built (%s); run __graft_entry__.build() -- there is no CPU fallback" % path)
        L = ctypes.CDLL(path)
        i, sz = ctypes.c_int, ctypes.c_size_t
        L.mpdiv_batch.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, _VOIDP, i, _VOIDP]
        L.mpdiv_batch_ex.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, _VOIDP, i, i, _VOIDP]
        L.mpdiv_batch_noalloc.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, _VOIDP, i, _VOIDP]
        L.mpdiv_batch_noalloc.restype = i
        L.shinv_batch_ex.argtypes = [_VOIDP, i, i, _VOIDP, i, i, i, _VOIDP]
        L.mplinop_batch.argtypes = [i, _VOIDP, i, _VOIDP, i, i, _VOIDP, i, _VOIDP, i, _VOIDP]
        L.mpmul_batch_ex.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, i, i, i, _VOIDP]
        L.mpmul_batch.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, i, i, _VOIDP]
        L.shinv_batch.argtypes = [_VOIDP, i, i, _VOIDP, i, i, _VOIDP]
        L.mpdiv_host_workspace_bytes.argtypes = [i, i, i]
        L.mpdiv_host_workspace_bytes.restype = sz
        L.mpdiv_batch_host.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP, _VOIDP, i, _VOIDP, sz, _VOIDP]
        L.mpdiv_imad_probe_threads.argtypes = []
        L.mpdiv_imad_probe.argtypes = [_VOIDP, i, i, ctypes.POINTER(ctypes.c_ulonglong), _VOIDP]
        L.mpdiv_mma_probe.argtypes = [i, i, i, i, _VOIDP, _VOIDP]
        L.mpdiv_mma_probe.restype = i
        L.mpdiv_mma_probe_macs.argtypes = [i, i, i]
        L.mpdiv_mma_probe_macs.restype = ctypes.c_ulonglong
        L.mpdiv_status.argtypes = [_VOIDP, ctypes.POINTER(ctypes.c_uint), i]
        L.mpdiv_status.restype = i
        L.mpdiv_debug_counters.argtypes = [ctypes.POINTER(ctypes.c_ulonglong), i, _VOIDP]
        L.mpdiv_seed_batch.argtypes = [_VOIDP, i, _VOIDP, i, _VOIDP]
        L.mpdiv_batch_launches.argtypes = [i, i, i]
        L.mpdiv_version.restype = ctypes.c_char_p
        L.mpdiv_strerror.argtypes = [i]
        L.mpdiv_strerror.restype = ctypes.c_char_p
        for name in ("mplinop_batch", "mpdiv_batch", "mpdiv_batch_ex", "shinv_batch_ex", "mpmul_batch", "mpmul_batch_ex", "shinv_batch", "mpdiv_batch_host",
                     "mpdiv_imad_probe_threads", "mpdiv_imad_probe", "mpdiv_debug_counters"):
            getattr(L, name).restype = i
        _LIB = L
    return _LIB


EXPORTS = ("mplinop_batch", "mpdiv_batch", "mpdiv_batch_ex", "mpdiv_batch_noalloc", "mpmul_batch", "mpmul_batch_ex", "shinv_batch", "shinv_batch_ex", "mpdiv_host_workspace_bytes",
           "mpdiv_batch_host", "mpdiv_imad_probe_threads", "mpdiv_imad_probe", "mpdiv_mma_probe", "mpdiv_mma_probe_macs",
           "mpdiv_debug_counters", "mpdiv_status", "mpdiv_seed_batch", "mpdiv_batch_launches", "mpdiv_version", "mpdiv_strerror")


def version() -> str:
    return lib().mpdiv_version().decode()


def strerror(code: int) -> str:
    return lib().mpdiv_strerror(int(code)).decode()


def _stream_ptr(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _check_dev(t: torch.Tensor, name: str):
    if not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor" % name)
    if t.dtype not in (torch.int32, torch.uint32):
        raise ValueError("%s must be int32/uint32" % name)
    if t.dim() != 2 or not t.is_contiguous():
        raise ValueError("%s must be a contiguous (batch, limbs) tensor" % name)


def _raise(code: int, what: str):
    if code != OK:
        raise MpdivError(code, what)


def mpdiv_batch(u: torch.Tensor, v: torch.Tensor, q: torch.Tensor | None = None,
                r: torch.Tensor | None = None, stream=None, variant: int | None = None):
    """q = floor(u / v), r = u - q*v per row.  q has u's shape, r has v's shape.
    variant: None -> mpdiv_batch (the library default), else mpdiv_batch_ex with these flags
    (a VARIANT_* value, optionally OR-ed with FLAG_* tuning switches)."""
    _check_dev(u, "u")
    _check_dev(v, "v")
    batch, ul = u.shape
    vl = v.shape[1]
    if v.shape[0] != batch:
        raise ValueError("batch mismatch")
    if q is None:
        q = torch.empty_like(u)
    if r is None:
        r = torch.empty_like(v)
    _check_dev(q, "q")
    _check_dev(r, "r")
    if tuple(q.shape) != (batch, ul) or tuple(r.shape) != (batch, vl):
        raise ValueError("q must be (batch, u_limbs) and r (batch, v_limbs)")
    if variant is None:
        _raise(lib().mpdiv_batch(u.data_ptr(), ul, v.data_ptr(), vl, q.data_ptr(), r.data_ptr(), batch,
                                 _stream_ptr(stream)), "mpdiv_batch")
    else:
        _raise(lib().mpdiv_batch_ex(u.data_ptr(), ul, v.data_ptr(), vl, q.data_ptr(), r.data_ptr(), batch,
                                    int(variant), _stream_ptr(stream)), "mpdiv_batch_ex")
    return q, r


def mpdiv_batch_noalloc(u: torch.Tensor, v: torch.Tensor, q: torch.Tensor, r: torch.Tensor, stream=None):
    """mpdiv_batch through the entry point that allocates nothing (static scratch inside the library, batch <=
    NOALLOC_MAX_BATCH); the caller passes every buffer.  Calls that overlap on the GPU race on the scratch."""
    for t, name in ((u, "u"), (v, "v"), (q, "q"), (r, "r")):
        _check_dev(t, name)
    batch, ul = u.shape
    vl = v.shape[1]
    if v.shape[0] != batch or tuple(q.shape) != (batch, ul) or tuple(r.shape) != (batch, vl):
        raise ValueError("v, q, r must be (batch, v_limbs), (batch, u_limbs), (batch, v_limbs)")
    _raise(lib().mpdiv_batch_noalloc(u.data_ptr(), ul, v.data_ptr(), vl, q.data_ptr(), r.data_ptr(), batch,
                                     _stream_ptr(stream)), "mpdiv_batch_noalloc")
    return q, r


def mpmul_batch(a: torch.Tensor, b: torch.Tensor, c_limbs: int, c: torch.Tensor | None = None, stream=None,
                engine: int | None = None):
    """c = (a * b) mod B^c_limbs per row.  engine: None -> mpmul_batch (IMAD), else mpmul_batch_ex."""
    _check_dev(a, "a")
    _check_dev(b, "b")
    batch = a.shape[0]
    if b.shape[0] != batch:
        raise ValueError("batch mismatch")
    if c is None:
        c = torch.empty((batch, c_limbs), dtype=a.dtype, device=a.device)
    _check_dev(c, "c")
    if engine is None:
        _raise(lib().mpmul_batch(a.data_ptr(), a.shape[1], b.data_ptr(), b.shape[1], c.data_ptr(), c_limbs, batch,
                                 _stream_ptr(stream)), "mpmul_batch")
    else:
        _raise(lib().mpmul_batch_ex(a.data_ptr(), a.shape[1], b.data_ptr(), b.shape[1], c.data_ptr(), c_limbs, batch,
                                    int(engine), _stream_ptr(stream)), "mpmul_batch_ex")
    return c


def mplinop_batch(op: int, a: torch.Tensor, b: torch.Tensor, shift: int, out_limbs: int, stream=None):
    """One linear building block per row (include/mpdiv.h); returns (out, flag)."""
    _check_dev(a, "a")
    _check_dev(b, "b")
    batch = a.shape[0]
    out = torch.empty((batch, out_limbs), dtype=a.dtype, device=a.device)
    flag = torch.empty((batch,), dtype=torch.int32, device=a.device)
    _raise(lib().mplinop_batch(int(op), a.data_ptr(), a.shape[1], b.data_ptr(), b.shape[1], int(shift), out.data_ptr(),
                               out_limbs, flag.data_ptr(), batch, _stream_ptr(stream)), "mplinop_batch")
    return out, flag


def shinv_batch(v: torch.Tensor, h: int, w_limbs: int, w: torch.Tensor | None = None, stream=None,
                variant: int | None = None):
    """w = floor(B^h / v) + lambda per row (the uncorrected Newton result).  variant None -> shinv_batch: the
    algorithm as printed, lambda in {0, 1} (Theorem 2); else shinv_batch_ex with these flags (VARIANT_CLIPPED:
    lambda in {-1, 0, 1})."""
    _check_dev(v, "v")
    batch = v.shape[0]
    if w is None:
        w = torch.empty((batch, w_limbs), dtype=v.dtype, device=v.device)
    _check_dev(w, "w")
    if variant is None:
        _raise(lib().shinv_batch(v.data_ptr(), v.shape[1], int(h), w.data_ptr(), w_limbs, batch,
                                 _stream_ptr(stream)), "shinv_batch")
    else:
        _raise(lib().shinv_batch_ex(v.data_ptr(), v.shape[1], int(h), w.data_ptr(), w_limbs, batch, int(variant),
                                    _stream_ptr(stream)), "shinv_batch_ex")
    return w


def batch_launches(u_limbs: int, batch: int, variant: int = VARIANT_DEFAULT) -> int:
    """Kernels one mpdiv_batch call of this shape launches (2 when the head of Refine runs in its own kernel)."""
    return int(lib().mpdiv_batch_launches(int(u_limbs), int(batch), int(variant)))


SEED_LIMBS = 24     # limbs per row of mpdiv_seed_batch (20 significant)


def seed_batch(v: torch.Tensor, w: torch.Tensor | None = None, stream=None):
    """w = floor(B^38 / (top 20 limbs of v)) per row: the 17-digit seed of Refine (include/mpdiv.h)."""
    _check_dev(v, "v")
    if w is None:
        w = torch.empty((v.shape[0], SEED_LIMBS), dtype=v.dtype, device=v.device)
    _check_dev(w, "w")
    if w.shape != (v.shape[0], SEED_LIMBS):
        raise ValueError("w must be batch x %d" % SEED_LIMBS)
    _raise(lib().mpdiv_seed_batch(v.data_ptr(), v.shape[1], w.data_ptr(), v.shape[0], _stream_ptr(stream)),
           "mpdiv_seed_batch")
    return w


def host_workspace_bytes(u_limbs: int, v_limbs: int, batch: int) -> int:
    return int(lib().mpdiv_host_workspace_bytes(u_limbs, v_limbs, batch))


def mpdiv_batch_host(u: torch.Tensor, v: torch.Tensor, q: torch.Tensor, r: torch.Tensor,
                     workspace: torch.Tensor, stream=None):
    """Host-buffer form: u, v, q, r are (pinned) CPU tensors, workspace a CUDA byte tensor.
    Enqueues H2D + division + D2H on the stream; the caller synchronises."""
    for t, name in ((u, "u"), (v, "v"), (q, "q"), (r, "r")):
        if t.is_cuda or not t.is_contiguous() or t.dtype not in (torch.int32, torch.uint32):
            raise ValueError("%s must be a contiguous int32/uint32 CPU tensor" % name)
    if not workspace.is_cuda:
        raise ValueError("workspace must be a CUDA tensor")
    batch, ul = u.shape
    vl = v.shape[1]
    _raise(lib().mpdiv_batch_host(u.data_ptr(), ul, v.data_ptr(), vl, q.data_ptr(), r.data_ptr(), batch,
                                  workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                  _stream_ptr(stream)), "mpdiv_batch_host")
    return q, r


def imad_probe(kind: int, iters: int, sink: torch.Tensor | None = None, stream=None):
    """Launch the integer-multiply probe; returns (limb products issued, sink tensor)."""
    n = lib().mpdiv_imad_probe_threads()
    if n <= 0:
        raise MpdivError(ERR_CUDA, "mpdiv_imad_probe_threads")
    if sink is None:
        sink = torch.empty(n, dtype=torch.int32, device="cuda")
    prod = ctypes.c_ulonglong(0)
    _raise(lib().mpdiv_imad_probe(sink.data_ptr(), int(kind), int(iters), ctypes.byref(prod),
                                  _stream_ptr(stream)), "mpdiv_imad_probe")
    return int(prod.value), sink


def mma_probe_launch(n_cols: int, issuers: int, iters: int, out: torch.Tensor, form: int = 0, stream=None):
    """Enqueue one probe launch (no synchronisation): for timing with events."""
    _raise(lib().mpdiv_mma_probe(int(n_cols), int(issuers), int(iters), int(form), out.data_ptr(), _stream_ptr(stream)),
           "mpdiv_mma_probe")


def mma_probe(n_cols: int, issuers: int = 1, iters: int = 2000, form: int = 0, stream=None):
    """Cycles per tcgen05.mma (M = 128, K = 32, u8, N = n_cols) of each issuing warp of block 0; synchronises.
    form 0: A in tensor memory; form 1: A from shared memory through the Toeplitz descriptor."""
    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    _raise(lib().mpdiv_mma_probe(int(n_cols), int(issuers), int(iters), int(form), out.data_ptr(), _stream_ptr(stream)),
           "mpdiv_mma_probe")
    torch.cuda.synchronize()
    return [c / (4.0 * iters) for c in out.tolist()[:issuers]]


COUNTER_NAMES = ("delta_neg", "delta_pos", "delta_multi", "one_limb", "u_lt_v", "v_zero", "sign_neg", "pow_b",
                 "tiles", "delta_neg_multi", "delta_out_of_range", "clipped_steps", "mma_products", "mma_wait_failures",
                 "seed_addbacks", "seeds", "mma_colsteps", "cluster_divs", "chunks", "mma_unit_cycles")


def debug_counters(reset: bool = False, stream=None) -> dict:
    out = (ctypes.c_ulonglong * NUM_COUNTERS)()
    _raise(lib().mpdiv_debug_counters(out, 1 if reset else 0, _stream_ptr(stream)), "mpdiv_debug_counters")
    return {k: int(out[i]) for i, k in enumerate(COUNTER_NAMES)}


def status(reset: bool = False, stream=None) -> int:
    """Sticky status bits of the current device (STATUS_*); synchronises the stream.  0 = all results exact."""
    flags = ctypes.c_uint(0)
    _raise(lib().mpdiv_status(_stream_ptr(stream), ctypes.byref(flags), 1 if reset else 0), "mpdiv_status")
    return int(flags.value)


def mma_probe_macs(n_cols: int, issuers: int, iters: int) -> int:
    """u8 x u8 multiply-accumulates one mpdiv_mma_probe launch executes."""
    return int(lib().mpdiv_mma_probe_macs(int(n_cols), int(issuers), int(iters)))
