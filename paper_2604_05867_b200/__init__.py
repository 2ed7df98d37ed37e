"""paper_2604_05867_b200 -- thin Python binding of libba (include/ba.h).

Argument marshalling only: every step of the BA hot path (output sweep, input sweep, reductions,
update) runs in the hand-written CUDA kernels of csrc/.  PyTorch provides device memory and the
CUDA stream (ba_create_ext); nothing here computes.  There is no CPU fallback: importing the
binding on a box without the built library, or creating a context without a CUDA device, raises.

The module-level functions carry the names of the C entry points (ba_create, ba_iterate,
ba_bounds, ba_get_p, ...); `BA` is a small convenience wrapper around a context.
"""
import ctypes
import os

import numpy as np

from . import build as _build

BA_OK, BA_EINVAL, BA_ENOMEM, BA_ECUDA, BA_ESTATE, BA_ENUMERIC = 0, -1, -2, -3, -4, -5
BA_MODE_ENUM, BA_MODE_FAST = 0, 1
BA_NMAX = 30
BA_NOALLOC_NMAX, BA_NOALLOC_MAXBLK = 26, 2048
_CODE_NAMES = {0: "BA_OK", -1: "BA_EINVAL", -2: "BA_ENOMEM", -3: "BA_ECUDA", -4: "BA_ESTATE", -5: "BA_ENUMERIC"}

EXPORTS = ["ba_create", "ba_iterate", "ba_bounds", "ba_get_p", "ba_scratch_bytes", "ba_create_ext",
           "ba_set_mode", "ba_set_exact", "ba_set_symmetry", "ba_set_p", "ba_get_q", "ba_get_D", "ba_stats", "ba_get_history",
           "ba_last_timing", "ba_setup_ms", "ba_measure_peaks", "ba_debug_emb_row", "ba_debug_emb_col", "ba_terms_per_sweep",
           "ba_debug_count_terms", "ba_debug_check_tables", "ba_destroy", "ba_last_error", "ba_in_final_noalloc",
           "ba_noalloc_last_error"]


class BAError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_CODE_NAMES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib_path():
    return _build.LIB


def load():
    """Load libba.so (building it with nvcc first if the source is newer). Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = ctypes.CDLL(path)
    vp, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)
    up = ctypes.POINTER(ctypes.c_uint)
    ullp = ctypes.POINTER(ctypes.c_ulonglong)
    L.ba_create.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.POINTER(vp)]
    L.ba_create_ext.argtypes = [ctypes.c_int, ctypes.c_double, vp, vp, vp, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    L.ba_scratch_bytes.argtypes = [ctypes.c_int]
    L.ba_scratch_bytes.restype = ctypes.c_size_t
    L.ba_iterate.argtypes = [vp, ctypes.c_int]
    L.ba_bounds.argtypes = [vp, dp, dp]
    L.ba_get_p.argtypes = [vp, dp]
    L.ba_get_q.argtypes = [vp, dp]
    L.ba_get_D.argtypes = [vp, dp]
    L.ba_set_p.argtypes = [vp, dp]
    L.ba_set_mode.argtypes = [vp, ctypes.c_int]
    L.ba_set_exact.argtypes = [vp, ctypes.c_int]
    L.ba_set_symmetry.argtypes = [vp, ctypes.c_int]
    L.ba_stats.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_longlong)]
    L.ba_get_history.argtypes = [vp, ctypes.c_int, dp]
    L.ba_last_timing.argtypes = [vp, dp]
    L.ba_setup_ms.argtypes = [vp, dp]
    L.ba_measure_peaks.argtypes = [dp]
    L.ba_debug_emb_row.argtypes = [vp, ctypes.c_uint, up]
    L.ba_debug_emb_col.argtypes = [vp, ctypes.c_uint, up]
    L.ba_terms_per_sweep.argtypes = [ctypes.c_int, ullp]
    L.ba_debug_count_terms.argtypes = [vp, ullp, ullp, ullp, ullp]
    L.ba_debug_check_tables.argtypes = [ctypes.c_int, ullp]
    L.ba_destroy.argtypes = [vp]
    L.ba_destroy.restype = None
    L.ba_last_error.argtypes = [vp]
    L.ba_last_error.restype = ctypes.c_char_p
    L.ba_in_final_noalloc.argtypes = [ctypes.c_int, vp, vp, vp, vp, vp, vp, vp]
    L.ba_noalloc_last_error.argtypes = []
    L.ba_noalloc_last_error.restype = ctypes.c_char_p
    for name in EXPORTS:
        getattr(L, name)
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class _Ctx:
    """Opaque handle + the torch tensors that back a ba_create_ext context."""

    def __init__(self, handle, n, tensors=None):
        self.handle = handle
        self.n = n
        self.tensors = tensors


def _check(ctx, rc):
    if rc != BA_OK:
        msg = load().ba_last_error(ctx.handle if ctx else None)
        raise BAError(rc, msg.decode() if msg else "")


def ba_scratch_bytes(n):
    return int(load().ba_scratch_bytes(int(n)))


def ba_create(n, d, device="cuda:0", use_torch_memory=True):
    """ba_create / ba_create_ext.  With use_torch_memory (default) p, q, D and the scratch are torch
    CUDA tensors and the kernels run on torch's current stream."""
    L = load()
    h = ctypes.c_void_p()
    if not use_torch_memory:
        rc = L.ba_create(int(n), float(d), ctypes.byref(h))
        if rc != BA_OK:
            raise BAError(rc, "ba_create failed")
        return _Ctx(h, n)
    import torch
    if not torch.cuda.is_available():
        raise BAError(BA_ECUDA, "no CUDA device: libba has no CPU fallback")
    if not (isinstance(n, int) and 1 <= n <= BA_NMAX):
        raise BAError(BA_EINVAL, "n out of range")
    dev = torch.device(device)
    torch.cuda.set_device(dev)
    NX, NY = 1 << n, (2 << n) - 1
    p = torch.empty(NX, dtype=torch.float64, device=dev)
    q = torch.empty(NY, dtype=torch.float64, device=dev)
    D = torch.empty(NX, dtype=torch.float64, device=dev)
    sb = ba_scratch_bytes(n)
    scratch = torch.empty(sb + 256, dtype=torch.uint8, device=dev)
    sptr = (scratch.data_ptr() + 255) & ~255
    stream = torch.cuda.current_stream(dev).cuda_stream
    rc = L.ba_create_ext(int(n), float(d), p.data_ptr(), q.data_ptr(), D.data_ptr(), sptr, sb,
                         ctypes.c_void_p(stream), ctypes.byref(h))
    if rc != BA_OK:
        raise BAError(rc, "ba_create_ext failed")
    return _Ctx(h, n, dict(p=p, q=q, D=D, scratch=scratch))


def ba_destroy(ctx):
    if ctx.handle:
        load().ba_destroy(ctx.handle)
        ctx.handle = None
        ctx.tensors = None


def ba_set_mode(ctx, mode):
    _check(ctx, load().ba_set_mode(ctx.handle, int(mode)))


def ba_set_exact(ctx, k):
    """Switch to the paper's exact channel BDC_{n,k} (before the first iteration)."""
    _check(ctx, load().ba_set_exact(ctx.handle, int(k)))


def ba_set_symmetry(ctx, on):
    """Complement symmetry p(x) = p(~x): the ENUM sweeps enumerate half the inputs / output prefixes."""
    _check(ctx, load().ba_set_symmetry(ctx.handle, int(on)))


def ba_iterate(ctx, k):
    _check(ctx, load().ba_iterate(ctx.handle, int(k)))


def ba_bounds(ctx):
    lo, up = ctypes.c_double(), ctypes.c_double()
    _check(ctx, load().ba_bounds(ctx.handle, ctypes.byref(lo), ctypes.byref(up)))
    return lo.value, up.value


def ba_stats(ctx):
    lz, it = ctypes.c_double(), ctypes.c_longlong()
    _check(ctx, load().ba_stats(ctx.handle, ctypes.byref(lz), ctypes.byref(it)))
    return lz.value, it.value


def ba_iters_done(ctx):
    it = ctypes.c_longlong()
    _check(ctx, load().ba_stats(ctx.handle, None, ctypes.byref(it)))
    return it.value


def ba_get_history(ctx, count):
    out = np.empty((count, 3), dtype=np.float64)
    _check(ctx, load().ba_get_history(ctx.handle, int(count), _dp(out)))
    return out


def ba_last_timing(ctx):
    ms = np.empty(4, dtype=np.float64)
    _check(ctx, load().ba_last_timing(ctx.handle, _dp(ms)))
    return dict(out_ms=ms[0], in_ms=ms[1], update_ms=ms[2], iter_ms=ms[3])


def ba_setup_ms(ctx):
    """Milliseconds of the one-off Hc pass the first ba_iterate ran."""
    v = ctypes.c_double()
    _check(ctx, load().ba_setup_ms(ctx.handle, ctypes.byref(v)))
    return float(v.value)


def ba_measure_peaks():
    """Pipe microbenchmarks on the current device: warp-instructions per clock per SM, SM MHz, SM count."""
    out = np.empty(6, dtype=np.float64)
    rc = load().ba_measure_peaks(_dp(out))
    if rc:
        raise BAError(rc, "ba_measure_peaks failed")
    return dict(dfma=out[0], idp2a=out[1], lds64=out[2], ffma=out[3], sm_mhz=out[4], sms=int(out[5]))


def ba_in_final_noalloc(n, Hc, S0, S1, p, D, out3, stream=None):
    """D = Hc - (S0 + S1) and out3 = {sum p D, max D, sum p 2^D} without any device allocation (ba.h): the first-stage
    partials sit in a static device array of libba.  Hc, S0, S1 (or None), p, D: float64 CUDA tensors of 2^n entries;
    out3: 3 entries; all on the current device.  Queued on `stream` (a torch.cuda.Stream; default: torch's current
    stream); does not synchronise."""
    import torch
    sized = 1 <= n <= BA_NOALLOC_NMAX                      # otherwise the library rejects the call before touching memory
    NX = 1 << n if sized else 0
    for name, t, need in (("Hc", Hc, NX), ("S0", S0, NX), ("S1", S1, NX), ("p", p, NX), ("D", D, NX), ("out3", out3, 3)):
        if t is None and name == "S1":
            continue
        if (t is None or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous()
                or (sized and t.numel() != need)):
            raise BAError(BA_EINVAL, f"ba_in_final_noalloc: {name} must be a contiguous float64 CUDA tensor of {need} entries")
    st = stream if stream is not None else torch.cuda.current_stream()
    L = load()
    rc = L.ba_in_final_noalloc(n, Hc.data_ptr(), S0.data_ptr(), S1.data_ptr() if S1 is not None else None, p.data_ptr(),
                               D.data_ptr(), out3.data_ptr(), st.cuda_stream)
    if rc:
        raise BAError(rc, L.ba_noalloc_last_error().decode())


def ba_get_p(ctx, out=None):
    """p (2^n doubles) into a new array, or into `out` (e.g. the numpy view of a pinned buffer)."""
    if out is None:
        out = np.empty(1 << ctx.n, dtype=np.float64)
    elif out.dtype != np.float64 or out.shape != (1 << ctx.n,) or not out.flags.c_contiguous:
        raise BAError(BA_EINVAL, "ba_get_p: out must be a contiguous float64 array of 2^n entries")
    _check(ctx, load().ba_get_p(ctx.handle, _dp(out)))
    return out


def ba_get_q(ctx):
    out = np.empty((2 << ctx.n) - 1, dtype=np.float64)
    _check(ctx, load().ba_get_q(ctx.handle, _dp(out)))
    return out


def ba_get_D(ctx):
    out = np.empty(1 << ctx.n, dtype=np.float64)
    _check(ctx, load().ba_get_D(ctx.handle, _dp(out)))
    return out


def ba_set_p(ctx, p):
    p = np.ascontiguousarray(p, dtype=np.float64)
    if p.shape != (1 << ctx.n,):
        raise BAError(BA_EINVAL, "ba_set_p: wrong shape")
    _check(ctx, load().ba_set_p(ctx.handle, _dp(p)))


def ba_debug_emb_row(ctx, x):
    out = np.zeros((2 << ctx.n) - 1, dtype=np.uint32)
    _check(ctx, load().ba_debug_emb_row(ctx.handle, int(x), out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint))))
    return out


def ba_debug_emb_col(ctx, yidx):
    out = np.zeros(1 << ctx.n, dtype=np.uint32)
    _check(ctx, load().ba_debug_emb_col(ctx.handle, int(yidx), out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint))))
    return out


def ba_terms_per_sweep(n):
    t = ctypes.c_ulonglong()
    rc = load().ba_terms_per_sweep(int(n), ctypes.byref(t))
    if rc != BA_OK:
        raise BAError(rc, "ba_terms_per_sweep")
    return t.value


def ba_debug_check_tables(m):
    """Host-only self-check of the pair tables for an m-bit low tile; returns (rc, [in_fast, in_riders, out_fast, out_riders])."""
    st = (ctypes.c_ulonglong * 4)()
    rc = load().ba_debug_check_tables(int(m), st)
    return rc, [int(x) for x in st]


def ba_debug_count_terms(ctx):
    v = [ctypes.c_ulonglong() for _ in range(4)]
    _check(ctx, load().ba_debug_count_terms(ctx.handle, *[ctypes.byref(x) for x in v]))
    return dict(in_terms=v[0].value, out_terms=v[1].value, in_emb_sum=v[2].value, out_emb_sum=v[3].value)


class BA:
    """Convenience wrapper: BA(n, d).iterate(k).bounds()."""

    def __init__(self, n, d, mode=BA_MODE_ENUM, p0=None, device="cuda:0"):
        self.ctx = ba_create(n, d, device=device)
        self.n, self.d = n, d
        ba_set_mode(self.ctx, mode)
        if p0 is not None:
            ba_set_p(self.ctx, p0)

    def iterate(self, k=1):
        ba_iterate(self.ctx, k)
        return self

    def bounds(self):
        return ba_bounds(self.ctx)

    def close(self):
        ba_destroy(self.ctx)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
