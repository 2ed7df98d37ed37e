"""ctypes loader for the CPU oracle (oracle/ba_oracle.c) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It never imports the CUDA package.

The wrapper only marshals numpy arrays; all arithmetic is in ba_oracle.c, whose header cites
the passages of PAPER.md ("P:line") each step follows.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ba_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    """Compile ba_oracle.c into oracle/liboracle.so with gcc (-O2, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_up = ctypes.POINTER(ctypes.c_uint32)
        L.orc_num_threads.restype = ctypes.c_int
        L.orc_emb_dense.argtypes = [ctypes.c_int, c_up]
        L.orc_emb_row.argtypes = [ctypes.c_int, ctypes.c_uint32, c_up]
        L.orc_D_row.argtypes = [ctypes.c_int, ctypes.c_double, c_up, c_dp, c_dp, ctypes.POINTER(ctypes.c_int64)]
        L.orc_weights.argtypes = [ctypes.c_int, ctypes.c_double, c_dp]
        L.orc_channel_from_emb.argtypes = [ctypes.c_int, ctypes.c_double, c_up, c_dp]
        L.orc_ba_step.argtypes = [ctypes.c_int64, ctypes.c_int64, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp]
        L.orc_ba_run.argtypes = [ctypes.c_int64, ctypes.c_int64, c_dp, c_dp, ctypes.c_int,
                                 c_dp, c_dp, c_dp, c_dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _up(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32))


def num_threads():
    return int(lib().orc_num_threads())


def sizes(n):
    return 1 << n, (1 << (n + 1)) - 1


def emb_dense(n):
    """E[x, idx(y)] = emb(y, x), uint32, by brute-force keep-mask enumeration."""
    NX, NY = sizes(n)
    E = np.zeros((NX, NY), dtype=np.uint32)
    rc = lib().orc_emb_dense(n, _up(E))
    if rc:
        raise ValueError(f"orc_emb_dense rc={rc}")
    return E


def emb_row(n, x):
    """Row x of the emb matrix by keep-mask enumeration of that one input; n <= 30."""
    NX, NY = sizes(n)
    row = np.empty(NY, dtype=np.uint32)
    rc = lib().orc_emb_row(n, int(x), _up(row))
    if rc:
        raise ValueError(f"orc_emb_row rc={rc}")
    return row


def D_row(n, d, row, q):
    """(D(x), number of non-zero terms) of one input from its emb row and q, by the definition."""
    row = np.ascontiguousarray(row, dtype=np.uint32)
    q = np.ascontiguousarray(q, dtype=np.float64)
    NX, NY = sizes(n)
    if row.shape != (NY,) or q.shape != (NY,):
        raise ValueError("D_row: row and q must have 2^(n+1)-1 entries")
    out = ctypes.c_double()
    nt = ctypes.c_int64()
    rc = lib().orc_D_row(n, float(d), _up(row), _dp(q), ctypes.byref(out), ctypes.byref(nt))
    if rc:
        raise ValueError(f"orc_D_row rc={rc}")
    return float(out.value), int(nt.value)


def weights(n, d):
    w = np.zeros(n + 1, dtype=np.float64)
    rc = lib().orc_weights(n, float(d), _dp(w))
    if rc:
        raise ValueError(f"orc_weights rc={rc}")
    return w


def channel(n, d, E=None):
    """Explicit channel matrix W[x, idx(y)] = emb(y,x) (1-d)^|y| d^(n-|y|) (north_star)."""
    if E is None:
        E = emb_dense(n)
    W = np.empty(E.shape, dtype=np.float64)
    rc = lib().orc_channel_from_emb(n, float(d), _up(np.ascontiguousarray(E)), _dp(W))
    if rc:
        raise ValueError(f"orc_channel_from_emb rc={rc}")
    return W


def ba_step(W, p):
    """One BA iteration on an explicit matrix. Returns dict(q, D, I, U, log2Z, p_next)."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    p = np.ascontiguousarray(p, dtype=np.float64)
    NX, NY = W.shape
    q = np.empty(NY)
    D = np.empty(NX)
    st = np.empty(3)
    pn = np.empty(NX)
    rc = lib().orc_ba_step(NX, NY, _dp(W), _dp(p), _dp(q), _dp(D), _dp(st), _dp(pn))
    if rc:
        raise ValueError(f"orc_ba_step rc={rc}")
    return dict(q=q, D=D, I=float(st[0]), U=float(st[1]), log2Z=float(st[2]), p_next=pn)


def ba_run(W, p0, K):
    """K BA iterations. Returns dict(hist[K,3]={I_t,U_t,log2Z_t}, p=p_K, q=q_{K-1}, D=D_{K-1}) (R6)."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    p0 = np.ascontiguousarray(p0, dtype=np.float64)
    NX, NY = W.shape
    hist = np.zeros((max(K, 1), 3))
    p = np.empty(NX)
    q = np.zeros(NY)
    D = np.zeros(NX)
    rc = lib().orc_ba_run(NX, NY, _dp(W), _dp(p0), int(K), _dp(hist), _dp(p), _dp(q), _dp(D))
    if rc:
        raise ValueError(f"orc_ba_run rc={rc}")
    return dict(hist=hist[:K], p=p, q=q, D=D)
