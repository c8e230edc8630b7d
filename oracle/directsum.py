"""ctypes loader for directsum.c (oracle).  Test infrastructure only.

`build()` compiles oracle/directsum.c with gcc -O2 -fopenmp into oracle/libdirectsum.so
(git-ignored); `__graft_entry__.build()` calls it so the checker exists on the GPU box.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libdirectsum.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "directsum.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, src])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        _lib.directsum_css.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ip, ip, dp, dp]
        _lib.directsum_css.restype = None
        _lib.directsum_cos_layer.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                             ip, ip, dp, dp]
        _lib.directsum_cos_layer.restype = None
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def css_mvm(theta, ix, iy, x):
    """q = W_s Sigma_ss W_s^T x from generators theta[N,2,N,2,L,L]; x: (N*2*nv,)."""
    lib = _load()
    N = theta.shape[0]
    C = 2 * N
    L = theta.shape[-1]
    n = (L + 1) // 2
    nv = ix.shape[0]
    th = np.ascontiguousarray(theta.reshape(C, C, L, L), dtype=np.float64)
    ixc = np.ascontiguousarray(ix, dtype=np.int32)
    iyc = np.ascontiguousarray(iy, dtype=np.int32)
    xv = np.ascontiguousarray(x, dtype=np.float64)
    q = np.empty(C * nv, dtype=np.float64)
    lib.directsum_css(_dp(th), C, n, nv, _ip(ixc), _ip(iyc), _dp(xv), _dp(q))
    return q


def cos_layer(xi_k, n, n_p, ix, iy, x):
    """g_k (n' x n') = Xi'_k x for one layer from xi_k[N,2,L,L]."""
    lib = _load()
    C = xi_k.shape[0] * xi_k.shape[1]
    L = xi_k.shape[-1]
    nv = ix.shape[0]
    t = np.ascontiguousarray(xi_k.reshape(C, L, L), dtype=np.float64)
    ixc = np.ascontiguousarray(ix, dtype=np.int32)
    iyc = np.ascontiguousarray(iy, dtype=np.int32)
    xv = np.ascontiguousarray(x, dtype=np.float64)
    g = np.empty(n_p * n_p, dtype=np.float64)
    lib.directsum_cos_layer(_dp(t), C, n, n_p, nv, _ip(ixc), _ip(iyc), _dp(xv), _dp(g))
    return g.reshape(n_p, n_p)


def n_threads() -> int:
    return len(os.sched_getaffinity(0))
