"""ctypes front end of the CPU oracle for the Jastrow u and p terms (oracle/jastrow_ref.c).  TEST
INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it.
It compiles jastrow_ref.c with gcc on first use (long double, OpenMP) and marshals numpy arrays; it contains
none of the method's arithmetic and nothing from the CUDA package.

Formulas: /root/reference/PAPER.md Eqs. 6-7 (lines 147-151); see jastrow_ref.c.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jastrow_ref.c")
_LIB = os.path.join(_HERE, "libjastrow_ref.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        i, d = ctypes.c_int, ctypes.c_double
        lib.jastrow_ref_batch.argtypes = [i, dp, i, dp, d, i, i, ip, ip, dp, i, i, dp, dp, dp, dp]
        lib.jastrow_ref_move_chain.argtypes = [i, dp, i, dp, d, i, i, ip, ip, dp, i, i, dp, i, ip, dp, dp, dp]
        lib.jastrow_ref_u.argtypes = [i, dp, d, i, d, dp, dp, dp]
        _lib = lib
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=ctypes.c_double):
    return a.ctypes.data_as(ctypes.POINTER(t))


def _cell9(cell, dim):
    c = np.zeros(9)
    c.reshape(3, 3)[:dim, :dim] = np.asarray(cell, dtype=np.float64).reshape(dim, dim)
    if dim == 2:
        c[8] = 1.0
    return c


def _terms(alpha, g_n, star, a):
    alpha = _d(alpha if alpha is not None else [])
    g_n = np.ascontiguousarray(g_n if g_n is not None else np.zeros((0, 3)), dtype=np.int32).reshape(-1, 3)
    star = np.ascontiguousarray(star if star is not None else [], dtype=np.int32)
    a = _d(a if a is not None else [0.0])
    return alpha, g_n, star, a


def batch(dim, cell, pos, alpha=None, L_u=0.0, C=3, g_n=None, star=None, a=None):
    """value [W], grad [W, n, dim], lap [W, n] of J = sum_{i<j} u(r_ij) + p(r_ij)."""
    pos = _d(pos)
    W, n, _ = pos.shape
    alpha, g_n, star, a = _terms(alpha, g_n, star, a)
    c = _cell9(cell, dim)
    value, grad, lap = np.zeros(W), np.zeros((W, n, dim)), np.zeros((W, n))
    rc = _load().jastrow_ref_batch(dim, _p(c), len(alpha) - 1, _p(alpha), float(L_u), int(C), len(g_n),
                                   _p(g_n, ctypes.c_int), _p(star, ctypes.c_int), _p(a), W, n, _p(pos),
                                   _p(value), _p(grad), _p(lap))
    assert rc == 0
    return value, grad, lap


def move_chain(dim, cell, pos, electron, new_r, alpha=None, L_u=0.0, C=3, g_n=None, star=None, a=None):
    """delta [S, W] of S sequential committed single-particle moves per walker; final positions."""
    pos = _d(pos)
    W, n, _ = pos.shape
    electron = np.ascontiguousarray(electron, dtype=np.int32)
    new_r = _d(new_r)
    S = electron.shape[0]
    alpha, g_n, star, a = _terms(alpha, g_n, star, a)
    c = _cell9(cell, dim)
    delta, pos_out = np.zeros((S, W)), np.zeros_like(pos)
    rc = _load().jastrow_ref_move_chain(dim, _p(c), len(alpha) - 1, _p(alpha), float(L_u), int(C), len(g_n),
                                        _p(g_n, ctypes.c_int), _p(star, ctypes.c_int), _p(a), W, n, _p(pos), S,
                                        _p(electron, ctypes.c_int), _p(new_r), _p(delta), _p(pos_out))
    assert rc == 0
    return delta, pos_out


def u(alpha, L_u, C, r):
    alpha = _d(alpha)
    v, d1, d2 = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _load().jastrow_ref_u(len(alpha) - 1, _p(alpha), float(L_u), int(C), float(r), ctypes.byref(v), ctypes.byref(d1),
                          ctypes.byref(d2))
    return v.value, d1.value, d2.value
