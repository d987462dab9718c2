"""ctypes front end of the CPU oracle for blip orbitals (oracle/blip_ref.c).  TEST INFRASTRUCTURE ONLY: only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it.  Marshals numpy arrays; none of
the method's arithmetic and nothing from the CUDA package.  Formulas: see blip_ref.c."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "blip_ref.c")
_LIB = os.path.join(_HERE, "libblip_ref.so")
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
        lib.blip_ref_eval.argtypes = [dp, ip, i, dp, i, dp, dp, dp, dp]
        lib.blip_ref_theta.argtypes = [d, dp, dp, dp]
        _lib = lib
    return _lib


def _p(a, t=ctypes.c_double):
    return a.ctypes.data_as(ctypes.POINTER(t))


def theta(x):
    f, d1, d2 = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _load().blip_ref_theta(float(x), ctypes.byref(f), ctypes.byref(d1), ctypes.byref(d2))
    return f.value, d1.value, d2.value


def evaluate(cell, coef, points):
    """coef [n_orb, N1, N2, N3]; points [P, 3] -> psi [P, n_orb], grad [P, 3, n_orb], lap [P, n_orb]."""
    cell = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    coef = np.ascontiguousarray(coef, dtype=np.float64)
    points = np.ascontiguousarray(points, dtype=np.float64).reshape(-1, 3)
    n_orb, grid = coef.shape[0], np.array(coef.shape[1:], dtype=np.int32)
    P = len(points)
    psi, grad, lap = np.zeros((P, n_orb)), np.zeros((P, 3, n_orb)), np.zeros((P, n_orb))
    rc = _load().blip_ref_eval(_p(cell), _p(grid, ctypes.c_int), n_orb, _p(coef), P, _p(points), _p(psi), _p(grad), _p(lap))
    assert rc == 0
    return psi, grad, lap
