"""ctypes front end of the CPU oracle (oracle/ewald_ref.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It compiles ewald_ref.c with gcc on first use (long double, OpenMP) and marshals numpy arrays;
it contains none of the method's arithmetic and nothing from the CUDA package.

Formulas: /root/reference/PAPER.md Eqs. 2-4 (lines 112-120); see ewald_ref.h.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ewald_ref.c")
_HDR = os.path.join(_HERE, "ewald_ref.h")
_LIB = os.path.join(_HERE, "libewald_ref.so")

_lib = None


def build(force=False):
    """Compile the oracle shared library next to its source (gcc, -O2, OpenMP)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        i, d = ctypes.c_int, ctypes.c_double
        lib.ewald_ref_num_g.argtypes = [i, dp, d]
        lib.ewald_ref_gplus.argtypes = [i, dp, d, ip]
        lib.ewald_ref_auto_cutoffs.argtypes = [i, dp, d, d, dp, dp]
        lib.ewald_ref_energy_pairwise.argtypes = [i, dp, d, d, d, i, dp, dp, dp]
        lib.ewald_ref_v_e.argtypes = [i, dp, d, d, d, dp, dp]
        lib.ewald_ref_v_m.argtypes = [i, dp, d, d, d, dp]
        lib.ewald_ref_energy_batch.argtypes = [i, dp, d, d, d, i, i, dp, dp, i, dp, dp, dp, dp, i]
        lib.ewald_ref_rho.argtypes = [i, dp, d, i, dp, dp, dp]
        lib.ewald_ref_move_chain.argtypes = [i, dp, d, d, d, i, i, dp, dp, i, dp, dp, i, ip, dp, dp,
                                             dp, i]
        lib.ewald_ref_max_threads.argtypes = []
        _lib = lib
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _cell9(cell, dim):
    c = np.zeros((3, 3))
    a = np.asarray(cell, dtype=np.float64)
    if a.size == 9:
        c[:] = a.reshape(3, 3)
    elif a.shape == (dim, dim):
        c[:dim, :dim] = a
    else:
        raise ValueError("cell must be (dim,dim) or 9 numbers")
    return _d(c.reshape(9))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (what, rc))


def max_threads():
    return int(_load().ewald_ref_max_threads())


def num_g(dim, cell, g_cutoff):
    c = _cell9(cell, dim)
    n = _load().ewald_ref_num_g(dim, _p(c), g_cutoff)
    if n < 0:
        raise RuntimeError("ewald_ref_num_g failed")
    return n


def gplus(dim, cell, g_cutoff):
    """Integer triples (n1,n2,n3) of the half set, lexicographic order; shape [num_g/2, 3]."""
    c = _cell9(cell, dim)
    n = num_g(dim, cell, g_cutoff) // 2
    out = np.zeros((n, 3), dtype=np.int32)
    _check(_load().ewald_ref_gplus(dim, _p(c), g_cutoff,
                                   out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))), "gplus")
    return out


def auto_cutoffs(dim, cell, kappa, tol=1e-17):
    c = _cell9(cell, dim)
    g, r = ctypes.c_double(), ctypes.c_double()
    _check(_load().ewald_ref_auto_cutoffs(dim, _p(c), kappa, tol, ctypes.byref(g), ctypes.byref(r)),
           "auto_cutoffs")
    return g.value, r.value


def energy_pairwise(dim, cell, kappa, g_cutoff, r_cutoff, pos, q):
    """Eq. 2 with Eqs. 3-4 evaluated literally (O-pair)."""
    c = _cell9(cell, dim)
    pos = _d(pos).reshape(-1, dim)
    q = _d(q)
    e = ctypes.c_double()
    _check(_load().ewald_ref_energy_pairwise(dim, _p(c), kappa, g_cutoff, r_cutoff, len(q), _p(pos),
                                             _p(q), ctypes.byref(e)), "energy_pairwise")
    return e.value


def v_e(dim, cell, kappa, g_cutoff, r_cutoff, r):
    c = _cell9(cell, dim)
    r = _d(r)
    v = ctypes.c_double()
    _check(_load().ewald_ref_v_e(dim, _p(c), kappa, g_cutoff, r_cutoff, _p(r), ctypes.byref(v)), "v_e")
    return v.value


def v_m(dim, cell, kappa, g_cutoff, r_cutoff):
    c = _cell9(cell, dim)
    v = ctypes.c_double()
    _check(_load().ewald_ref_v_m(dim, _p(c), kappa, g_cutoff, r_cutoff, ctypes.byref(v)), "v_m")
    return v.value


def energy_batch(dim, cell, kappa, g_cutoff, r_cutoff, pos, q, ion_pos=None, ion_q=None,
                 n_threads=0):
    """O-rho energies. pos: [n_walkers, n, dim]. Returns (energies [W], components [W,4])."""
    c = _cell9(cell, dim)
    q = _d(q)
    n = len(q)
    pos = _d(pos).reshape(-1, n, dim) if n else np.zeros((np.shape(pos)[0], 0, dim))
    nw = pos.shape[0]
    n_ion = 0 if ion_q is None else len(ion_q)
    ip = _d(ion_pos).reshape(n_ion, dim) if n_ion else None
    iq = _d(ion_q) if n_ion else None
    e = np.zeros(nw)
    comp = np.zeros((nw, 4))
    _check(_load().ewald_ref_energy_batch(dim, _p(c), kappa, g_cutoff, r_cutoff, nw, n, _p(pos),
                                          _p(q), n_ion, _p(ip), _p(iq), _p(e), _p(comp),
                                          n_threads), "energy_batch")
    return e, comp


def rho(dim, cell, g_cutoff, pos, q):
    """rho(G) on the half set (order of gplus) as a complex array."""
    c = _cell9(cell, dim)
    q = _d(q)
    pos = _d(pos).reshape(len(q), dim)
    n = num_g(dim, cell, g_cutoff) // 2
    out = np.zeros((n, 2))
    _check(_load().ewald_ref_rho(dim, _p(c), g_cutoff, len(q), _p(pos), _p(q), _p(out)), "rho")
    return out[:, 0] + 1j * out[:, 1]


def move_chain(dim, cell, kappa, g_cutoff, r_cutoff, pos, q, electron, new_r, ion_pos=None,
               ion_q=None, want_rho=False, n_threads=0):
    """Incremental single-move oracle.

    pos [W,n,dim] (a copy is updated and returned), electron [S,W] int, new_r [S,W,dim].
    Returns (delta_e [S,W], final_pos [W,n,dim], rho [W,num_g/2] complex or None).
    """
    c = _cell9(cell, dim)
    q = _d(q)
    n = len(q)
    pos = np.array(pos, dtype=np.float64).reshape(-1, n, dim).copy()
    nw = pos.shape[0]
    electron = np.ascontiguousarray(electron, dtype=np.int32).reshape(-1, nw)
    ns = electron.shape[0]
    new_r = _d(new_r).reshape(ns, nw, dim)
    n_ion = 0 if ion_q is None else len(ion_q)
    ip = _d(ion_pos).reshape(n_ion, dim) if n_ion else None
    iq = _d(ion_q) if n_ion else None
    de = np.zeros((ns, nw))
    rho_out = np.zeros((nw, num_g(dim, cell, g_cutoff) // 2, 2)) if want_rho else None
    _check(_load().ewald_ref_move_chain(dim, _p(c), kappa, g_cutoff, r_cutoff, nw, n, _p(pos), _p(q),
                                        n_ion, _p(ip), _p(iq), ns,
                                        electron.ctypes.data_as(ctypes.POINTER(ctypes.c_int)),
                                        _p(new_r), _p(de), _p(rho_out), n_threads), "move_chain")
    rho_c = None if rho_out is None else rho_out[..., 0] + 1j * rho_out[..., 1]
    return de, pos, rho_c
