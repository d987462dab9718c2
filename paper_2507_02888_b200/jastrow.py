"""ctypes binding of include/jastrow.h (same names, argument marshalling only; every step runs in the CUDA
kernels of csrc/jastrow_kernels.cuh).  Raises if the library is missing or a call fails."""
import ctypes

import numpy as np

from . import ewald as _E

SYMBOLS = ["jastrow_setup", "jastrow_batch", "jastrow_load_walkers", "jastrow_move_delta_batch",
           "jastrow_profile_enable", "jastrow_profile_read", "jastrow_last_error", "jastrow_destroy"]

_sigs_done = False


def _lib():
    global _sigs_done
    lib = _E.load_library()
    if not _sigs_done:
        vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        sig = {"jastrow_setup": (i, [ctypes.POINTER(vp), i, dp, i, dp, d, i, i, ip, ip, i, dp, i, vp]),
               "jastrow_batch": (i, [vp, i, i, i, vp, vp, vp, vp]),
               "jastrow_load_walkers": (i, [vp, i, i, i, vp]),
               "jastrow_move_delta_batch": (i, [vp, i, vp, vp, vp, i, vp]),
               "jastrow_profile_enable": (i, [vp, i]),
               "jastrow_profile_read": (i, [vp, dp, ip]),
               "jastrow_last_error": (ctypes.c_char_p, [vp]),
               "jastrow_destroy": (None, [vp])}
        for name, (res, args) in sig.items():
            f = getattr(lib, name)
            f.restype, f.argtypes = res, args
        _sigs_done = True
    return lib


class JastrowContext:
    def __init__(self, handle, dim):
        self.handle, self.dim = handle, dim

    def close(self):
        if self.handle:
            _lib().jastrow_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _check(ctx, status):
    if status != 0:
        msg = _lib().jastrow_last_error(ctx.handle if ctx else None)
        raise _E.EwaldError(status, (msg or b"").decode())


def jastrow_setup(dim, cell, alpha=None, l_u=0.0, c_exp=3, g_n=None, star=None, a=None, device=0, stream=None):
    c = _E._cell9(cell, dim)
    alpha = np.ascontiguousarray(alpha if alpha is not None else [], dtype=np.float64)
    g_n = np.ascontiguousarray(g_n if g_n is not None else np.zeros((0, 3)), dtype=np.int32).reshape(-1, 3)
    star = np.ascontiguousarray(star if star is not None else [], dtype=np.int32)
    a = np.ascontiguousarray(a if a is not None else [0.0], dtype=np.float64)
    h = ctypes.c_void_p()
    ip = ctypes.POINTER(ctypes.c_int)
    st = _lib().jastrow_setup(ctypes.byref(h), dim, _E._dp(c), len(alpha) - 1, _E._dp(alpha), float(l_u), int(c_exp),
                              len(g_n), g_n.ctypes.data_as(ip), star.ctypes.data_as(ip), len(a), _E._dp(a), int(device),
                              ctypes.c_void_p(stream) if stream else None)
    if st != 0:
        raise _E.EwaldError(st, "jastrow_setup failed")
    return JastrowContext(h, dim)


def jastrow_batch(ctx, n_particles, positions, value, grad=None, lap=None):
    """positions: CUDA [W, dim, n_pad]; value: CUDA float64 [W]; grad: CUDA float64 [W, dim, n_pad]; lap: [W, n_pad]."""
    w, npad = positions.shape[0], _E.ewald_padded_n(n_particles)
    if tuple(positions.shape) != (w, ctx.dim, npad):
        raise ValueError("positions must have shape [W, %d, %d]" % (ctx.dim, npad))
    _E._expect(value, "value", "float64", (w,))
    _E._expect(grad, "grad", "float64", (w, ctx.dim, npad))
    _E._expect(lap, "lap", "float64", (w, npad))
    _check(ctx, _lib().jastrow_batch(ctx.handle, w, n_particles, _E._prec_of(positions.dtype),
                                     _E._dev_ptr(positions, "positions"), _E._dev_ptr(value, "value"),
                                     _E._dev_ptr(grad, "grad"), _E._dev_ptr(lap, "lap")))


def jastrow_load_walkers(ctx, n_particles, positions):
    w, npad = positions.shape[0], _E.ewald_padded_n(n_particles)
    if tuple(positions.shape) != (w, ctx.dim, npad):
        raise ValueError("positions must have shape [W, %d, %d]" % (ctx.dim, npad))
    ctx.loaded = (w, n_particles, _E._dtype_name(positions))
    _check(ctx, _lib().jastrow_load_walkers(ctx.handle, w, n_particles, _E._prec_of(positions.dtype),
                                            _E._dev_ptr(positions, "positions")))


def jastrow_move_delta_batch(ctx, walker, electron, new_r, commit, delta):
    m = walker.shape[0]
    _E._expect(walker, "walker", "int32", (m,))
    _E._expect(electron, "electron", "int32", (m,))
    _E._expect(new_r, "new_r", getattr(ctx, "loaded", (0, 0, _E._dtype_name(new_r)))[2], (m, ctx.dim))
    _E._expect(delta, "delta", "float64", (m,))
    _check(ctx, _lib().jastrow_move_delta_batch(ctx.handle, m, _E._dev_ptr(walker, "walker"), _E._dev_ptr(electron, "electron"),
                                                _E._dev_ptr(new_r, "new_r"), int(commit), _E._dev_ptr(delta, "delta")))


def jastrow_profile_enable(ctx, on=True):
    _check(ctx, _lib().jastrow_profile_enable(ctx.handle, int(bool(on))))


def jastrow_profile_read(ctx):
    ms, cnt = ctypes.c_double(), ctypes.c_int()
    _check(ctx, _lib().jastrow_profile_read(ctx.handle, ctypes.byref(ms), ctypes.byref(cnt)))
    return ms.value, cnt.value


def jastrow_destroy(ctx):
    ctx.close()
