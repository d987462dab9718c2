"""ctypes binding of include/blip.h (same names, argument marshalling only; the evaluation runs in blip_kernel of
csrc/blip_api.cu).  Raises if the library is missing or a call fails."""
import ctypes

import numpy as np

from . import ewald as _E

SYMBOLS = ["blip_setup", "blip_eval_batch", "blip_profile_enable", "blip_profile_read", "blip_last_error", "blip_destroy"]
_sigs_done = False


def _lib():
    global _sigs_done
    lib = _E.load_library()
    if not _sigs_done:
        vp, i = ctypes.c_void_p, ctypes.c_int
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        sig = {"blip_setup": (i, [ctypes.POINTER(vp), dp, ip, i, dp, i, vp]),
               "blip_eval_batch": (i, [vp, i, i, i, vp, vp, vp, vp]),
               "blip_profile_enable": (i, [vp, i]),
               "blip_profile_read": (i, [vp, dp, ip]),
               "blip_last_error": (ctypes.c_char_p, [vp]),
               "blip_destroy": (None, [vp])}
        for name, (res, args) in sig.items():
            f = getattr(lib, name)
            f.restype, f.argtypes = res, args
        _sigs_done = True
    return lib


class BlipContext:
    def __init__(self, handle, n_orb):
        self.handle, self.n_orb = handle, n_orb

    def close(self):
        if self.handle:
            _lib().blip_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _check(ctx, status):
    if status != 0:
        msg = _lib().blip_last_error(ctx.handle if ctx else None)
        raise _E.EwaldError(status, (msg or b"").decode())


def blip_setup(cell, coef, device=0, stream=None):
    """coef: numpy [n_orb, N1, N2, N3]."""
    cell = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    coef = np.ascontiguousarray(coef, dtype=np.float64)
    if coef.ndim != 4:
        raise ValueError("coef must have shape [n_orb, N1, N2, N3]")
    grid = np.array(coef.shape[1:], dtype=np.int32)
    h = ctypes.c_void_p()
    st = _lib().blip_setup(ctypes.byref(h), _E._dp(cell), grid.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), coef.shape[0],
                           _E._dp(coef), int(device), ctypes.c_void_p(stream) if stream else None)
    if st != 0:
        raise _E.EwaldError(st, "blip_setup failed")
    return BlipContext(h, coef.shape[0])


def blip_eval_batch(ctx, n_points, points, psi, grad=None, lap=None):
    """points: CUDA [3, n_pad]; psi: CUDA float64 [n_points, n_orb]; grad: [n_points, 3, n_orb]; lap: [n_points, n_orb]."""
    if len(points.shape) != 2 or points.shape[0] != 3 or points.shape[1] < n_points:
        raise ValueError("points must have shape [3, n_pad >= n_points]")
    _E._expect(psi, "psi", "float64", (n_points, ctx.n_orb))
    _E._expect(grad, "grad", "float64", (n_points, 3, ctx.n_orb))
    _E._expect(lap, "lap", "float64", (n_points, ctx.n_orb))
    _check(ctx, _lib().blip_eval_batch(ctx.handle, int(n_points), int(points.shape[1]), _E._prec_of(points.dtype),
                                       _E._dev_ptr(points, "points"), _E._dev_ptr(psi, "psi"),
                                       _E._dev_ptr(grad, "grad"), _E._dev_ptr(lap, "lap")))


def blip_profile_enable(ctx, on=True):
    _check(ctx, _lib().blip_profile_enable(ctx.handle, int(bool(on))))


def blip_profile_read(ctx):
    ms, cnt = ctypes.c_double(), ctypes.c_int()
    _check(ctx, _lib().blip_profile_read(ctx.handle, ctypes.byref(ms), ctypes.byref(cnt)))
    return ms.value, cnt.value


def blip_destroy(ctx):
    ctx.close()
