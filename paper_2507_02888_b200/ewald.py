"""Thin ctypes binding of include/ewald.h (argument marshalling only; every step runs in the CUDA library).

Same names as the C ABI: ewald_setup, ewald_set_fixed_charges, ewald_energy_batch,
ewald_energy_batch_host, ewald_load_walkers, ewald_move_delta_batch, ewald_move_delta_batch_host,
ewald_move_delta, ewald_get_rho, ...  Device buffers are torch CUDA tensors (PyTorch is used for device
memory and streams only); host buffers are numpy arrays.  There is no CPU fallback: if the shared
library cannot be built/loaded, or no CUDA device is usable, the calls raise.
"""
import ctypes
import os

import numpy as np

from . import build as _build

EWALD_F64, EWALD_F32 = 0, 1
_STATUS = {0: "EWALD_OK", 1: "EWALD_EINVAL", 2: "EWALD_ESINGULAR", 3: "EWALD_ERANGE",
           4: "EWALD_ESTATE", 5: "EWALD_ECUDA", 6: "EWALD_ENOMEM"}

# every symbol include/ewald.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ["ewald_padded_n", "ewald_setup", "ewald_setup_summary", "ewald_oct_plan_summary", "ewald_mma_plan_summary",
           "ewald_pair_table_eval",
           "ewald_destroy", "ewald_set_stream", "ewald_set_recip_variant", "ewald_set_real_variant",
           "ewald_set_fixed_charges", "ewald_energy_batch", "ewald_energy_batch_host", "ewald_recip_energy_static",
           "ewald_load_walkers", "ewald_move_delta_batch", "ewald_move_delta_batch_host",
           "ewald_move_delta", "ewald_num_g", "ewald_num_images", "ewald_r_cutoff", "ewald_get_g",
           "ewald_get_rho", "ewald_get_positions", "ewald_get_constants", "ewald_probe_fma", "ewald_probe_dmma",
           "ewald_profile_enable", "ewald_profile_read", "ewald_launch_count", "ewald_launch_shape",
           "ewald_last_error", "ewald_version"]


class EwaldError(RuntimeError):
    def __init__(self, status, message):
        self.status = status
        super().__init__("%s: %s" % (_STATUS.get(status, status), message))


class _Opts(ctypes.Structure):
    _fields_ = [("r_cutoff", ctypes.c_double), ("device", ctypes.c_int), ("stream", ctypes.c_void_p)]


_lib = None


def library_path():
    return _build.LIB


def load_library():
    """Load (building first if the sources are newer) libewald_b200.so; raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    lib = ctypes.CDLL(path)
    vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    sig = {
        "ewald_padded_n": (i, [i]),
        "ewald_setup": (i, [ctypes.POINTER(vp), i, dp, d, d, ctypes.POINTER(_Opts)]),
        "ewald_setup_summary": (i, [i, dp, d, d, d, ip, ip, ip, dp, dp]),
        "ewald_pair_table_eval": (i, [i, d, i, dp, dp]),
        "ewald_oct_plan_summary": (i, [i, dp, d, d, i, ip, ip, ip, dp, dp]),
        "ewald_mma_plan_summary": (i, [i, dp, d, d, ip, ip, dp, dp]),
        "ewald_destroy": (None, [vp]),
        "ewald_set_stream": (i, [vp, vp]),
        "ewald_set_recip_variant": (i, [vp, i]),
        "ewald_set_real_variant": (i, [vp, i]),
        "ewald_set_fixed_charges": (i, [vp, i, dp, dp]),
        "ewald_energy_batch": (i, [vp, i, i, i, vp, vp, vp, vp]),
        "ewald_energy_batch_host": (i, [vp, i, i, i, vp, vp, vp, vp]),
        "ewald_recip_energy_static": (i, [vp, i, i, i, vp, vp, vp]),
        "ewald_load_walkers": (i, [vp, i, i, i, vp, vp]),
        "ewald_move_delta_batch": (i, [vp, i, vp, vp, vp, i, vp]),
        "ewald_move_delta_batch_host": (i, [vp, i, vp, vp, vp, i, vp]),
        "ewald_move_delta": (i, [vp, i, i, dp, i, dp]),
        "ewald_num_g": (i, [vp]),
        "ewald_num_images": (i, [vp]),
        "ewald_r_cutoff": (d, [vp]),
        "ewald_get_g": (i, [vp, ip]),
        "ewald_get_rho": (i, [vp, i, dp]),
        "ewald_get_positions": (i, [vp, i, dp]),
        "ewald_get_constants": (i, [vp, dp, dp, dp]),
        "ewald_probe_fma": (i, [vp, i, i, dp]),
        "ewald_probe_dmma": (i, [vp, i, dp]),
        "ewald_profile_enable": (i, [vp, i]),
        "ewald_profile_read": (i, [vp, dp, ip]),
        "ewald_launch_shape": (i, [vp, i, ip]),
        "ewald_launch_count": (ctypes.c_longlong, [vp]),
        "ewald_last_error": (ctypes.c_char_p, [vp]),
        "ewald_version": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


class EwaldContext:
    """Owns one ewald_ctx*."""

    def __init__(self, handle, dim):
        self.handle = handle
        self.dim = dim

    def close(self):
        if self.handle:
            load_library().ewald_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _check(ctx, status):
    if status != 0:
        msg = load_library().ewald_last_error(ctx.handle if ctx else None)
        raise EwaldError(status, (msg or b"").decode())


def _cell9(cell, dim):
    a = np.asarray(cell, dtype=np.float64)
    c = np.zeros((3, 3))
    if a.size == 9:
        c[:] = a.reshape(3, 3)
    elif a.shape == (dim, dim):
        c[:dim, :dim] = a
    else:
        raise ValueError("cell must be (dim,dim) or 9 numbers")
    return np.ascontiguousarray(c.reshape(9))


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _prec_of(dtype):
    name = str(dtype).replace("torch.", "")
    if name == "float64":
        return EWALD_F64
    if name == "float32":
        return EWALD_F32
    raise TypeError("positions must be float64 or float32, got %s" % dtype)


def _dev_ptr(t, what):
    if t is None:
        return None
    if not (hasattr(t, "is_cuda") and t.is_cuda and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor" % what)
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def _dtype_name(t):
    return str(t.dtype).replace("torch.", "")


def _expect(t, what, dtype, shape):
    """Argument check of the binding (no arithmetic): dtype and shape of a tensor / array, None allowed."""
    if t is None:
        return
    if _dtype_name(t) != dtype:
        raise TypeError("%s must be %s, got %s" % (what, dtype, _dtype_name(t)))
    if tuple(t.shape) != tuple(shape):
        raise ValueError("%s must have shape %s, got %s" % (what, tuple(shape), tuple(t.shape)))


def _check_batch(ctx, n_particles, positions, charges, energies=None, components=None):
    if len(positions.shape) != 3 or positions.shape[1] != ctx.dim or positions.shape[2] != ewald_padded_n(n_particles):
        raise ValueError("positions must have shape [W, %d, %d] (SoA, n padded to 4), got %s"
                         % (ctx.dim, ewald_padded_n(n_particles), tuple(positions.shape)))
    _prec_of(positions.dtype)
    _expect(charges, "charges", _dtype_name(positions), (n_particles,))
    _expect(energies, "energies", "float64", (positions.shape[0],))
    _expect(components, "components", "float64", (positions.shape[0], 4))


def ewald_padded_n(n):
    return load_library().ewald_padded_n(n)


def to_soa(pos, dtype=np.float64):
    """[W, n, dim] points -> the library's [W, dim, n_pad] layout (zero padded); layout only."""
    pos = np.asarray(pos)
    w, n, dim = pos.shape
    out = np.zeros((w, dim, ewald_padded_n(n)), dtype=dtype)
    out[:, :, :n] = np.transpose(pos, (0, 2, 1))
    return out


def ewald_setup(dim, cell, gamma, g_cutoff, r_cutoff=0.0, device=0, stream=None):
    lib = load_library()
    h = ctypes.c_void_p()
    c = _cell9(cell, dim)
    opts = _Opts(float(r_cutoff), int(device), ctypes.c_void_p(stream) if stream else None)
    st = lib.ewald_setup(ctypes.byref(h), dim, _dp(c), float(gamma), float(g_cutoff), ctypes.byref(opts))
    if st != 0:
        raise EwaldError(st, "ewald_setup failed (no usable CUDA device?)" if st == 5 else "ewald_setup failed")
    return EwaldContext(h, dim)


def ewald_setup_summary(dim, cell, gamma, g_cutoff, r_cutoff=0.0):
    """Host-only dry run of the setup tables: dict(num_g, num_images, n_max, xi_r, v_m)."""
    c = _cell9(cell, dim)
    ng, ni, nm = ctypes.c_int(), ctypes.c_int(), (ctypes.c_int * 3)()
    xi, vm = ctypes.c_double(), ctypes.c_double()
    st = load_library().ewald_setup_summary(dim, _dp(c), float(gamma), float(g_cutoff), float(r_cutoff),
                                            ctypes.byref(ng), ctypes.byref(ni), nm, ctypes.byref(xi),
                                            ctypes.byref(vm))
    if st != 0:
        raise EwaldError(st, "ewald_setup_summary failed")
    return dict(num_g=ng.value, num_images=ni.value, n_max=list(nm), xi_r=xi.value, v_m=vm.value)


def ewald_oct_plan_summary(dim, cell, gamma, g_cutoff, n_walkers_per_cta=1):
    """Host-only: work plan of the octant-form reciprocal kernel (any cell)."""
    c = _cell9(cell, dim)
    ni, nb, nw = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    ws, fm = ctypes.c_double(), ctypes.c_double()
    st = load_library().ewald_oct_plan_summary(dim, _dp(c), float(gamma), float(g_cutoff),
                                               int(n_walkers_per_cta), ctypes.byref(ni), ctypes.byref(nb),
                                               ctypes.byref(nw), ctypes.byref(ws), ctypes.byref(fm))
    if st != 0:
        raise EwaldError(st, "ewald_oct_plan_summary failed")
    return dict(n_items=ni.value, npb=nb.value, n_warps=nw.value, weight_sum=ws.value,
                fma_per_particle=fm.value)


def ewald_mma_plan_summary(dim, cell, gamma, g_cutoff):
    """Host-only: plan of the tensor-core form of the octant kernel (any cell)."""
    c = _cell9(cell, dim)
    ns, wp = ctypes.c_int(), ctypes.c_int()
    ws, dq = ctypes.c_double(), ctypes.c_double()
    st = load_library().ewald_mma_plan_summary(dim, _dp(c), float(gamma), float(g_cutoff), ctypes.byref(ns),
                                               ctypes.byref(wp), ctypes.byref(ws), ctypes.byref(dq))
    if st != 0:
        raise EwaldError(st, "ewald_mma_plan_summary failed")
    return {"n_slots": ns.value, "walkers_per_pass": wp.value, "weight_sum": ws.value, "dmma_per_quad": dq.value}


def ewald_pair_table_eval(prec, t_max, t):
    """Host-only: the setup's piecewise polynomial for F(t) = erfc(sqrt t)/sqrt t evaluated at t (array)."""
    t = np.ascontiguousarray(t, dtype=np.float64)
    out = np.zeros_like(t)
    st = load_library().ewald_pair_table_eval(int(prec), float(t_max), t.size, _dp(t), _dp(out))
    if st != 0:
        raise EwaldError(st, "ewald_pair_table_eval failed")
    return out


def ewald_destroy(ctx):
    ctx.close()


def ewald_set_real_variant(ctx, variant):
    """0 default (FP64 kernels evaluate the far shell t >= 16 in FP32), 1 every term in FP64."""
    _check(ctx, load_library().ewald_set_real_variant(ctx.handle, int(variant)))


def ewald_set_recip_variant(ctx, variant):
    """0 automatic, 1 complex half-set reciprocal kernel, 2 octant-form kernel."""
    _check(ctx, load_library().ewald_set_recip_variant(ctx.handle, int(variant)))


def ewald_set_stream(ctx, stream):
    _check(ctx, load_library().ewald_set_stream(ctx.handle, ctypes.c_void_p(stream) if stream else None))


def ewald_set_fixed_charges(ctx, pos, q):
    q = np.ascontiguousarray(q, dtype=np.float64)
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(len(q), ctx.dim)
    _check(ctx, load_library().ewald_set_fixed_charges(ctx.handle, len(q), _dp(pos), _dp(q)))


def ewald_energy_batch(ctx, n_particles, positions, charges, energies, components=None):
    """positions: CUDA tensor [W, dim, n_pad]; charges: CUDA [n]; energies: CUDA float64 [W]."""
    _check_batch(ctx, n_particles, positions, charges, energies, components)
    w = positions.shape[0]
    _check(ctx, load_library().ewald_energy_batch(
        ctx.handle, w, n_particles, _prec_of(positions.dtype), _dev_ptr(positions, "positions"),
        _dev_ptr(charges, "charges"), _dev_ptr(energies, "energies"), _dev_ptr(components, "components")))


EWALD_STATIC_SCRATCH_BYTES = 1 << 20  # include/ewald.h


def ewald_recip_energy_static(ctx, n_particles, positions, charges, e_recip):
    """E_recip per walker with the kernel's scratch in the library's static device array: allocates nothing.
    positions: CUDA tensor [W, dim, n_pad]; charges: CUDA [n]; e_recip: CUDA float64 [W]."""
    _check_batch(ctx, n_particles, positions, charges, e_recip)
    _check(ctx, load_library().ewald_recip_energy_static(
        ctx.handle, positions.shape[0], n_particles, _prec_of(positions.dtype), _dev_ptr(positions, "positions"),
        _dev_ptr(charges, "charges"), _dev_ptr(e_recip, "e_recip")))


def ewald_energy_batch_host(ctx, n_particles, positions, charges, energies, components=None):
    """Same with numpy arrays (positions [W, dim, n_pad]); copies inside the call, synchronises."""
    _check_batch(ctx, n_particles, positions, charges, energies, components)
    w = positions.shape[0]
    if not (positions.flags.c_contiguous and charges.flags.c_contiguous and energies.flags.c_contiguous):
        raise TypeError("host arrays must be C-contiguous")
    _check(ctx, load_library().ewald_energy_batch_host(
        ctx.handle, w, n_particles, _prec_of(positions.dtype), _host_ptr(positions), _host_ptr(charges),
        _host_ptr(energies), _host_ptr(components)))


def ewald_load_walkers(ctx, n_particles, positions, charges):
    _check_batch(ctx, n_particles, positions, charges)
    ctx.loaded = (positions.shape[0], n_particles, _dtype_name(positions))
    _check(ctx, load_library().ewald_load_walkers(
        ctx.handle, positions.shape[0], n_particles, _prec_of(positions.dtype),
        _dev_ptr(positions, "positions"), _dev_ptr(charges, "charges")))


def ewald_move_delta_batch(ctx, walker, electron, new_r, commit, delta_e):
    """walker, electron: CUDA int32 [M]; new_r: CUDA [M, dim] in the loaded precision; delta_e: CUDA float64 [M]."""
    m = walker.shape[0]
    _expect(walker, "walker", "int32", (m,))
    _expect(electron, "electron", "int32", (m,))
    _expect(new_r, "new_r", getattr(ctx, "loaded", (0, 0, _dtype_name(new_r)))[2], (m, ctx.dim))
    _expect(delta_e, "delta_e", "float64", (m,))
    _check(ctx, load_library().ewald_move_delta_batch(
        ctx.handle, walker.shape[0], _dev_ptr(walker, "walker"), _dev_ptr(electron, "electron"),
        _dev_ptr(new_r, "new_r"), int(commit), _dev_ptr(delta_e, "delta_e")))


def ewald_move_delta_batch_host(ctx, walker, electron, new_r, commit, delta_e):
    m = walker.shape[0]
    _expect(walker, "walker", "int32", (m,))
    _expect(electron, "electron", "int32", (m,))
    _expect(new_r, "new_r", getattr(ctx, "loaded", (0, 0, _dtype_name(new_r)))[2], (m, ctx.dim))
    _expect(delta_e, "delta_e", "float64", (m,))
    _check(ctx, load_library().ewald_move_delta_batch_host(
        ctx.handle, walker.shape[0], _host_ptr(walker), _host_ptr(electron), _host_ptr(new_r),
        int(commit), _host_ptr(delta_e)))


def ewald_move_delta(ctx, walker, electron, new_r, commit=True):
    r = np.ascontiguousarray(new_r, dtype=np.float64)
    de = ctypes.c_double()
    _check(ctx, load_library().ewald_move_delta(ctx.handle, int(walker), int(electron), _dp(r),
                                                int(commit), ctypes.byref(de)))
    return de.value


def ewald_num_g(ctx):
    return load_library().ewald_num_g(ctx.handle)


def ewald_num_images(ctx):
    return load_library().ewald_num_images(ctx.handle)


def ewald_r_cutoff(ctx):
    return load_library().ewald_r_cutoff(ctx.handle)


def ewald_get_g(ctx):
    out = np.zeros((ewald_num_g(ctx) // 2, 3), dtype=np.int32)
    _check(ctx, load_library().ewald_get_g(ctx.handle, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
    return out


def ewald_get_rho(ctx, walker):
    out = np.zeros((ewald_num_g(ctx) // 2, 2))
    _check(ctx, load_library().ewald_get_rho(ctx.handle, int(walker), _dp(out)))
    return out[:, 0] + 1j * out[:, 1]


def ewald_get_positions(ctx, walker, n_particles):
    loaded = getattr(ctx, "loaded", None)
    if loaded is not None and n_particles != loaded[1]:
        raise ValueError("n_particles = %d, but %d particles per walker are loaded" % (n_particles, loaded[1]))
    out = np.zeros((n_particles, ctx.dim))
    _check(ctx, load_library().ewald_get_positions(ctx.handle, int(walker), _dp(out)))
    return out


def ewald_get_constants(ctx):
    xi, vm, ef = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(ctx, load_library().ewald_get_constants(ctx.handle, ctypes.byref(xi), ctypes.byref(vm),
                                                   ctypes.byref(ef)))
    return xi.value, vm.value, ef.value


def ewald_probe_fma(ctx, prec, iters=4096):
    f = ctypes.c_double()
    _check(ctx, load_library().ewald_probe_fma(ctx.handle, int(prec), int(iters), ctypes.byref(f)))
    return f.value


def ewald_probe_dmma(ctx, iters=4096):
    """FLOP/s of the FP64 tensor cores (m8n8k4 DMMA), the denominator of the tensor-core reciprocal kernel."""
    f = ctypes.c_double()
    _check(ctx, load_library().ewald_probe_dmma(ctx.handle, int(iters), ctypes.byref(f)))
    return f.value


KERNEL_CLASSES = ("recip", "real", "combine", "move")


def ewald_profile_enable(ctx, on=True):
    _check(ctx, load_library().ewald_profile_enable(ctx.handle, int(bool(on))))


def ewald_profile_read(ctx):
    """{class: (device ms, launches)} accumulated since the last read; synchronises and resets."""
    ms, cnt = (ctypes.c_double * 4)(), (ctypes.c_int * 4)()
    _check(ctx, load_library().ewald_profile_read(ctx.handle, ms, cnt))
    return {k: (ms[i], cnt[i]) for i, k in enumerate(KERNEL_CLASSES)}


def ewald_launch_shape(ctx, which):
    """Shape of the last real-space (which = 0) or move (which = 1) launch of the context, as a dict."""
    out = (ctypes.c_int * 8)()
    _check(ctx, load_library().ewald_launch_shape(ctx.handle, int(which), out))
    keys = ("threads", "smem_bytes", "cap_near", "cap_far", "near_bins", "far_bins", "ctas", "far_once")
    return dict(zip(keys, list(out)))


def ewald_launch_count(ctx):
    return load_library().ewald_launch_count(ctx.handle)


def ewald_version():
    return load_library().ewald_version().decode()
