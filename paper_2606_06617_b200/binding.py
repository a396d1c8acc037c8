"""Thin Python binding of libpswf_lr.so (ctypes): argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch appears only as the owner of device
memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream()``).  Names mirror
include/pswf_lr.h.  There is no CPU fallback: loading fails loudly when the shared library is
missing and plan creation fails loudly when no CUDA device is usable.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpswf_lr.so")

PSWF_LR_F32, PSWF_LR_F64 = 0, 1
N_STAGES = 6
STAGE_NAMES = ("bin_sort", "spread", "fft_forward", "scale_reduce", "fft_inverse", "gather")

ERR_INVALID_ARG, ERR_UNSUPPORTED_EXPONENT, ERR_GRID_TOO_COARSE, ERR_ALLOC, ERR_CUDA, ERR_CUFFT = \
    -1, -2, -3, -4, -5, -6
ERR_BUSY, ERR_TOO_LARGE = -7, -8


class PswfLrError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pswf_lr error %d: %s" % (code, msg))
        self.code = code


class Opts(ctypes.Structure):
    _fields_ = [("r_c", ctypes.c_double), ("c_window", ctypes.c_double), ("precision", ctypes.c_int),
                ("max_atoms", ctypes.c_int), ("zero_mode", ctypes.c_int), ("kernel_path", ctypes.c_int),
                ("poly_eps", ctypes.c_double), ("host_only", ctypes.c_int), ("debug_spectrum", ctypes.c_int)]


class Info(ctypes.Structure):
    _fields_ = [("r_c", ctypes.c_double), ("c", ctypes.c_double), ("c_window", ctypes.c_double),
                ("eta", ctypes.c_double), ("w", ctypes.c_int), ("precision", ctypes.c_int),
                ("n_channels", ctypes.c_int), ("n_distinct_p", ctypes.c_int), ("grid", ctypes.c_int * 3),
                ("window_degree", ctypes.c_int), ("kernel_degree", ctypes.c_int),
                ("kernel_panels", ctypes.c_int), ("modes_in_ball", ctypes.c_longlong),
                ("workspace_bytes", ctypes.c_longlong), ("fast_stencil", ctypes.c_int),
                ("band_limited_fft", ctypes.c_int), ("band_kmax", ctypes.c_int * 3),
                ("own_kernel_launches", ctypes.c_longlong), ("memsets", ctypes.c_longlong),
                ("cufft_execs", ctypes.c_longlong), ("graph_replays", ctypes.c_longlong)]


EXPORTS = ("pswf_lr_plan_create", "pswf_lr_plan_create_ex", "pswf_lr_plan_create_cell", "pswf_lr_execute", "pswf_lr_execute_host",
           "pswf_lr_submit_host", "pswf_lr_wait_host",
           "pswf_lr_execute_real", "pswf_lr_eval_real", "pswf_lr_self_coefficient", "pswf_lr_suggest_parameters", "pswf_lr_set_virial", "pswf_lr_virial",
           "pswf_lr_channel_energies", "pswf_lr_get_info", "pswf_lr_set_profiling", "pswf_lr_stage_ms",
           "pswf_lr_debug_copy", "pswf_lr_debug_cell_starts", "pswf_lr_exclusive_scan_static", "pswf_lr_eval_window", "pswf_lr_eval_kernel", "pswf_lr_destroy",
           "pswf_lr_error_string", "pswf_lr_version")

_lib = None


def lib():
    """Load libpswf_lr.so (built by ``python -m paper_2606_06617_b200.build``).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libpswf_lr.so is missing at %s: build it with "
                              "`python -m paper_2606_06617_b200.build` (nvcc, sm_100a). "
                              "There is no CPU fallback." % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, ip, dp = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)
        L.pswf_lr_plan_create.argtypes = [ctypes.POINTER(vp), dp, ctypes.POINTER(ip), ip, ctypes.c_double,
                                          ctypes.POINTER(ip), ip]
        L.pswf_lr_plan_create_ex.argtypes = L.pswf_lr_plan_create.argtypes + [ctypes.POINTER(Opts)]
        L.pswf_lr_plan_create_cell.argtypes = L.pswf_lr_plan_create_ex.argtypes
        L.pswf_lr_submit_host.argtypes = [vp, ip, vp, vp, dp, vp, vp]
        L.pswf_lr_wait_host.argtypes = [vp]
        L.pswf_lr_execute.argtypes = [vp, ip, vp, vp, vp, vp, vp, vp]
        L.pswf_lr_execute_host.argtypes = [vp, ip, vp, vp, dp, vp, vp, vp]
        L.pswf_lr_execute_real.argtypes = [vp, ip, vp, vp, vp, vp, vp, ip, vp]
        L.pswf_lr_eval_real.argtypes = [vp, ip, ip, dp, dp, dp]
        L.pswf_lr_self_coefficient.argtypes = [vp, ip, dp]
        L.pswf_lr_suggest_parameters.argtypes = [dp, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ip),
                                                 ctypes.POINTER(ip), dp]
        L.pswf_lr_set_virial.argtypes = [vp, ip]
        L.pswf_lr_virial.argtypes = [vp, vp, vp]
        L.pswf_lr_channel_energies.argtypes = [vp, vp, vp]
        L.pswf_lr_get_info.argtypes = [vp, ctypes.POINTER(Info)]
        L.pswf_lr_set_profiling.argtypes = [vp, ip]
        L.pswf_lr_stage_ms.argtypes = [vp, dp, ctypes.POINTER(ip)]
        L.pswf_lr_debug_copy.argtypes = [vp, ip, vp, vp]
        L.pswf_lr_debug_cell_starts.argtypes = [vp, vp, vp]
        L.pswf_lr_exclusive_scan_static.argtypes = [vp, ip, vp]
        L.pswf_lr_eval_window.argtypes = [vp, ip, dp, dp, dp]
        L.pswf_lr_eval_kernel.argtypes = [vp, ip, ip, dp, dp]
        L.pswf_lr_destroy.argtypes = [vp]
        for name in EXPORTS:
            getattr(L, name).restype = ip
        L.pswf_lr_error_string.restype = ctypes.c_char_p
        L.pswf_lr_error_string.argtypes = [ip]
        L.pswf_lr_version.restype = ctypes.c_char_p
        L.pswf_lr_version.argtypes = []
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise PswfLrError(rc, lib().pswf_lr_error_string(rc).decode())


def _ptr(t):
    """Raw device (or host) pointer of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return ctypes.c_void_p(t.ctypes.data)
    return ctypes.c_void_p(t.data_ptr())


SCAN_STATIC_MAX = 1 << 24


def exclusive_scan_static(counts, n, stream=None):
    """pswf_lr_exclusive_scan_static: in-place exclusive scan of the int32 device tensor counts[n + 1]
    (counts[n] receives the total) with the library's static scratch; allocates nothing."""
    _check(lib().pswf_lr_exclusive_scan_static(_ptr(counts), int(n), ctypes.c_void_p(stream or 0)))


def suggest_parameters(box, eps_tot, r_c):
    """(grid, w, c) for a target tolerance: Eq. (27)-(29) as read in include/pswf_lr.h (host only)."""
    bx = (ctypes.c_double * 3)(*[float(v) for v in box])
    grid = (ctypes.c_int * 3)()
    w = ctypes.c_int(0)
    c = ctypes.c_double(0.0)
    _check(lib().pswf_lr_suggest_parameters(bx, float(eps_tot), float(r_c), grid, ctypes.byref(w), ctypes.byref(c)))
    return list(grid), w.value, c.value


class Plan:
    """pswf_lr_plan_create_ex / pswf_lr_execute / pswf_lr_destroy."""

    def __init__(self, box, grid, w, c, exponents, r_c=0.0, c_window=0.0, precision="f32", max_atoms=0,
                 zero_mode=0, kernel_path=0, poly_eps=0.0, host_only=False, debug_spectrum=False):
        self._h = ctypes.c_void_p()
        L = lib()
        self.precision = {"f32": PSWF_LR_F32, "f64": PSWF_LR_F64}[precision]
        o = Opts(r_c, c_window, self.precision, int(max_atoms), zero_mode, kernel_path, poly_eps,
                 1 if host_only else 0, 1 if debug_spectrum else 0)
        grid_a = (ctypes.c_int * 3)(*[int(g) for g in grid])
        ex = (ctypes.c_int * len(exponents))(*[int(p) for p in exponents])
        box_np = np.asarray(box, dtype=np.float64)
        if box_np.ndim == 2:     # 3x3 cell, rows = lattice vectors
            cell_a = (ctypes.c_double * 9)(*[float(b) for b in box_np.reshape(9)])
            _check(L.pswf_lr_plan_create_cell(ctypes.byref(self._h), cell_a, grid_a, int(w), float(c), ex,
                                              len(exponents), ctypes.byref(o)))
        else:
            box_a = (ctypes.c_double * 3)(*[float(b) for b in box_np])
            _check(L.pswf_lr_plan_create_ex(ctypes.byref(self._h), box_a, grid_a, int(w), float(c), ex,
                                            len(exponents), ctypes.byref(o)))
        self.n_channels = len(exponents)
        self.grid = [int(g) for g in grid]

    # -- lifetime --
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().pswf_lr_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    # -- queries --
    def info(self):
        i = Info()
        _check(lib().pswf_lr_get_info(self._h, ctypes.byref(i)))
        d = {k: getattr(i, k) for k, _ in Info._fields_ if k not in ("grid", "band_kmax")}
        d["grid"] = list(i.grid)
        d["band_kmax"] = list(i.band_kmax)
        return d

    def eval_window(self, z):
        z = np.ascontiguousarray(z, dtype=np.float64)
        W, dW = np.empty_like(z), np.empty_like(z)
        dp = ctypes.POINTER(ctypes.c_double)
        _check(lib().pswf_lr_eval_window(self._h, z.size, z.ctypes.data_as(dp), W.ctypes.data_as(dp),
                                         dW.ctypes.data_as(dp)))
        return W, dW

    def eval_kernel(self, p, k):
        k = np.ascontiguousarray(k, dtype=np.float64)
        out = np.empty_like(k)
        dp = ctypes.POINTER(ctypes.c_double)
        _check(lib().pswf_lr_eval_kernel(self._h, int(p), k.size, k.ctypes.data_as(dp), out.ctypes.data_as(dp)))
        return out

    # -- compute --
    def execute(self, n_atoms, pos, q, E=None, phi=None, F=None, stream=None):
        """Device tensors (torch) in the plan precision; E is a float64 device tensor of 1 element."""
        _check(lib().pswf_lr_execute(self._h, int(n_atoms), _ptr(pos), _ptr(q), _ptr(E), _ptr(phi), _ptr(F),
                                     ctypes.c_void_p(stream or 0)))

    def execute_real(self, n_atoms, pos, q, E=None, phi=None, F=None, accumulate=False, stream=None):
        """Real-space complement - self term (device tensors); accumulate=True adds to E, phi, F."""
        _check(lib().pswf_lr_execute_real(self._h, int(n_atoms), _ptr(pos), _ptr(q), _ptr(E), _ptr(phi), _ptr(F),
                                          1 if accumulate else 0, ctypes.c_void_p(stream or 0)))

    def eval_real(self, p, r):
        r = np.ascontiguousarray(r, dtype=np.float64)
        L, dL = np.empty_like(r), np.empty_like(r)
        dp = ctypes.POINTER(ctypes.c_double)
        _check(lib().pswf_lr_eval_real(self._h, int(p), r.size, r.ctypes.data_as(dp), L.ctypes.data_as(dp),
                                       dL.ctypes.data_as(dp)))
        return L, dL

    def self_coefficient(self, p):
        v = ctypes.c_double(0.0)
        _check(lib().pswf_lr_self_coefficient(self._h, int(p), ctypes.byref(v)))
        return v.value

    def execute_host(self, n_atoms, pos, q, E=None, phi=None, F=None, stream=None):
        """Host buffers (numpy arrays or pinned torch CPU tensors); E: float64 host array of 1."""
        Ep = None
        if E is not None:
            Ep = ctypes.cast(_ptr(E), ctypes.POINTER(ctypes.c_double))
        _check(lib().pswf_lr_execute_host(self._h, int(n_atoms), _ptr(pos), _ptr(q), Ep, _ptr(phi), _ptr(F),
                                          ctypes.c_void_p(stream or 0)))

    def submit_host(self, n_atoms, pos, q, E=None, phi=None, F=None):
        """Pipelined form of execute_host (at most two submissions in flight); see pswf_lr_submit_host."""
        Ep = None
        if E is not None:
            Ep = ctypes.cast(_ptr(E), ctypes.POINTER(ctypes.c_double))
        _check(lib().pswf_lr_submit_host(self._h, int(n_atoms), _ptr(pos), _ptr(q), Ep, _ptr(phi), _ptr(F)))

    def wait_host(self):
        _check(lib().pswf_lr_wait_host(self._h))

    def set_virial(self, enabled):
        _check(lib().pswf_lr_set_virial(self._h, 1 if enabled else 0))

    def virial(self, out, stream=None):
        """out: float64 device tensor of 6 (xx, yy, zz, xy, xz, yz)."""
        _check(lib().pswf_lr_virial(self._h, _ptr(out), ctypes.c_void_p(stream or 0)))

    def channel_energies(self, out, stream=None):
        _check(lib().pswf_lr_channel_energies(self._h, _ptr(out), ctypes.c_void_p(stream or 0)))

    def debug_copy(self, what, dst, stream=None):
        _check(lib().pswf_lr_debug_copy(self._h, int(what), _ptr(dst), ctypes.c_void_p(stream or 0)))

    def debug_cell_starts(self, dst, stream=None):
        _check(lib().pswf_lr_debug_cell_starts(self._h, _ptr(dst), ctypes.c_void_p(stream or 0)))

    def set_profiling(self, enabled):
        _check(lib().pswf_lr_set_profiling(self._h, 1 if enabled else 0))

    def stage_ms(self):
        ms = (ctypes.c_double * N_STAGES)()
        n = ctypes.c_int(0)
        _check(lib().pswf_lr_stage_ms(self._h, ms, ctypes.byref(n)))
        return dict(zip(STAGE_NAMES, list(ms))), n.value
