"""Thin ctypes binding of libteuk.so (include/teuk.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; there is no CPU fallback and this module
imports nothing but the library.  If the shared library is missing or has no CUDA device, calls fail loudly.
PyTorch tensors may be passed wherever a device array is expected (their data_ptr() is used) and
`Solver.use_torch_stream()` makes the solver enqueue on torch's current stream.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libteuk.so")

TEUK_OK, TEUK_EINVAL, TEUK_ENOMEM, TEUK_ECUDA, TEUK_ENONFINITE = 0, -1, -2, -3, -4
SYMBOLS = ["teuk_select_device", "teuk_measure_fp64", "teuk_create", "teuk_set_initial", "teuk_set_source", "teuk_set_source_terms", "teuk_step", "teuk_step_noalloc", "teuk_extract",
           "teuk_get_state", "teuk_set_option", "teuk_get_stat", "teuk_sync", "teuk_destroy",
           "teuk_last_error"]


class TeukError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libteuk error %d: %s" % (code, msg))
        self.code = code


class teuk_grid(C.Structure):
    _fields_ = [("rs_min", C.c_double), ("rs_max", C.c_double), ("n_r", C.c_int32), ("n_theta", C.c_int32)]


_dp = C.POINTER(C.c_double)


class teuk_orbit(C.Structure):
    _fields_ = [("n_samples", C.c_int64), ("rs_p", _dp), ("theta_p", _dp), ("amp_re", _dp), ("amp_im", _dp),
                ("sigma_r", C.c_double), ("sigma_theta", C.c_double), ("half_window", C.c_int32)]


_lib = None


def load():
    """Load libteuk.so (must have been built in-tree by paper_1206_0270_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libteuk.so not built: run `python -m paper_1206_0270_b200.build` "
                          "(the CUDA extension is required; there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.teuk_create.argtypes = [C.POINTER(vp), C.c_double, C.c_double, C.POINTER(C.c_int32), C.c_int32,
                              C.POINTER(teuk_grid), C.c_double]
    L.teuk_select_device.argtypes = [C.c_int32]
    L.teuk_measure_fp64.argtypes = [C.c_int32, _dp]
    L.teuk_set_initial.argtypes = [vp, vp, vp, vp, vp, C.c_int32]
    L.teuk_set_source.argtypes = [vp, C.POINTER(teuk_orbit)]
    _ip = C.POINTER(C.c_int32)
    L.teuk_set_source_terms.argtypes = [vp, C.c_int32, _ip, _ip, _dp, _dp]
    L.teuk_step.argtypes = [vp, C.c_int64]
    L.teuk_step_noalloc.argtypes = [vp, C.POINTER(vp), C.c_int64, C.c_int64, C.POINTER(vp)]
    L.teuk_extract.argtypes = [vp, C.c_double, _dp, _dp, _dp, _dp, C.c_int64, C.POINTER(C.c_int64)]
    L.teuk_get_state.argtypes = [vp, vp, vp, vp, vp, C.c_int32]
    L.teuk_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
    L.teuk_get_stat.argtypes = [vp, C.c_char_p, C.POINTER(C.c_int64)]
    L.teuk_sync.argtypes = [vp]
    L.teuk_destroy.argtypes = [vp]
    L.teuk_destroy.restype = None
    L.teuk_last_error.argtypes = [vp]
    L.teuk_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("teuk_destroy", "teuk_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _ptr(a):
    """Host numpy array, torch tensor (host or device) or None -> (address, is_device)."""
    if a is None:
        return None, None
    if hasattr(a, "data_ptr"):  # torch tensor
        return C.c_void_p(a.data_ptr()), bool(a.is_cuda)
    return C.c_void_p(a.ctypes.data), False


def measure_fp64(kind):
    """teuk_measure_fp64: lane-operations per second of FP64 instruction kind 0..3 on the current device."""
    v = C.c_double(0.0)
    rc = load().teuk_measure_fp64(int(kind), C.byref(v))
    if rc != TEUK_OK:
        raise TeukError(rc, load().teuk_last_error(None).decode())
    return v.value


class Solver:
    """One teuk_solver handle.  Field arrays are [n_modes][n_r][n_theta] float64, theta fastest."""

    def __init__(self, a, M, modes, rs_min, rs_max, n_r, n_theta, dt, device=None):
        """`device`: CUDA device index (default: torch's current device if the caller uses torch, else the device
        current in the thread).  Selecting it calls teuk_select_device, which makes that device current in the
        calling thread for the library's CUDA runtime and leaves it so (like torch.cuda.set_device)."""
        self._lib = load()
        if device is None:
            import sys
            torch = sys.modules.get("torch")      # only if the caller already uses torch
            if torch is not None and torch.cuda.is_available() and torch.cuda.is_initialized():
                device = torch.cuda.current_device()
        if device is not None:
            rc = self._lib.teuk_select_device(int(device))
            if rc != TEUK_OK:
                raise TeukError(rc, self._lib.teuk_last_error(None).decode())
        self.modes = [int(m) for m in modes]
        self.shape = (len(self.modes), int(n_r), int(n_theta))
        self.dt = float(dt)
        self._h = C.c_void_p()
        m = (C.c_int32 * len(self.modes))(*self.modes)
        g = teuk_grid(float(rs_min), float(rs_max), int(n_r), int(n_theta))
        rc = self._lib.teuk_create(C.byref(self._h), float(a), float(M), m, len(self.modes), C.byref(g), self.dt)
        if rc != TEUK_OK:
            raise TeukError(rc, self._lib.teuk_last_error(None).decode())

    @classmethod
    def from_config(cls, cfg):
        s = cls(cfg.a, cfg.M, cfg.modes, cfg.rs_min, cfg.rs_max, cfg.n_r, cfg.n_theta, cfg.dt)
        if cfg.outer_bc:
            s.set_option("outer_bc", cfg.outer_bc)
        return s

    def _check(self, rc):
        if rc != TEUK_OK:
            raise TeukError(rc, self._lib.teuk_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.teuk_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _fields(self, arrs, output=False):
        ptrs, dev = [], None
        for a in arrs:
            if a is not None and not hasattr(a, "data_ptr"):
                if output:      # the library writes through the pointer: a hidden copy would be filled instead
                    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous
                            and a.flags.writeable):
                        raise TypeError("output arrays must be writeable C-contiguous float64 numpy arrays")
                else:
                    a = np.ascontiguousarray(a, dtype=np.float64)
                assert a.shape == self.shape, (a.shape, self.shape)
            elif a is not None:
                assert tuple(a.shape) == self.shape and a.is_contiguous() and a.element_size() == 8
            p, d = _ptr(a)
            if d is not None:
                assert dev is None or dev == d, "mix of host and device arrays"
                dev = d
            ptrs.append((p, a))
        return ptrs, bool(dev)

    def set_initial(self, phi_re=None, phi_im=None, pi_re=None, pi_im=None):
        ptrs, dev = self._fields([phi_re, phi_im, pi_re, pi_im])
        self._check(self._lib.teuk_set_initial(self._h, *[p for p, _ in ptrs], 1 if dev else 0))

    def set_source(self, orbit):
        if orbit is None:
            self._check(self._lib.teuk_set_source(self._h, None))
            return
        ns = int(orbit["n_samples"])
        keep = [np.ascontiguousarray(orbit[k], dtype=np.float64) for k in ("rs_p", "theta_p", "amp_re", "amp_im")]
        assert keep[0].shape == (ns,) and keep[2].shape == (self.shape[0], ns)
        o = teuk_orbit(ns, *[k.ctypes.data_as(_dp) for k in keep], float(orbit["sigma_r"]),
                       float(orbit["sigma_theta"]), int(orbit["half_window"]))
        self._check(self._lib.teuk_set_source(self._h, C.byref(o)))

    def set_source_terms(self, terms):
        """teuk_set_source_terms: `terms` = list of (order_r, order_theta, amp[n_modes][n_samples] complex); an empty
        list restores the single term of the trajectory table."""
        nt = len(terms)
        if nt == 0:
            self._check(self._lib.teuk_set_source_terms(self._h, 0, None, None, None, None))
            return
        orr = (C.c_int32 * nt)(*[int(t[0]) for t in terms])
        oth = (C.c_int32 * nt)(*[int(t[1]) for t in terms])
        amp = np.stack([np.asarray(t[2], dtype=np.complex128) for t in terms])
        assert amp.ndim == 3 and amp.shape[1] == self.shape[0], amp.shape
        ar, ai = np.ascontiguousarray(amp.real), np.ascontiguousarray(amp.imag)
        self._check(self._lib.teuk_set_source_terms(self._h, nt, orr, oth, ar.ctypes.data_as(_dp),
                                                    ai.ctypes.data_as(_dp)))

    def step(self, n=1):
        self._check(self._lib.teuk_step(self._h, int(n)))

    def step_noalloc(self, fields_in, n0, n, fields_out):
        """teuk_step_noalloc: advance the 4 DEVICE tensors `fields_in` (level n0; None = zeros) by n iterations into
        the 4 device tensors `fields_out` (None = skip) with the resident kernel, allocating nothing."""
        def pack(arrs):
            a4 = (C.c_void_p * 4)()
            for k, a in enumerate(arrs):
                if a is None:
                    a4[k] = None
                    continue
                assert hasattr(a, "data_ptr") and a.is_cuda, "teuk_step_noalloc takes device tensors"
                assert tuple(a.shape) == self.shape and a.is_contiguous() and a.element_size() == 8
                a4[k] = a.data_ptr()
            return a4
        self._check(self._lib.teuk_step_noalloc(self._h, pack(fields_in), int(n0), int(n), pack(fields_out)))

    def add_observer(self, rs_obs, weights=None):
        """First teuk_extract call with a new rs_obs: arms the observer."""
        w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float64)
        n = C.c_int64(0)
        self._check(self._lib.teuk_extract(self._h, float(rs_obs), None if w is None else w.ctypes.data_as(_dp),
                                           None, None, None, 0, C.byref(n)))

    def extract(self, rs_obs, capacity=None, allow_nonfinite=False):
        """Samples recorded since the previous call: (t[k], w[k][n_modes] complex)."""
        cap = int(capacity) if capacity is not None else int(self.stat("steps")) + 1
        t = np.empty(cap)
        wr = np.empty((cap, self.shape[0]))
        wi = np.empty((cap, self.shape[0]))
        n = C.c_int64(0)
        rc = self._lib.teuk_extract(self._h, float(rs_obs), None, t.ctypes.data_as(_dp), wr.ctypes.data_as(_dp),
                                    wi.ctypes.data_as(_dp), cap, C.byref(n))
        if not (allow_nonfinite and rc == TEUK_ENONFINITE):
            self._check(rc)
        k = n.value
        return t[:k].copy(), (wr[:k] + 1j * wi[:k])

    def get_state(self, out=None):
        """Host copy of (phi_re, phi_im, pi_re, pi_im); or fill 4 given arrays/tensors."""
        if out is None:
            out = [np.empty(self.shape) for _ in range(4)]
        ptrs, dev = self._fields(list(out), output=True)
        self._check(self._lib.teuk_get_state(self._h, *[p for p, _ in ptrs], 1 if dev else 0))
        return tuple(out)

    def set_option(self, key, value):
        self._check(self._lib.teuk_set_option(self._h, key.encode(), int(value)))

    def use_torch_stream(self):
        import torch
        self.set_option("stream", torch.cuda.current_stream().cuda_stream)

    def stat(self, key):
        v = C.c_int64(0)
        self._check(self._lib.teuk_get_stat(self._h, key.encode(), C.byref(v)))
        return v.value

    def sync(self):
        self._check(self._lib.teuk_sync(self._h))
