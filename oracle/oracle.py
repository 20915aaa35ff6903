"""ctypes wrapper around oracle/liboracle.so (teuk_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It must never be imported by paper_1206_0270_b200 (a test checks that).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

# idle OpenMP threads sleep instead of spinning: on an oversubscribed host (another job on the cores) spinning
# barriers make the row loops of the oracle many times slower
os.environ.setdefault("OMP_WAIT_POLICY", "passive")

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "teuk_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

CXXFLAGS = ["-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-fcx-limited-range",
            "-ffp-contract=off", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no -ffast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++"] + CXXFLAGS + ["-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


# A second build of the SAME source whose only difference is rounding: FMA contraction allowed (the default build
# forbids it).  tests/long_parity.py runs it next to the oracle to measure how far two correct implementations
# of the iteration drift apart on long runs (the oracle-vs-oracle' arm); nothing else uses it.
_LIB_FMA = os.path.join(_HERE, "liboracle_fma.so")
CXXFLAGS_FMA = [f for f in CXXFLAGS if f != "-ffp-contract=off"] + ["-mfma", "-ffp-contract=fast"]


def build_fma(force: bool = False) -> str:
    if force or not os.path.exists(_LIB_FMA) or os.path.getmtime(_LIB_FMA) < os.path.getmtime(_SRC):
        tmp = _LIB_FMA + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++"] + CXXFLAGS_FMA + ["-o", tmp, _SRC])
        os.replace(tmp, _LIB_FMA)
    return _LIB_FMA


_lib = None
_lib_fma = None
_dp = C.POINTER(C.c_double)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def lib_fma():
    """The differently rounded build (see build_fma)."""
    global _lib_fma
    if _lib_fma is None:
        _lib_fma = _declare(C.CDLL(build_fma()))
    return _lib_fma


def lib():
    global _lib
    if _lib is None:
        _lib = _declare(C.CDLL(build()))
    return _lib


def _declare(L):
    if True:
        L.orc_r_of_rstar.argtypes = [C.c_double, C.c_double, C.c_double, _dp, _dp, _dp]
        L.orc_r_of_rstar.restype = None
        L.orc_coefficients.argtypes = [C.c_double, C.c_double, C.c_int, C.c_double, C.c_double, _dp]
        L.orc_coefficients.restype = None
        L.orc_gauss.argtypes = [C.c_double, C.c_double]
        L.orc_gauss.restype = C.c_double
        L.orc_create.argtypes = [C.c_double, C.c_double, C.POINTER(C.c_int32), C.c_int32, C.c_double,
                                 C.c_double, C.c_int32, C.c_int32, C.c_double, C.c_int32]
        L.orc_create.restype = C.c_void_p
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_set_initial.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.orc_set_initial.restype = None
        L.orc_set_source.argtypes = [C.c_void_p, C.c_int64, _dp, _dp, _dp, _dp, C.c_double, C.c_double,
                                     C.c_int32]
        L.orc_set_source.restype = None
        L.orc_add_observer.argtypes = [C.c_void_p, C.c_double, _dp]
        L.orc_add_observer.restype = C.c_int32
        L.orc_step.argtypes = [C.c_void_p, C.c_int64]
        L.orc_step.restype = C.c_int32
        L.orc_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.orc_get_state.restype = None
        L.orc_get_half.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.orc_get_half.restype = None
        L.orc_step_count.argtypes = [C.c_void_p]
        L.orc_step_count.restype = C.c_int64
        L.orc_get_waveform.argtypes = [C.c_void_p, C.c_int32, _dp, _dp, _dp, C.c_int64]
        L.orc_get_waveform.restype = C.c_int64
        L.orc_source_field.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int32, _dp, _dp]
        L.orc_source_field.restype = None
        L.orc_set_source_kind.argtypes = [C.c_void_p, C.c_int32]
        L.orc_set_source_kind.restype = None
        L.orc_delta.argtypes = [C.c_int32, C.c_double, C.c_double]
        L.orc_delta.restype = C.c_double
        _ip = C.POINTER(C.c_int32)
        L.orc_set_source_terms.argtypes = [C.c_void_p, C.c_int32, _ip, _ip, _dp, _dp]
        L.orc_set_source_terms.restype = C.c_int32
        L.orc_profile_deriv.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_double]
        L.orc_profile_deriv.restype = C.c_double
    return L


def r_of_rstar(M, a, x):
    r, d, D = C.c_double(), C.c_double(), C.c_double()
    lib().orc_r_of_rstar(M, a, x, C.byref(r), C.byref(d), C.byref(D))
    return r.value, d.value, D.value


def coefficients(M, a, m, x, theta):
    """dict of b, bx, cL, kappa, alpha, gamma, beta, r, Delta at (x = r*, theta)."""
    out = np.zeros(13)
    lib().orc_coefficients(M, a, int(m), x, theta, _p(out))
    return dict(b=out[0], bx=out[1], cL=out[2], kappa=complex(out[3], out[4]),
                alpha=complex(out[5], out[6]), gamma=complex(out[7], out[8]),
                beta=complex(out[9], out[10]), r=out[11], Delta=out[12])


def gauss(y, sigma):
    return lib().orc_gauss(y, sigma)


def delta(kind, y, h):
    """Discrete delta of kind 1 (two-point) or 2 (four-point) at offset y = x_i - x_p, grid spacing h."""
    return lib().orc_delta(int(kind), float(y), float(h))


def profile_deriv(kind, order, y, width):
    """order-th y-derivative of deposit profile `kind` (0 Gaussian of width sigma, 1 / 2 discrete deltas on spacing h)."""
    return lib().orc_profile_deriv(int(kind), int(order), float(y), float(width))


class OracleSolver:
    """Plain CPU solver.  Arrays are [n_modes][n_r][n_theta] float64, theta fastest."""

    def __init__(self, a, M, modes, rs_min, rs_max, n_r, n_theta, dt, outer_bc=0, library=None):
        self._L = library if library is not None else lib()
        self.modes = list(modes)
        self.shape = (len(self.modes), n_r, n_theta)
        m = (C.c_int32 * len(self.modes))(*self.modes)
        self._h = self._L.orc_create(a, M, m, len(self.modes), rs_min, rs_max, n_r, n_theta, dt, outer_bc)
        if not self._h:
            raise ValueError("orc_create: invalid parameters")
        self.dt = dt
        self._keep = []

    @classmethod
    def from_config(cls, cfg, library=None):
        return cls(cfg.a, cfg.M, cfg.modes, cfg.rs_min, cfg.rs_max, cfg.n_r, cfg.n_theta, cfg.dt,
                   cfg.outer_bc, library=library)

    def close(self):
        if self._h:
            self._L.orc_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    @staticmethod
    def _arr(a, shape):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == tuple(shape), (a.shape, shape)
        return a

    def set_initial(self, phi_re=None, phi_im=None, pi_re=None, pi_im=None):
        arrs = [self._arr(a, self.shape) for a in (phi_re, phi_im, pi_re, pi_im)]
        self._L.orc_set_initial(self._h, *[_p(a) for a in arrs])

    def set_source(self, orbit):
        if orbit is None:
            self._L.orc_set_source(self._h, 0, None, None, None, None, 1.0, 1.0, 0)
            return
        ns = int(orbit["n_samples"])
        xs = self._arr(orbit["rs_p"], (ns,))
        th = self._arr(orbit["theta_p"], (ns,))
        ar = self._arr(orbit["amp_re"], (len(self.modes), ns))
        ai = self._arr(orbit["amp_im"], (len(self.modes), ns))
        self._L.orc_set_source(self._h, ns, _p(xs), _p(th), _p(ar), _p(ai), float(orbit["sigma_r"]),
                             float(orbit["sigma_theta"]), int(orbit["half_window"]))

    def set_source_kind(self, kind):
        """0 Gaussian (default), 1 two-point, 2 four-point discrete delta."""
        if kind not in (0, 1, 2):
            raise ValueError("source kind must be 0, 1 or 2")
        self._L.orc_set_source_kind(self._h, int(kind))

    def set_source_terms(self, terms):
        """f2: `terms` = list of (order_r, order_theta, amp[n_modes][n_samples] complex) replacing the monopole of
        the installed trajectory; an empty list restores it."""
        nt = len(terms)
        orr = (C.c_int32 * max(nt, 1))(*[int(t[0]) for t in terms])
        oth = (C.c_int32 * max(nt, 1))(*[int(t[1]) for t in terms])
        amp = np.ascontiguousarray(np.stack([np.asarray(t[2], dtype=np.complex128) for t in terms])) if nt else \
            np.zeros((0,), dtype=np.complex128)
        ar, ai = np.ascontiguousarray(amp.real), np.ascontiguousarray(amp.imag)
        if self._L.orc_set_source_terms(self._h, nt, orr, oth, _p(ar), _p(ai)) != 0:
            raise ValueError("bad source terms (orders 0..2, a trajectory must be installed first)")

    def add_observer(self, rs_obs, weights=None):
        w = self._arr(weights, (self.shape[2],))
        k = self._L.orc_add_observer(self._h, float(rs_obs), _p(w))
        if k < 0:
            raise ValueError("observer outside the grid")
        return k

    def step(self, n=1):
        if self._L.orc_step(self._h, int(n)) != 0:
            raise ValueError("trajectory table too short")

    @property
    def step_count(self):
        return self._L.orc_step_count(self._h)

    def get_state(self):
        out = [np.empty(self.shape) for _ in range(4)]
        self._L.orc_get_state(self._h, *[_p(a) for a in out])
        return tuple(out)

    def get_half(self):
        shp = (self.shape[0], self.shape[1] - 1, self.shape[2])
        out = [np.empty(shp) for _ in range(4)]
        self._L.orc_get_half(self._h, *[_p(a) for a in out])
        return tuple(out)

    def waveform(self, obs=0):
        """(t[n], w[n][n_modes] complex) recorded so far."""
        n = self._L.orc_get_waveform(self._h, obs, None, None, None, 0)
        t = np.empty(n)
        wr = np.empty((n, self.shape[0]))
        wi = np.empty((n, self.shape[0]))
        self._L.orc_get_waveform(self._h, obs, _p(t), _p(wr), _p(wi), n)
        return t, wr + 1j * wi

    def source_field(self, mode_index, sample, half):
        rows = self.shape[1] - 1 if half else self.shape[1]
        re = np.empty((rows, self.shape[2]))
        im = np.empty((rows, self.shape[2]))
        self._L.orc_source_field(self._h, mode_index, sample, 1 if half else 0, _p(re), _p(im))
        return re + 1j * im
