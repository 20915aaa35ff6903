"""Seeded synthetic workloads: the five BASELINE.json configs with every free choice fixed.

This module is the ONLY code the CUDA path (``paper_1206_0270_b200/csrc``) shares with the CPU checker the
tests compare it with.  It generates *inputs* (grids' parameters, initial
data, sampled particle trajectories with their source amplitudes, observer weights).  It
contains none of the solver's arithmetic: no Lax-Wendroff stage, no Teukolsky coefficient,
no tortoise-coordinate *inversion*, no Gaussian deposit.

Recipe source: SURVEY.md section 8(d) table "Synthetic inputs" and 8(c) readings A1, A7, A9
(reference: PAPER.md:114 Gaussian-smeared source, "trajectory ... generated
separately", PAPER.md:189 production grid).  Seeds: numpy.random.default_rng(12060270 + id).

Textbook Kerr geodesic relations used for the trajectories (Bardeen, Press & Teukolsky 1972):
circular equatorial prograde  Omega = sqrt(M) / (r0^1.5 + a sqrt(M)),
u^t = (1 + a sqrt(M)/r0^1.5) / sqrt(1 - 3M/r0 + 2 a sqrt(M)/r0^1.5).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Sequence

import numpy as np

SEED_BASE = 12060270


@dataclasses.dataclass(frozen=True)
class Config:
    """One workload.  dt is stored as a multiple of dx."""

    cid: int
    name: str
    a: float
    M: float
    modes: Sequence[int]
    rs_min: float
    rs_max: float
    n_r: int
    n_theta: int
    dt_over_dx: float
    steps: int
    observers: Sequence[float]
    initial: str  # "pulse", "random4", "zero"
    source: Optional[str]  # None, "circular", "eccentric", "inspiral"
    outer_bc: int = 0  # 0 = OUTGOING (default), 1 = DIRICHLET

    @property
    def dx(self) -> float:
        return (self.rs_max - self.rs_min) / (self.n_r - 1)

    @property
    def dtheta(self) -> float:
        return math.pi / self.n_theta

    @property
    def dt(self) -> float:
        return self.dt_over_dx * self.dx

    @property
    def n_modes(self) -> int:
        return len(self.modes)

    @property
    def n_pts(self) -> int:
        return self.n_modes * self.n_r * self.n_theta

    def scaled(self, **kw) -> "Config":
        return dataclasses.replace(self, **kw)


CONFIGS: Dict[int, Config] = {
    1: Config(1, "schwarzschild_512x32", 0.0, 1.0, (2,), -50.0, 150.0, 512, 32, 0.04, 2000,
              (30.0,), "pulse", None),
    2: Config(2, "kerr09_4096x64", 0.9, 1.0, (2,), -100.0, 400.0, 4096, 64, 0.05, 20000,
              (300.0, 120.0), "random4", None),
    3: Config(3, "kerr09_circular_16000x64", 0.9, 1.0, (2,), -100.0, 900.0, 16000, 64, 0.1, 100000,
              (800.0, 50.0), "zero", "circular"),
    4: Config(4, "kerr07_modes0to4_eccentric_16000x64", 0.7, 1.0, (0, 1, 2, 3, 4), -100.0, 900.0,
              16000, 64, 0.05, 50000, (50.0,), "zero", "eccentric"),
    5: Config(5, "kerr099_production_131072x128", 0.99, 1.0, (2,), -200.0, 1800.0, 131072, 128,
              0.125, 200000, (1500.0, 50.0), "zero", "inspiral"),
    # Not a BASELINE.json config: the (r, theta) grid of the paper's own Table 1 measurement,
    # 32000 x 304, with config 3's physics.  Exercises the theta-segmented kernel path.
    6: Config(6, "paper_table1_grid_32000x304", 0.9, 1.0, (2,), -100.0, 1900.0, 32000, 304, 0.0125, 20000,
              (50.0,), "zero", "circular"),
}


def grid_axes(cfg: Config):
    """x_i = rs_min + i dx (both end points), theta_j = (j + 1/2) dtheta."""
    x = cfg.rs_min + cfg.dx * np.arange(cfg.n_r, dtype=np.float64)
    theta = (np.arange(cfg.n_theta, dtype=np.float64) + 0.5) * cfg.dtheta
    return x, theta


def initial_data(cfg: Config):
    """Return (phi_re, phi_im, pi_re, pi_im), each [n_modes][n_r][n_theta], C-contiguous.

    Pi(0) = 0 literally.  Gaussian exp(-(x-c)^2/w^2)."""
    x, theta = grid_axes(cfg)
    shape = (cfg.n_modes, cfg.n_r, cfg.n_theta)
    phi = np.zeros(shape, dtype=np.complex128)
    s2 = np.sin(theta) ** 2
    if cfg.initial == "pulse":
        prof = np.exp(-((x - 20.0) ** 2) / 4.0)
        for k in range(cfg.n_modes):
            phi[k] = prof[:, None] * s2[None, :]
    elif cfg.initial == "random4":
        rng = np.random.default_rng(SEED_BASE + cfg.cid)
        c = rng.uniform(0.0, 100.0, 4)
        w = rng.uniform(1.0, 4.0, 4)
        are = rng.standard_normal(4)
        aim = rng.standard_normal(4)
        prof = np.zeros(cfg.n_r, dtype=np.complex128)
        for k in range(4):
            prof += (are[k] + 1j * aim[k]) * np.exp(-((x - c[k]) ** 2) / w[k] ** 2)
        for k in range(cfg.n_modes):
            phi[k] = prof[:, None] * s2[None, :]
    elif cfg.initial == "zero":
        pass
    else:
        raise ValueError(cfg.initial)
    z = np.zeros(shape, dtype=np.float64)
    return (np.ascontiguousarray(phi.real), np.ascontiguousarray(phi.imag), z, z.copy())


def random_state(cfg: Config, seed: int):
    """Seeded smooth-free random state (all four planes non-zero) for one-step parity tests."""
    rng = np.random.default_rng(seed)
    shape = (cfg.n_modes, cfg.n_r, cfg.n_theta)
    return tuple(np.ascontiguousarray(rng.standard_normal(shape)) for _ in range(4))


def observer_weights(cfg: Config):
    """W_j = (1 + cos theta_j)^2 sin theta_j dtheta."""
    _, theta = grid_axes(cfg)
    return np.ascontiguousarray((1.0 + np.cos(theta)) ** 2 * np.sin(theta) * cfg.dtheta)


# ----------------------------------------------------------------------------------------------
# Particle trajectories (workload generation; "trajectory ... generated separately")
# ----------------------------------------------------------------------------------------------

def _horizons(M: float, a: float):
    root = math.sqrt(M * M - a * a)
    return M + root, M - root


def tortoise_forward(r, M: float, a: float):
    """x(r) with the constant of SURVEY.md 8(c) C.1 (forward map only; the solvers invert it
    themselves and a test checks the round trip)."""
    r = np.asarray(r, dtype=np.float64)
    rp, rm = _horizons(M, a)
    cp = 2.0 * M * rp / (rp - rm)
    x = r + cp * np.log((r - rp) / (2.0 * M))
    if a != 0.0:
        cm = 2.0 * M * rm / (rp - rm)
        x = x - cm * np.log((r - rm) / (2.0 * M))
    return x


def azimuth_shift(r, M: float, a: float):
    """phi~ - phi = a/(r+ - r-) ln((r - r+)/(r - r-))  (zero for a = 0)."""
    r = np.asarray(r, dtype=np.float64)
    if a == 0.0:
        return np.zeros_like(r)
    rp, rm = _horizons(M, a)
    return a / (rp - rm) * np.log((r - rp) / (r - rm))


def circular_frequency(r0, M: float, a: float):
    r0 = np.asarray(r0, dtype=np.float64)
    return math.sqrt(M) / (r0 ** 1.5 + a * math.sqrt(M))


def circular_ut(r0, M: float, a: float):
    r0 = np.asarray(r0, dtype=np.float64)
    v = a * math.sqrt(M) / r0 ** 1.5
    return (1.0 + v) / np.sqrt(1.0 - 3.0 * M / r0 + 2.0 * v)


def _eccentric_constants(p: float, e: float, M: float, a: float):
    """E, L_z of the bound equatorial prograde geodesic with turning points pM/(1 +- e):
    Newton on R(r_peri) = R(r_apo) = 0 with
    R(r) = [E(r^2+a^2) - a L]^2 - Delta [r^2 + (L - a E)^2]   (textbook radial potential)."""
    r1, r2 = p * M / (1.0 + e), p * M / (1.0 - e)

    def R(r, E, L):
        D = r * r - 2.0 * M * r + a * a
        return (E * (r * r + a * a) - a * L) ** 2 - D * (r * r + (L - a * E) ** 2)

    # Schwarzschild start
    E = math.sqrt(((p - 2.0) ** 2 - 4.0 * e * e) / (p * (p - 3.0 - e * e)))
    L = p * M / math.sqrt(p - 3.0 - e * e)
    for _ in range(100):
        f = np.array([R(r1, E, L), R(r2, E, L)])
        h = 1e-7
        J = np.array([[(R(r, E + h, L) - R(r, E - h, L)) / (2 * h),
                       (R(r, E, L + h) - R(r, E, L - h)) / (2 * h)] for r in (r1, r2)])
        d = np.linalg.solve(J, f)
        E, L = E - d[0], L - d[1]
        if abs(d[0]) + abs(d[1]) < 1e-15:
            break
    return E, L


def _eccentric_rates(chi, p, e, M, a, E, L):
    """d(chi)/dt, d(phi)/dt, u^t, r at anomaly chi, r = pM/(1 + e cos chi) (equatorial)."""
    r = p * M / (1.0 + e * math.cos(chi))
    D = r * r - 2.0 * M * r + a * a
    P = E * (r * r + a * a) - a * L
    ut = ((r * r + a * a) * P / D - a * (a * E - L)) / (r * r)
    dphi_dtau = (a * P / D - (a * E - L)) / (r * r)
    r3 = 2.0 * M / (1.0 - E * E) - p * M / (1.0 + e) - p * M / (1.0 - e)
    dchi_dtau = math.sqrt((1.0 - E * E) * (r - r3) * (1.0 + e * math.cos(chi)) ** 2
                          / ((1.0 - e * e) * r ** 3))
    return dchi_dtau / ut, dphi_dtau / ut, ut, r


def orbit_table(cfg: Config, n_steps: Optional[int] = None, t0: float = 0.0):
    """Sampled trajectory for teuk_set_source: sample k is at t = t0 + k dt/2, k = 0..2 n_steps.

    Returns a dict with rs_p, theta_p [n_samples]; amp_re, amp_im [n_modes][n_samples];
    sigma_r = 4 dx, sigma_theta = 4 dtheta, half_window = 24, and
    A'_m(t) = (2 mu/u^t) R2_p / (Sigma_p^2 r_p^3 sin theta_p) exp(-i m phi~_p),  mu = 1."""
    if cfg.source is None:
        return None
    n_steps = cfg.steps if n_steps is None else n_steps
    ns = 2 * n_steps + 1
    hdt = 0.5 * cfg.dt
    t = t0 + hdt * np.arange(ns, dtype=np.float64)
    M, a = cfg.M, cfg.a
    if cfg.source == "circular":
        r0 = np.full(ns, 10.0)
        ut = circular_ut(r0, M, a)
        phi = circular_frequency(10.0, M, a) * t
    elif cfg.source == "inspiral":
        T = cfg.steps * cfg.dt  # always the config's full run length, also for short tables
        r0 = 12.0 - 6.0 * t / T
        ut = circular_ut(r0, M, a)
        om = circular_frequency(r0, M, a)
        # phi(t) = int_0^t Omega dt' by Simpson's rule on every sample interval (quadrature,
        # SURVEY.md 8(c) A7), plus one fine Simpson sum over [0, t0] when the table starts late.
        tm = 0.5 * (t[:-1] + t[1:])
        fm = circular_frequency(12.0 - 6.0 * tm / T, M, a)
        seg = hdt / 6.0 * (om[:-1] + 4.0 * fm + om[1:])
        phi = np.concatenate([[0.0], np.cumsum(seg)])
        if t0 != 0.0:
            s = np.linspace(0.0, t0, 2 * 32768 + 1)
            f = circular_frequency(12.0 - 6.0 * s / T, M, a)
            hs = t0 / (2 * 32768)
            phi = phi + hs / 3.0 * (f[0] + f[-1] + 4.0 * f[1:-1:2].sum() + 2.0 * f[2:-1:2].sum())
    elif cfg.source == "eccentric":
        p, e = 8.0, 0.3
        E, L = _eccentric_constants(p, e, M, a)
        r0 = np.zeros(ns)
        ut = np.zeros(ns)
        phi = np.zeros(ns)
        chi, ph = 0.0, 0.0
        if t0 != 0.0:
            raise ValueError("eccentric table starts at t0 = 0")
        for k in range(ns):
            _, _, u, r = _eccentric_rates(chi, p, e, M, a, E, L)
            r0[k], ut[k], phi[k] = r, u, ph
            # RK4 in t with step dt/2 on (chi, phi)
            k1 = _eccentric_rates(chi, p, e, M, a, E, L)
            k2 = _eccentric_rates(chi + 0.5 * hdt * k1[0], p, e, M, a, E, L)
            k3 = _eccentric_rates(chi + 0.5 * hdt * k2[0], p, e, M, a, E, L)
            k4 = _eccentric_rates(chi + hdt * k3[0], p, e, M, a, E, L)
            chi += hdt / 6.0 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0])
            ph += hdt / 6.0 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1])
    else:
        raise ValueError(cfg.source)
    theta_p = np.full(ns, 0.5 * math.pi)
    rp, rm = _horizons(M, a)
    Delta = (r0 - rp) * (r0 - rm)
    R2 = r0 * r0 + a * a
    sn = np.sin(theta_p)
    Sig2 = R2 * R2 - a * a * Delta * sn * sn
    mag = (2.0 / ut) * R2 / (Sig2 * r0 ** 3 * sn)
    phit = phi + azimuth_shift(r0, M, a)
    amp = np.stack([mag * np.exp(-1j * m * phit) for m in cfg.modes])
    return dict(
        rs_p=np.ascontiguousarray(tortoise_forward(r0, M, a)),
        theta_p=np.ascontiguousarray(theta_p),
        amp_re=np.ascontiguousarray(amp.real),
        amp_im=np.ascontiguousarray(amp.imag),
        sigma_r=4.0 * cfg.dx,
        sigma_theta=4.0 * cfg.dtheta,
        half_window=24,
        n_samples=ns,
    )


def small_test_configs() -> List[Config]:
    """Scaled-down variants used by parity tests: several warps/tiles, ragged tails, all features."""
    c1, c3, c4 = CONFIGS[1], CONFIGS[3], CONFIGS[4]
    return [
        c1,
        c1.scaled(name="schw_ragged_301x32", n_r=301),
        CONFIGS[2].scaled(name="kerr09_small_777x64", n_r=777, rs_min=-40.0, rs_max=60.0,
                          observers=(30.0,), steps=300),
        c3.scaled(name="kerr09_circ_small_1203x64", n_r=1203, rs_min=-30.0, rs_max=45.0,
                  observers=(30.0,), steps=300),
        c4.scaled(name="kerr07_modes_small_997x64", n_r=997, rs_min=-30.0, rs_max=32.0,
                  observers=(25.0,), steps=200),
        CONFIGS[5].scaled(name="kerr099_small_1500x128", n_r=1500, rs_min=-20.0, rs_max=40.0,
                          dt_over_dx=0.05, observers=(30.0,), steps=200),
    ]
