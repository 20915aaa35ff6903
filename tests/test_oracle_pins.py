"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU needed).

The paper prints no field values, so the oracle is pinned by:
  P1  computer-algebra substitution of Psi = e^{im phi~} r^3 Phi into PAPER.md:68-76 (Eq. 1),
      done here with sympy, plus the stored Table C values and the tortoise inversion;
  P2  second-order self-convergence (PAPER.md:88 "second-order Lax-Wendroff", :102);
  P3  Schwarzschild l = 2 quasinormal frequency 0.3737 - 0.0890i (BASELINE.json north_star),
      for even and odd m (both pole-parity branches of PAPER.md:104);
  P3b Kerr a = 0.9, l = m = 2: 0.6716 - 0.0649i (textbook, Berti et al. tables);
  P4  (m, theta) -> (-m, pi - theta) reflection with complex conjugation;
  P5  a = 0 keeps real data exactly real;
  P6  linearity / exact power-of-two scaling / zero stays zero;
  P7  unit norm, support and time-level placement of the Gaussian deposit;
  P8  closed forms of the radial edge rows, domain of dependence;
  P9  discrete-delta deposits: the step-function construction in exact rationals, moment
      conditions with their known remainders, cubic interpolation, mass / centre / support of the 2D deposit.
"""
import math
import os

import numpy as np
import pytest

from paper_1206_0270_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------ P1
def _table_c():
    rows = []
    for line in open(os.path.join(GOLDEN, "table_c.txt")):
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split("|")
        a, m, r, th = left.split()
        v = [float(t) for t in right.split()]
        rows.append((float(a), int(m), float(r), float(th), v))
    return rows


def test_p1_table_c(orc):
    """Stored CAS values of Eq. (1)'s reduction (SURVEY.md 8(c) Table C)."""
    for a, m, r, th, v in _table_c():
        c = orc.coefficients(1.0, a, m, v[0], th)
        got = [c["b"], c["bx"], c["kappa"].real, c["kappa"].imag, c["alpha"].real, c["alpha"].imag,
               c["gamma"].real, c["gamma"].imag, c["cL"]]
        assert abs(c["r"] - r) < 1e-12 * r
        for g, e in zip(got, v[1:]):
            assert abs(g - e) <= 5e-13 * max(1.0, abs(e)) and abs(g - e) <= 2e-11 * max(abs(e), 1e-3), (a, m, r, g, e)


@pytest.mark.parametrize("a_num,a_den,m,r_val,th_val", [
    (9, 10, 2, "3", "1.0471975511965976"),
    (99, 100, 2, "3/2", "1/10"),
    (7, 10, 4, "10", "3"),
    (0, 1, 2, "3", "1.5707963267948966"),
    (9, 10, -3, "2.2", "2.5"),
    (99, 100, 1, "1.1510", "0.7"),   # close to the horizon r+ = 1.14107
    (7, 10, 0, "40", "1.2"),
])
def test_p1_cas_substitution(orc, a_num, a_den, m, r_val, th_val):
    """Brute force: apply the operator of PAPER.md:68-76 (Eq. 1) to
    Psi = e^{i m phi~(r)} r^3 F(t, x(r), theta) for seven monomial F with sympy and read off every
    coefficient of  F_tt = b^2 F_xx + beta F_x + alpha F_t + gamma F + cL (F_thth + cot F_th)."""
    sp = pytest.importorskip("sympy")
    t, r, th, ph, X = sp.symbols("t r theta phi X", real=True)
    M = sp.Integer(1)
    a = sp.Rational(a_num, a_den)
    s = -2
    rp = M + sp.sqrt(M * M - a * a)
    rm = M - sp.sqrt(M * M - a * a)
    Delta = r * r - 2 * M * r + a * a
    R2 = r * r + a * a
    Sig2 = R2 ** 2 - a * a * Delta * sp.sin(th) ** 2
    xr = r + 2 * M * rp / (rp - rm) * sp.log((r - rp) / (2 * M))
    pht = ph
    if a != 0:
        xr = xr - 2 * M * rm / (rp - rm) * sp.log((r - rm) / (2 * M))
        pht = ph + a / (rp - rm) * sp.log((r - rp) / (r - rm))
    point = {r: sp.Rational(r_val) if "/" in r_val else sp.Float(r_val, 40),
             th: sp.Rational(th_val) if "/" in th_val else sp.Float(th_val, 40),
             t: sp.Rational(7, 10), ph: sp.Rational(3, 10)}

    def eq1_lhs(Psi):
        sn, cs = sp.sin(th), sp.cos(th)
        return (-(R2 ** 2 / Delta - a * a * sn ** 2) * sp.diff(Psi, t, 2)
                - 4 * M * a * r / Delta * sp.diff(Psi, t, ph)
                - 2 * s * (r - M * (r * r - a * a) / Delta + sp.I * a * cs) * sp.diff(Psi, t)
                + Delta ** (-s) * sp.diff(Delta ** (s + 1) * sp.diff(Psi, r), r)
                + sp.diff(sn * sp.diff(Psi, th), th) / sn
                + (1 / sn ** 2 - a * a / Delta) * sp.diff(Psi, ph, 2)
                + 2 * s * (a * (r - M) / Delta + sp.I * cs / sn ** 2) * sp.diff(Psi, ph)
                - (s * s * cs ** 2 / sn ** 2 - s) * Psi)

    def reduced(F):  # value of [F_tt - (b^2 F_xx + ...)] implied by Eq. (1)
        Psi = sp.exp(sp.I * m * pht) * r ** 3 * F.subs(X, xr)
        v = eq1_lhs(Psi) / (-(Sig2 / Delta) * r ** 3 * sp.exp(sp.I * m * pht))
        return complex(sp.N(v.subs(point), 30))

    tv = float(point[t])
    thv = float(point[th])
    xv = float(sp.N(xr.subs(point), 30))
    v1 = reduced(sp.Integer(1) + 0 * X)
    gamma = -v1
    alpha = -reduced(t + 0 * X) - gamma * tv
    norm = reduced(t * t / 2 + 0 * X) + alpha * tv + gamma * tv * tv / 2
    beta = -reduced(X) - gamma * xv
    b2 = -reduced(X * X / 2) - beta * xv - gamma * xv * xv / 2
    cot_term = -reduced(th + 0 * X) - gamma * thv           # = cL cot(theta)
    cL_a = (-reduced(th * th / 2 + 0 * X) - gamma * thv * thv / 2) / (1 + thv / math.tan(thv))
    b_sym = R2 / sp.sqrt(Sig2)
    bx = float(sp.N((Delta / R2 * sp.diff(b_sym, r)).subs(point), 30))
    assert abs(norm - 1) < 1e-13            # the F_tt coefficient of Eq. (1) is -Sigma^2/Delta
    assert abs(b2.imag) < 1e-13 and abs(cot_term - cL_a / math.tan(thv)) < 1e-12 * abs(cL_a) + 1e-15

    c = orc.coefficients(1.0, float(a), m, xv, thv)

    def close(got, exp, what):
        tol = 2e-11 * max(abs(exp), 1e-3)
        assert abs(got - exp) <= tol, (what, got, exp)

    close(c["r"], float(point[r]), "r(x)")
    close(c["b"] ** 2, b2.real, "b^2")
    close(c["cL"], cL_a.real, "cL")
    close(c["alpha"], alpha, "alpha")
    close(c["beta"], beta, "beta")
    close(c["gamma"], gamma, "gamma")
    close(c["bx"], bx, "b_x")
    b = math.sqrt(b2.real)
    close(c["kappa"], beta - alpha * b - b * bx, "kappa = beta - alpha b - b b_x")


@pytest.mark.parametrize("a", [0.0, 0.7, 0.9, 0.99])
def test_p1_tortoise_inversion(orc, a):
    """r(x) against a 40-digit root of the closed-form tortoise map; Delta from delta = r - r+
    stays accurate where r - r+ is far below one ulp of r."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 60
    M = mp.mpf(1)
    am = mp.mpf(a)
    rp = M + mp.sqrt(M * M - am * am)
    rm = M - mp.sqrt(M * M - am * am)
    cp = 2 * M * rp / (rp - rm)
    cm = 2 * M * rm / (rp - rm)
    for x in [-200.0, -100.0, -50.0, -20.0, -5.0, 0.0, 1.93503434588429, 7.5, 50.0, 400.0, 1800.0]:
        # unknown y = ln(r - r+), exact in multiprecision
        f = lambda y: rp + mp.e ** y + cp * (y - mp.log(2 * M)) - (cm * mp.log((mp.e ** y + rp - rm) / (2 * M)) if a else 0) - x
        y0 = (mp.mpf(x) - rp) / cp + mp.log(2 * M) if x < 2 * float(rp) else mp.log(x)
        y = mp.findroot(f, y0)
        d = mp.e ** y
        r_ref, D_ref = rp + d, d * (d + rp - rm)
        r, delta, Delta = orc.r_of_rstar(1.0, a, x)
        assert abs(r - float(r_ref)) <= 4e-15 * float(r_ref) + 1e-13 * (x > 100)
        assert abs(delta - float(d)) <= 1e-12 * float(d)
        assert abs(Delta - float(D_ref)) <= 1e-12 * float(D_ref)
    if a == 0.0:  # textbook Schwarzschild closed form x = r + 2M ln(r/2M - 1)
        for rr in [2.0001, 2.5, 3.0, 10.0, 100.0]:
            x = rr + 2.0 * math.log(rr / 2.0 - 1.0)
            assert abs(orc.r_of_rstar(1.0, 0.0, x)[0] - rr) < 1e-13 * rr


def test_p1_workload_tortoise_roundtrip(orc):
    """The trajectory generator's forward map and the oracle's inversion are written separately."""
    for a in [0.0, 0.7, 0.99]:
        for rr in [1.5 + 0.7 * (a < 0.9) + 0.6 * (a == 0.0), 6.0, 10.0, 12.0]:
            x = float(wl.tortoise_forward(rr, 1.0, a))
            assert abs(orc.r_of_rstar(1.0, a, x)[0] - rr) < 1e-13 * rr


# ------------------------------------------------------------------------------------ helpers
def _pulse_run(orc, n_r, n_theta, a, m, cfl, T, shape, x_obs=50.0, rs=(-50.0, 150.0)):
    dx = (rs[1] - rs[0]) / (n_r - 1)
    dt = cfl * dx
    o = orc.OracleSolver(a, 1.0, [m], rs[0], rs[1], n_r, n_theta, dt)
    x = rs[0] + dx * np.arange(n_r)
    th = (np.arange(n_theta) + 0.5) * math.pi / n_theta
    ang = {"sin2": np.sin(th) ** 2, "y22": (1 + np.cos(th)) ** 2, "y21": np.sin(th) * (1 + np.cos(th)),
           "y20": np.sin(th) ** 2}[shape]
    o.set_initial(np.ascontiguousarray((np.exp(-(x - 20.0) ** 2 / 4.0)[:, None] * ang[None, :])[None]))
    harm = {0: np.sin(th) ** 2, 1: np.sin(th) * (1 + np.cos(th)), 2: (1 + np.cos(th)) ** 2}[abs(m)]
    o.add_observer(x_obs, harm * np.sin(th) * math.pi / n_theta)
    o.step(int(round(T / dt)))
    t, w = o.waveform()
    o.close()
    return t, w[:, 0]


def _prony(t, w, t0, t1, n_poles):
    """Linear-prediction fit  w(t) = sum_k c_k exp(-i omega_k t)  on [t0, t1]; returns omega_k."""
    sel = (t >= t0) & (t <= t1)
    tt, ww = t[sel], w[sel]
    stride = max(1, int(round(1.0 / (tt[1] - tt[0]))))
    ww = ww[::stride]
    h = (tt[1] - tt[0]) * stride
    N, p = len(ww), n_poles
    A = np.stack([ww[k:N - p + k] for k in range(p)], axis=1)
    c = np.linalg.lstsq(A, ww[p:], rcond=None)[0]
    z = np.roots(np.concatenate([[1.0], -c[::-1]]))
    return 1j * np.log(z) / h


# ------------------------------------------------------------------------------------------ P2
def test_p2_second_order_convergence(orc):
    """Halving (dx, dtheta, dt) twice divides the waveform error by 4."""
    runs = []
    for k in (1, 2, 4):
        t, w = _pulse_run(orc, 384 * k + 1, 12 * k, 0.0, 2, 0.08, 120.0, "sin2")
        runs.append((t[k - 1::k], w[k - 1::k]))
    n = min(len(r[0]) for r in runs)
    tc = runs[0][0][:n]
    assert np.allclose(tc, runs[1][0][:n]) and np.allclose(tc, runs[2][0][:n])
    wc, wm, wf = [r[1][:n] for r in runs]
    sel = (tc >= 40.0) & (tc <= 120.0)
    ratio = np.linalg.norm(wc[sel] - wm[sel]) / np.linalg.norm(wm[sel] - wf[sel])
    assert np.linalg.norm(wf[sel]) > 10.0
    assert 3.5 < ratio < 5.0, ratio


# ------------------------------------------------------------------------------------------ P3
@pytest.mark.parametrize("m,shape", [(2, "y22"), (1, "y21"), (2, "sin2"), (0, "y20")])
def test_p3_schwarzschild_qnm(orc, m, shape):
    """Ringdown frequency M omega = 0.3737 - 0.0890i, independent of m for a = 0."""
    t, w = _pulse_run(orc, 1025, 32, 0.0, m, 0.08, 170.0, shape)
    assert np.all(w.imag == 0.0)
    om = _prony(t, w.real, 110.0, 170.0, 2)
    om = om[np.argmax(om.real)]
    assert abs(om - (0.3737 - 0.0890j)) < 1.5e-3, om


def test_p3b_kerr_qnm(orc):
    """Kerr a = 0.9, l = m = 2 fundamental mode M omega = 0.6716 - 0.0649i: pins every a != 0 term."""
    t, w = _pulse_run(orc, 1537, 24, 0.9, 2, 0.16, 200.0, "y22")
    for (t0, t1) in [(110.0, 190.0), (100.0, 160.0)]:
        om = _prony(t, w, t0, t1, 6)
        om = om[np.argmin(abs(om - (0.6716 - 0.0649j)))]
        assert abs(om - (0.6716 - 0.0649j)) < 4e-3, om


# ------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("m", [2, 1])
def test_p4_reflection_invariant(orc, m):
    """Phi_{-m}(x, pi - theta) = conj Phi_{+m}(x, theta) for data related the same way."""
    n_r, n_th, a = 257, 16, 0.9
    rs = (-30.0, 70.0)
    dx = (rs[1] - rs[0]) / (n_r - 1)
    x = rs[0] + dx * np.arange(n_r)
    th = (np.arange(n_th) + 0.5) * math.pi / n_th
    f = (np.exp(-(x - 15.0) ** 2 / 9.0) * np.exp(0.7j * x))[:, None] * (np.sin(th) ** 2 * (1.3 + np.cos(th)) * np.exp(0.4j * th))[None, :]
    g = 0.3 * (np.exp(-(x - 5.0) ** 2 / 4.0))[:, None] * (np.sin(th) ** 2 * np.exp(-0.2j * th))[None, :]
    outs = []
    for sign in (+1, -1):
        o = orc.OracleSolver(a, 1.0, [sign * m], rs[0], rs[1], n_r, n_th, 0.1 * dx)
        ff, gg = (f, g) if sign > 0 else (np.conj(f[:, ::-1]), np.conj(g[:, ::-1]))
        o.set_initial(*[np.ascontiguousarray(q[None]) for q in (ff.real, ff.imag, gg.real, gg.imag)])
        o.step(600)
        s = o.get_state()
        outs.append((s[0][0] + 1j * s[1][0], s[2][0] + 1j * s[3][0]))
        o.close()
    for q in (0, 1):
        ref = outs[0][q]
        err = np.linalg.norm(outs[1][q][:, ::-1] - np.conj(ref)) / np.linalg.norm(ref)
        assert err < 1e-12, err
    # and the symmetry is not vacuous: +m and -m differ without the reflection
    assert np.linalg.norm(outs[1][0] - outs[0][0]) > 1e-3 * np.linalg.norm(outs[0][0])


# ------------------------------------------------------------------------------------------ P5
def test_p5_schwarzschild_stays_real(orc):
    cfg = wl.CONFIGS[1]
    o = orc.OracleSolver.from_config(cfg)
    o.set_initial(*wl.initial_data(cfg))
    o.step(300)
    s = o.get_state()
    assert np.all(s[1] == 0.0) and np.all(s[3] == 0.0)
    assert np.abs(s[0]).max() > 0.1 and np.abs(s[2]).max() > 0.01


# ------------------------------------------------------------------------------------------ P6
def _small_sourced(orc, scale=1.0, initial=None, source=True):
    cfg = wl.small_test_configs()[3].scaled(n_r=301, steps=60)
    o = orc.OracleSolver.from_config(cfg)
    if initial is not None:
        o.set_initial(*initial)
    if source:
        orb = wl.orbit_table(cfg)
        orb["amp_re"] = orb["amp_re"] * scale
        orb["amp_im"] = orb["amp_im"] * scale
        o.set_source(orb)
    o.add_observer(30.0, wl.observer_weights(cfg))
    o.step(60)
    return cfg, o.get_state(), o.waveform()[1]


def test_p6_linearity(orc):
    cfg, s1, w1 = _small_sourced(orc, 1.0)
    _, s2, w2 = _small_sourced(orc, 2.0)
    assert max(np.abs(q).max() for q in s1) > 0.0
    for q1, q2 in zip(s1, s2):
        assert np.array_equal(2.0 * q1, q2)          # scaling by 2 is exact in binary FP
    assert np.array_equal(2.0 * w1, w2)
    _, s0, _ = _small_sourced(orc, source=False)
    assert all(np.all(q == 0.0) for q in s0)         # zero data, no source: stays zero
    ini = wl.random_state(cfg, 7)
    _, sa, _ = _small_sourced(orc, initial=ini, source=False)
    _, sb, _ = _small_sourced(orc, initial=ini, source=True)
    for qa, qb, q1 in zip(sa, sb, s1):               # superposition of data and source responses
        assert np.linalg.norm(qb - qa - q1) <= 1e-12 * np.linalg.norm(qb)


# ------------------------------------------------------------------------------------------ P7
def test_p7_source_norm_support_and_time_levels(orc):
    cfg = wl.small_test_configs()[3].scaled(n_r=401)
    orb = wl.orbit_table(cfg, n_steps=4)
    orb["amp_re"] = np.ones_like(orb["amp_re"])
    orb["amp_im"] = np.zeros_like(orb["amp_im"])
    o = orc.OracleSolver.from_config(cfg)
    o.set_source(orb)
    x, th = wl.grid_axes(cfg)
    for half in (False, True):
        T = o.source_field(0, 0, half)
        assert abs(T.real.sum() * cfg.dx * cfg.dtheta - 1.0) < 1e-8       # unit mass
        assert np.all(T.imag == 0.0)
        nz = np.argwhere(T.real != 0.0)
        assert nz[:, 0].max() - nz[:, 0].min() == 48 and nz[:, 1].max() - nz[:, 1].min() == 48
        xs = (x[:-1] + 0.5 * cfg.dx) if half else x
        i_pk, j_pk = np.unravel_index(np.argmax(T.real), T.shape)
        assert abs(xs[i_pk] - orb["rs_p"][0]) <= 0.5 * cfg.dx + 1e-12
        assert abs(th[j_pk] - orb["theta_p"][0]) <= 0.5 * cfg.dtheta + 1e-12
        # first moment = particle position (Gaussian centred on the particle, not on a cell)
        assert abs((T.real * xs[:, None]).sum() * cfg.dx * cfg.dtheta - orb["rs_p"][0]) < 1e-6
    # closed form of the first iteration from zero data: the half step sees sample 0 at the
    # half points, the full step sees sample 1 at the nodes (C.5, C.6).
    for k_on in (0, 1):
        o2 = orc.OracleSolver.from_config(cfg)
        ob = dict(orb)
        ob["amp_re"] = np.zeros_like(orb["amp_re"])
        ob["amp_re"][:, k_on] = 1.0
        o2.set_source(ob)
        o2.step(1)
        phi_re, phi_im, pi_re, pi_im = o2.get_state()
        hs = o2.get_half()
        if k_on == 0:
            Th = o.source_field(0, 0, True)
            assert np.allclose(hs[2][0], 0.5 * cfg.dt * Th.real, rtol=1e-14, atol=0)
            assert np.all(hs[0] == 0.0)
            exp_phi = cfg.dt * 0.5 * (hs[2][0][1:] + hs[2][0][:-1])          # Phi^1 = dt * Pi~
            assert np.allclose(phi_re[0][1:-1], exp_phi, rtol=1e-13, atol=1e-300)
        else:
            Tn = o.source_field(0, 1, False)
            assert np.all(hs[2] == 0.0) and np.all(phi_re == 0.0)
            assert np.allclose(pi_re[0][1:-1], cfg.dt * Tn.real[1:-1], rtol=1e-14, atol=0)
        o2.close()


# ------------------------------------------------------------------------------------------ P8
def test_p8_outer_edge_branches_and_domain_of_dependence(orc):
    """Radial edge conditions.  One iteration moves information by one row, so after n
    iterations the two outer-edge branches (Dirichlet as printed / outgoing, reading A6) may differ only in
    the last n+1 rows, bit for bit elsewhere; the Dirichlet edge rows are exactly zero; with b = 1 (a = 0)
    the outgoing edge advects Phi outwards: Phi' = Phi - dt (Phi_N - Phi_{N-1})/dx."""
    cfg = wl.CONFIGS[1].scaled(name="edge", n_r=80, rs_min=40.0, rs_max=40.0 + 79 * 0.4, steps=12)
    ini = wl.random_state(cfg, 3)
    n = 12
    out = []
    for bc in (0, 1):
        o = orc.OracleSolver.from_config(cfg.scaled(outer_bc=bc))
        o.set_initial(*ini)
        o.step(1)
        first = o.get_state()
        o.step(n - 1)
        out.append((first, o.get_state()))
        o.close()
    (f0, s0), (f1, s1) = out
    for a, b in zip(s0, s1):
        assert np.array_equal(a[:, : cfg.n_r - n - 1], b[:, : cfg.n_r - n - 1])
        assert not np.array_equal(a[:, -n:], b[:, -n:])
    for q in range(4):
        assert np.all(f1[q][:, 0] == 0.0) and np.all(f1[q][:, -1] == 0.0)      # Dirichlet: both edges
        assert np.all(f0[q][:, 0] == 0.0)                                      # inner edge always
    assert np.all(f0[2][:, -1] == 0.0) and np.all(f0[3][:, -1] == 0.0)         # outgoing: Pi = 0
    for q in (0, 1):                                                           # a = 0: b = 1 exactly
        exp = ini[q][:, -1] - cfg.dt * 1.0 * (ini[q][:, -1] - ini[q][:, -2]) / cfg.dx
        assert np.allclose(f0[q][:, -1], exp, rtol=1e-14, atol=1e-15)


# ------------------------------------------------------------------------------------------ P9
def test_p9_discrete_delta_is_the_difference_of_a_discrete_step(orc):
    """"define a step function on a discrete grid and apply the finite-difference derivative".
    Done literally in exact rational arithmetic: ramp -> (first difference) discrete step -> (difference)
    discrete delta; the oracle's closed form must reproduce it."""
    from fractions import Fraction as Fr
    h = Fr(1, 8)
    for xp in (Fr(37, 64), Fr(5, 8), Fr(-3, 16) + Fr(1, 1024), Fr(99, 128)):
        xs = [Fr(i) * h for i in range(-12, 13)]
        ramp = [max(x - xp, Fr(0)) for x in xs]
        step = [(ramp[i + 1] - ramp[i]) / h for i in range(len(xs) - 1)]            # H_{i+1/2}
        assert all(0 <= v <= 1 for v in step) and step[0] == 0 and step[-1] == 1
        assert sum(1 for v in step if 0 < v < 1) <= 1                                # one partial cell
        delta = [(step[i] - step[i - 1]) / h for i in range(1, len(step))]           # at xs[1:-1]
        for x, d in zip(xs[1:-1], delta):
            got = orc.delta(1, float(x - xp), float(h))
            assert got == float(d), (xp, x, got, d)                                  # dyadic inputs: exact
        assert sum(delta) * h == 1
        assert sum(d * x for d, x in zip(delta, xs[1:-1])) * h == xp


@pytest.mark.parametrize("kind,order", [(1, 1), (2, 3)])
def test_p9_discrete_delta_moments(orc, kind, order):
    """sum_i d_i (x_i - x_p)^k h = delta_{k0} up to the order of the rule; the next moment is the known
    non-zero remainder (so a wrong support, sign or a dropped factor fails)."""
    rng = np.random.default_rng(909 + kind)
    for _ in range(20):
        h = rng.uniform(0.01, 2.0)
        xp = rng.uniform(-3.0, 3.0)
        k0 = math.floor(xp / h)
        g = xp / h - k0
        xs = (k0 + np.arange(-4, 6)) * h
        d = np.array([orc.delta(kind, x - xp, h) for x in xs])
        assert np.count_nonzero(d) <= 2 * kind
        for k in range(order + 1):
            mom = np.sum(d * (xs - xp) ** k) * h
            assert abs(mom - (1.0 if k == 0 else 0.0)) < 1e-12 * max(1.0, h ** k), (kind, k, mom)
        nxt = np.sum(d * (xs - xp) ** (order + 1)) * h
        if kind == 1:
            exp = g * (1 - g) * h * h                                 # linear interpolation remainder
        else:
            exp = -(g + 1) * g * (g - 1) * (g - 2) * h ** 4          # cubic Lagrange remainder of y^4
        assert abs(nxt - exp) < 1e-11 * max(1.0, h ** 4), (kind, nxt, exp)


def test_p9_four_point_delta_is_cubic_interpolation(orc):
    rng = np.random.default_rng(9092)
    h = 0.37
    for _ in range(10):
        xp = rng.uniform(-1, 1)
        k0 = math.floor(xp / h)
        xs = (k0 + np.arange(-1, 3)) * h                              # the four nodes around x_p
        f = rng.normal(size=4)
        lagr = np.polyval(np.polyfit(xs, f, 3), xp)                   # library cubic through the nodes
        got = sum(orc.delta(2, x - xp, h) * fv for x, fv in zip(xs, f)) * h
        assert abs(got - lagr) < 1e-11


@pytest.mark.parametrize("kind", [1, 2])
def test_p9_discrete_delta_deposit(orc, kind):
    """The 2D deposit: mass A', centred on the particle, support 2x2 / 4x4 points, on both stage grids."""
    cfg = wl.small_test_configs()[3].scaled(n_r=401)
    orb = wl.orbit_table(cfg, n_steps=4)
    orb["amp_re"] = np.full_like(orb["amp_re"], 1.5)
    orb["amp_im"] = np.full_like(orb["amp_im"], -0.5)
    o = orc.OracleSolver.from_config(cfg)
    o.set_source(orb)
    o.set_source_kind(kind)
    x, th = wl.grid_axes(cfg)
    for half in (False, True):
        for ks in (0, 3):
            T = o.source_field(0, ks, half)
            xs = (x[:-1] + 0.5 * cfg.dx) if half else x
            w = cfg.dx * cfg.dtheta
            assert abs(T.sum() * w - (1.5 - 0.5j)) < 1e-12
            assert abs((T.real * xs[:, None]).sum() * w / 1.5 - orb["rs_p"][ks]) < 1e-11
            assert abs((T.real * th[None, :]).sum() * w / 1.5 - orb["theta_p"][ks]) < 1e-12
            nz = np.argwhere(T != 0.0)
            assert nz[:, 0].max() - nz[:, 0].min() <= 2 * kind - 1
            assert nz[:, 1].max() - nz[:, 1].min() <= 2 * kind - 1
    # evolution: the deposit enters Pi exactly as the Gaussian does (same time levels, P7)
    ob = dict(orb)
    ob["amp_re"] = np.zeros_like(orb["amp_re"]); ob["amp_im"] = np.zeros_like(orb["amp_im"])
    ob["amp_re"][:, 0] = 1.0
    o2 = orc.OracleSolver.from_config(cfg)
    o2.set_source(ob)
    o2.set_source_kind(kind)
    o2.step(1)
    o.set_source(ob)
    Th = o.source_field(0, 0, True)
    hs = o2.get_half()
    assert np.allclose(hs[2][0], 0.5 * cfg.dt * Th.real, rtol=1e-14, atol=0)
    assert np.count_nonzero(hs[2][0]) == np.count_nonzero(Th.real) > 0


# ------------------------------------------------------------------------------------------ P10
# The waveform tap ("waveform at a fixed r*"): cell index i0, interpolation
# fraction f, the (1 - f) / f pairing, the weights' column and the mode index.
def _tap_case():
    a, n_r, n_th, rs = 0.6, 41, 12, (-10.0, 30.0)
    dx = (rs[1] - rs[0]) / (n_r - 1)
    x_obs = rs[0] + (17 + 0.37) * dx                       # off node: f = 0.37 (up to rounding)
    rng = np.random.default_rng(1206)
    W = rng.uniform(0.5, 2.0, n_th) * np.where(np.arange(n_th) % 2, 1.0, -1.0)   # distinct, both signs
    return a, n_r, n_th, rs, dx, x_obs, W


def test_p10_tap_is_the_interpolated_weighted_sum_of_the_state(orc):
    """Every recorded sample equals sum_j W_j [(1 - f) Phi_{i0,j} + f Phi_{i0+1,j}] evaluated here, with numpy and
    with i0, f from exact rational arithmetic, on the state the oracle hands out at that iteration."""
    from fractions import Fraction
    a, n_r, n_th, rs, dx, x_obs, W = _tap_case()
    modes = [2, -1, 0]
    o = orc.OracleSolver(a, 1.0, modes, rs[0], rs[1], n_r, n_th, 0.05 * dx)
    rng = np.random.default_rng(7)
    o.set_initial(*[rng.standard_normal((3, n_r, n_th)) for _ in range(4)])
    o.add_observer(x_obs, W)
    v = (Fraction(x_obs) - Fraction(rs[0])) / Fraction(dx)          # exact value of (x_obs - x_min)/dx
    i0 = int(v // 1)
    f = float(v - i0)
    assert i0 == 17 and abs(f - 0.37) < 1e-12
    for n in range(1, 6):
        o.step(1)
        pr, pim, _, _ = o.get_state()
        phi = pr + 1j * pim
        t, w = o.waveform(0)
        assert len(t) == n and t[-1] == pytest.approx(n * 0.05 * dx, rel=1e-14)
        want = ((1.0 - f) * phi[:, i0, :] + f * phi[:, i0 + 1, :]) @ W
        assert np.all(np.abs(want) > 1e-3)
        assert np.allclose(w[-1], want, rtol=1e-13, atol=0), (n, w[-1], want)
        # a plausible mistake must fail: swapped pairing, neighbouring cell, unweighted sum
        for wrong in ((f * phi[:, i0, :] + (1.0 - f) * phi[:, i0 + 1, :]) @ W,
                      ((1.0 - f) * phi[:, i0 + 1, :] + f * phi[:, i0 + 2, :]) @ W,
                      ((1.0 - f) * phi[:, i0, :] + f * phi[:, i0 + 1, :]).sum(axis=1)):
            assert not np.allclose(w[-1], wrong, rtol=1e-6, atol=0)
    o.close()


@pytest.mark.parametrize("jstar", [0, 5, 11])
def test_p10_tap_closed_form_on_a_field_linear_in_x(orc, jstar):
    """Phi(x, theta_j) = (c0 + c1 x) delta_{j,j*}, Pi = 0, frozen by a time step of 1e-13 dx: linear interpolation
    is exact on it, so the tap is W_{j*} (c0 + c1 x_obs) -- a closed form that knows nothing about i0 or f.
    A wrong f or a swapped pairing moves x by a fraction of dx, a wrong column picks another weight."""
    a, n_r, n_th, rs, dx, x_obs, W = _tap_case()
    x = rs[0] + dx * np.arange(n_r)
    c0, c1 = 0.3 - 0.2j, 0.05 + 0.11j
    o = orc.OracleSolver(a, 1.0, [2, 3], rs[0], rs[1], n_r, n_th, 1e-13 * dx)
    phi = np.zeros((2, n_r, n_th), dtype=complex)
    phi[0, :, jstar] = c0 + c1 * x
    phi[1, :, jstar] = 2.0 * (c0 + c1 * x).conjugate()           # second mode: pins the mode index
    o.set_initial(np.ascontiguousarray(phi.real), np.ascontiguousarray(phi.imag), None, None)
    o.add_observer(x_obs, W)
    o.step(1)
    _, w = o.waveform(0)
    o.close()
    want = np.array([W[jstar] * (c0 + c1 * x_obs), W[jstar] * 2.0 * (c0 + c1 * x_obs).conjugate()])
    assert np.allclose(w[0], want, rtol=1e-10, atol=0), (w[0], want)
    moved = W[jstar] * (c0 + c1 * (x_obs + 0.26 * dx))             # (1 - f) <-> f swapped
    assert abs(w[0][0] - moved) > 1e-4 * abs(want[0])


def test_p10_tap_default_weights_and_node_observer(orc):
    """weights = NULL means W_j = 1 (reading B2); an observer on a node has f = 0 and reads that row."""
    a, n_r, n_th, rs, dx, _, _ = _tap_case()
    o = orc.OracleSolver(a, 1.0, [2], rs[0], rs[1], n_r, n_th, 0.05 * dx)
    rng = np.random.default_rng(3)
    o.set_initial(*[rng.standard_normal((1, n_r, n_th)) for _ in range(4)])
    o.add_observer(rs[0] + 20 * dx, None)
    o.step(3)
    pr, pim, _, _ = o.get_state()
    _, w = o.waveform(0)
    o.close()
    assert np.allclose(w[-1, 0], (pr[0, 20] + 1j * pim[0, 20]).sum(), rtol=1e-12, atol=0)


# ------------------------------------------------------------------------------------------ P11
# The trajectory / amplitude generator (workloads.orbit_table).  It feeds
# BOTH sides of every sourced parity test, so a mistake in it is invisible there: it is pinned here against the
# Boyer-Lindquist metric itself, closed forms, a finer quadrature and hand-worked amplitudes.
def _bl_metric_equatorial(r, M, a):
    """Covariant Boyer-Lindquist components at theta = pi/2 [textbook]: g_tt, g_tphi, g_phiphi, g_rr."""
    return (-(1.0 - 2.0 * M / r), -2.0 * M * a / r, r * r + a * a + 2.0 * M * a * a / r,
            r * r / (r * r - 2.0 * M * r + a * a))


@pytest.mark.parametrize("a", [0.0, 0.7, 0.9, 0.99])
@pytest.mark.parametrize("r0", [6.5, 10.0, 12.0])
def test_p11_circular_orbit_satisfies_the_metric(a, r0):
    """u = u^t (1, 0, 0, Omega): normalisation g(u, u) = -1 and the radial geodesic equation
    d_r g_tt + 2 Omega d_r g_tphi + Omega^2 d_r g_phiphi = 0 (r-derivatives by central differences)."""
    M = 1.0
    Om = float(wl.circular_frequency(r0, M, a))
    ut = float(wl.circular_ut(r0, M, a))
    gtt, gtp, gpp, _ = _bl_metric_equatorial(r0, M, a)
    assert ut * ut * (gtt + 2.0 * gtp * Om + gpp * Om * Om) == pytest.approx(-1.0, rel=1e-13)
    h = 1e-4
    lo, hi = _bl_metric_equatorial(r0 - h, M, a), _bl_metric_equatorial(r0 + h, M, a)
    d = [(p - q) / (2 * h) for p, q in zip(hi, lo)]
    assert abs(d[0] + 2.0 * Om * d[1] + Om * Om * d[2]) < 1e-9
    assert Om > 0.0                                                     # prograde
    if a == 0.0:
        assert Om == pytest.approx(r0 ** -1.5, rel=1e-15)
        assert ut == pytest.approx((1.0 - 3.0 * M / r0) ** -0.5, rel=1e-15)


@pytest.mark.parametrize("a", [0.0, 0.7])
def test_p11_eccentric_constants_and_rates(a):
    """E, L of the p = 8, e = 0.3 orbit: the Schwarzschild closed forms at a = 0; u_r = 0 at both turning points
    written with the INVERSE metric (g^tt E^2 - 2 g^tphi E L + g^phiphi L^2 = -1), not with the radial potential
    the generator solves; along the orbit g(u, u) = -1 with u^r = (dr/dchi)(dchi/dtau); prograde; e -> 0 limit."""
    M, p, e = 1.0, 8.0, 0.3
    E, L = wl._eccentric_constants(p, e, M, a)
    if a == 0.0:
        assert E == pytest.approx(math.sqrt(((p - 2) ** 2 - 4 * e * e) / (p * (p - 3 - e * e))), rel=1e-13)
        assert L == pytest.approx(p * M / math.sqrt(p - 3 - e * e), rel=1e-13)
    for r in (p * M / (1 + e), p * M / (1 - e)):
        gtt, gtp, gpp, _ = _bl_metric_equatorial(r, M, a)
        det = gtt * gpp - gtp * gtp
        itt, itp, ipp = gpp / det, -gtp / det, gtt / det              # inverse of the (t, phi) block
        assert itt * E * E - 2.0 * itp * E * L + ipp * L * L == pytest.approx(-1.0, abs=2e-12)
    assert 0.0 < E < 1.0 and L > 0.0
    for chi in (0.3, 1.7, 3.0, 4.4):
        dchi_dt, dphi_dt, ut, r = wl._eccentric_rates(chi, p, e, M, a, E, L)
        assert r == pytest.approx(p * M / (1 + e * math.cos(chi)), rel=1e-15)
        gtt, gtp, gpp, grr = _bl_metric_equatorial(r, M, a)
        ur = (p * M * e * math.sin(chi) / (1 + e * math.cos(chi)) ** 2) * dchi_dt * ut
        uphi = dphi_dt * ut
        norm = gtt * ut * ut + 2.0 * gtp * ut * uphi + gpp * uphi * uphi + grr * ur * ur
        assert norm == pytest.approx(-1.0, abs=1e-11), (chi, norm)
        # conserved quantities from the velocities: E = -u_t, L = u_phi
        assert -(gtt * ut + gtp * uphi) == pytest.approx(E, rel=1e-12)
        assert gtp * ut + gpp * uphi == pytest.approx(L, rel=1e-12)
    # e -> 0: the circular orbit of radius p M
    E0, L0 = wl._eccentric_constants(10.0, 1e-7, M, a)
    _, dphi_dt, ut, _ = wl._eccentric_rates(0.4, 10.0, 1e-7, M, a, E0, L0)
    assert dphi_dt == pytest.approx(float(wl.circular_frequency(10.0, M, a)), rel=1e-6)
    assert ut == pytest.approx(float(wl.circular_ut(10.0, M, a)), rel=1e-6)


def test_p11_eccentric_table_integrates_its_own_rates():
    """The RK4 table of config 4's orbit: phi and r at sample k against an independent high-order quadrature of
    dphi/dchi = (dphi/dt)/(dchi/dt) and dt/dchi (scipy.integrate.quad) up to the same anomaly."""
    from scipy import integrate
    cfg = wl.CONFIGS[4].scaled(n_r=4001, steps=400)                 # dt = 0.05 dx, dx = 0.25: 801 samples, t <= 5
    tab = wl.orbit_table(cfg)
    M, a, p, e = cfg.M, cfg.a, 8.0, 0.3
    E, L = wl._eccentric_constants(p, e, M, a)
    r_tab = _r_from_tortoise(tab["rs_p"], M, a)
    # anomaly at the last sample from its radius (chi in (0, pi) on the outgoing branch)
    chi_end = math.acos((p * M / r_tab[-1] - 1.0) / e)
    T, _ = integrate.quad(lambda c: 1.0 / wl._eccentric_rates(c, p, e, M, a, E, L)[0], 0.0, chi_end, epsabs=1e-13)
    PH, _ = integrate.quad(lambda c: wl._eccentric_rates(c, p, e, M, a, E, L)[1] /
                           wl._eccentric_rates(c, p, e, M, a, E, L)[0], 0.0, chi_end, epsabs=1e-13)
    assert T == pytest.approx(cfg.steps * cfg.dt, rel=1e-9)
    phit = PH + float(wl.azimuth_shift(r_tab[-1], M, a))
    for k, m in enumerate(cfg.modes):
        amp = tab["amp_re"][k, -1] + 1j * tab["amp_im"][k, -1]
        assert np.angle(amp * np.exp(1j * m * phit)) == pytest.approx(0.0, abs=1e-8)


def _r_from_tortoise(x, M, a):
    """Invert wl.tortoise_forward by bisection (test helper; the forward map is pinned by P1)."""
    rp = M + math.sqrt(M * M - a * a)
    out = []
    for xv in np.atleast_1d(x):
        lo, hi = rp * (1 + 1e-15), 1e4
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if float(wl.tortoise_forward(mid, M, a)) < xv:
                lo = mid
            else:
                hi = mid
        out.append(0.5 * (lo + hi))
    return np.array(out)


def test_p11_inspiral_phase_against_a_finer_quadrature():
    """Config 5's phase phi(t) = int Omega(r0(t')) dt' (Simpson per sample interval) against adaptive quadrature
    of the same integrand, at three sample times and for a table that starts late (t0 > 0)."""
    from scipy import integrate
    cfg = wl.CONFIGS[5]
    n = 3000
    tab = wl.orbit_table(cfg, n_steps=n)
    T = cfg.steps * cfg.dt
    om = lambda t: float(wl.circular_frequency(12.0 - 6.0 * t / T, cfg.M, cfg.a))
    r_tab = _r_from_tortoise(tab["rs_p"][[0, n, 2 * n]], cfg.M, cfg.a)
    for q, k in enumerate((0, n, 2 * n)):
        t = 0.5 * cfg.dt * k
        assert r_tab[q] == pytest.approx(12.0 - 6.0 * t / T, rel=1e-10)   # r0(t) linear from 12 towards 6
        phi, _ = integrate.quad(om, 0.0, t, epsabs=1e-14, epsrel=1e-14)
        phit = phi + float(wl.azimuth_shift(r_tab[q], cfg.M, cfg.a))
        amp = tab["amp_re"][0, k] + 1j * tab["amp_im"][0, k]
        assert np.angle(amp * np.exp(2j * phit)) == pytest.approx(0.0, abs=1e-10)
    t0 = 0.37 * T
    late = wl.orbit_table(cfg, n_steps=10, t0=t0)
    phi, _ = integrate.quad(om, 0.0, t0, epsabs=1e-13, epsrel=1e-13, limit=200)
    r0 = 12.0 - 6.0 * t0 / T
    amp = late["amp_re"][0, 0] + 1j * late["amp_im"][0, 0]
    assert np.angle(amp * np.exp(2j * (phi + float(wl.azimuth_shift(r0, cfg.M, cfg.a))))) == pytest.approx(0.0, abs=1e-8)


def _golden_amplitudes():
    rows = []
    for line in open(os.path.join(GOLDEN, "source_amplitude.txt")):
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split("|")
        rows.append(([float(v) for v in left.split()], [float(v) for v in right.split()]))
    return rows


def test_p11_amplitude_golden_values():
    """A'_m = (2 mu/u^t) R2 / (Sigma^2 r^3 sin theta) exp(-i m phi~) at the hand-worked points
    of tests/golden/source_amplitude.txt (derivation in the file), against the generated table of config 3's orbit."""
    for (a, r0, m, t), (mag, phase) in _golden_amplitudes():
        cfg = wl.CONFIGS[3].scaled(a=a, modes=(int(m),), n_r=1001, rs_min=-100.0, rs_max=900.0, dt_over_dx=t / 100.0,
                                   steps=100)                            # sample 200 is at t
        assert r0 == 10.0
        tab = wl.orbit_table(cfg)
        amp = tab["amp_re"][0, 200] + 1j * tab["amp_im"][0, 200]
        assert abs(amp) == pytest.approx(mag, rel=1e-13)
        assert np.angle(amp * np.exp(-1j * phase)) == pytest.approx(0.0, abs=1e-11)
        assert tab["theta_p"][200] == pytest.approx(math.pi / 2, rel=1e-16)
        assert tab["sigma_r"] == pytest.approx(4 * cfg.dx) and tab["sigma_theta"] == pytest.approx(4 * cfg.dtheta)
        assert tab["half_window"] == 24 and tab["n_samples"] == 201


# ------------------------------------------------------------------------------------------ P12
# f2: deposit of a SUM of rank-1 terms whose profiles are the delta
# function's first and second derivatives.  The physical coefficients are not in the paper; what is pinned is the
# mechanism: each derivative profile acts on grid functions as (-1)^k d^k/dx^k at the particle.
def _lagrange_weights(nodes, xp, order):
    """d^order/dx^order at xp of the Lagrange basis polynomials on `nodes`, in exact rational arithmetic."""
    from fractions import Fraction
    out = []
    for i, xi in enumerate(nodes):
        poly = [Fraction(1)]                                    # coefficients of L_i, lowest power first
        for q, xq in enumerate(nodes):
            if q == i:
                continue
            den = xi - xq
            poly = [(poly[k - 1] if k > 0 else 0) - (xq * poly[k] if k < len(poly) else 0) for k in range(len(poly) + 1)]
            poly = [c / den for c in poly]
        for _ in range(order):
            poly = [k * poly[k] for k in range(1, len(poly))] or [Fraction(0)]
        out.append(sum(c * xp ** k for k, c in enumerate(poly)))
    return out


@pytest.mark.parametrize("kind,order", [(1, 1), (2, 1), (2, 2)])
def test_p12_discrete_delta_derivatives_are_lagrange_derivatives(orc, kind, order):
    """delta^(k) weights on the stencil around x_p = x_k + gamma h are (-1)^k L_i^(k)(x_p)/h (exact rationals on
    dyadic h, gamma: the oracle's floats must agree to the last bits), incl. gamma = 0 (particle on a node) and
    the points just outside the stencil (weight 0)."""
    from fractions import Fraction
    h = Fraction(1, 4)
    npts = 2 if kind == 1 else 4
    for gam in (Fraction(0), Fraction(1, 8), Fraction(1, 2), Fraction(13, 16), Fraction(1023, 1024)):
        k = 7
        xp = (k + gam) * h
        first = k if kind == 1 else k - 1
        nodes = [(first + q) * h for q in range(npts)]
        want = [(-1) ** order * w / h for w in _lagrange_weights(nodes, xp, order)]
        for q in range(-2, npts + 2):
            y = float((first + q) * h - xp)
            got = orc.profile_deriv(kind, order, y, float(h))
            exp = float(want[q]) if 0 <= q < npts else 0.0
            assert got == pytest.approx(exp, rel=4e-15, abs=1e-300), (kind, order, gam, q, got, exp)


@pytest.mark.parametrize("kind,order,degree", [(1, 1, 1), (2, 1, 3), (2, 2, 3)])
def test_p12_discrete_delta_derivative_moments(orc, kind, order, degree):
    """sum_i P^(k)(x_i - x_p) (x_i - x_p)^q h = (-1)^k k! delta_{qk} for every q up to the degree of the rule."""
    h = 0.37
    for gam in (0.0, 0.21, 0.5, 0.93):
        xp = 5 * h + gam * h
        xs = h * np.arange(0, 12)
        w = np.array([orc.profile_deriv(kind, order, x - xp, h) for x in xs])
        assert np.count_nonzero(w) <= (2 if kind == 1 else 4)
        for q in range(degree + 1):
            mom = float((w * (xs - xp) ** q).sum() * h)
            exp = (-1) ** order * math.factorial(order) if q == order else 0.0
            assert mom == pytest.approx(exp, abs=2e-12 / h ** max(order - q, 0)), (kind, order, gam, q, mom)


def test_p12_gaussian_derivatives(orc):
    """g' and g'' against mpmath's numerical derivative of the printed Gaussian (C.6), and their
    discrete moments on a 6-sigma window: sum g' (x - x_p) h = -1, sum g'' (x - x_p)^2 h = 2, lower moments 0."""
    import mpmath as mp
    mp.mp.dps = 40
    sig = 0.8
    g = lambda y: mp.exp(-y * y / (2 * mp.mpf(sig) ** 2)) / (mp.mpf(sig) * mp.sqrt(2 * mp.pi))
    for y in (-2.3, -0.4, 0.0, 0.05, 0.8, 3.1):
        for order in (0, 1, 2):
            want = float(mp.diff(g, mp.mpf(y), order))
            assert orc.profile_deriv(0, order, y, sig) == pytest.approx(want, rel=1e-13, abs=1e-15), (y, order)   # abs: g'' vanishes at y = sigma
    h = sig / 4.0                                                   # the configs' width: sigma = 4 cells
    xp = 10.3 * h
    xs = h * np.arange(-20, 45)
    for order in (1, 2):
        w = np.array([orc.profile_deriv(0, order, x - xp, sig) for x in xs])
        for q in range(3):
            mom = float((w * (xs - xp) ** q).sum() * h)
            exp = (-1) ** order * math.factorial(order) if q == order else 0.0
            assert mom == pytest.approx(exp, abs=1e-7), (order, q, mom)


@pytest.mark.parametrize("kind", [0, 2])
def test_p12_multi_term_deposit(orc, kind):
    """The 2D deposit of a sum of terms: superposition of single-term fields, each term's moments
    (sum T (x - x_p)^p (theta - theta_p)^q dx dtheta = A (-1)^(a+b) a! b! iff (p, q) = (a, b), else 0 for p <= a,
    q <= b), the stage grids and time levels of P7, and that an empty term list restores the monopole."""
    cfg = wl.small_test_configs()[3].scaled(name="terms", n_r=401, rs_min=-10.0, rs_max=30.0, steps=4)
    orb = wl.orbit_table(cfg)
    ns, nm = orb["n_samples"], cfg.n_modes
    rng = np.random.default_rng(5)
    specs = [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]
    amps = [(rng.standard_normal((nm, ns)) + 1j * rng.standard_normal((nm, ns))) for _ in specs]
    x = cfg.rs_min + cfg.dx * np.arange(cfg.n_r)
    xh = x[:-1] + 0.5 * cfg.dx
    th = (np.arange(cfg.n_theta) + 0.5) * cfg.dtheta
    o = orc.OracleSolver.from_config(cfg)
    o.set_source(orb)
    o.set_source_kind(kind)
    mono = o.source_field(0, 1, False)
    tol = 1e-5 if kind == 0 else 1e-10      # Gaussian: the window cuts the tails at 6 sigma (y^2 g'' there is 1e-6 of its peak)
    singles = []
    for (a_, b_), A in zip(specs, amps):
        o.set_source_terms([(a_, b_, A)])
        for half, ks, xs in ((False, 1, x), (True, 2, xh)):
            T = o.source_field(0, ks, half)
            dxp, dthp = xs - orb["rs_p"][ks], th - orb["theta_p"][ks]
            for p_ in range(a_ + 1):
                for q_ in range(b_ + 1):
                    mom = (T * (dxp[:, None] ** p_) * (dthp[None, :] ** q_)).sum() * cfg.dx * cfg.dtheta
                    exp = A[0, ks] * (-1) ** (a_ + b_) * math.factorial(a_) * math.factorial(b_) if (p_, q_) == (a_, b_) else 0.0
                    scale = abs(A[0, ks]) / (cfg.dx ** (a_ - p_) * cfg.dtheta ** (b_ - q_))
                    assert abs(mom - exp) <= tol * scale, (kind, a_, b_, p_, q_, half, mom, exp)
        singles.append(o.source_field(0, 1, False))
    o.set_source_terms(list((a_, b_, A) for (a_, b_), A in zip(specs, amps)))
    both = o.source_field(0, 1, False)
    assert np.allclose(both, sum(singles), rtol=1e-13, atol=1e-13 * np.abs(both).max())
    # time levels: from zero data, Pi^1 at the nodes = dt T(sample 1) + what the half step (sample 0) feeds in;
    # with the amplitudes of sample 0 zeroed only the full step's deposit remains
    A0 = [A.copy() for A in amps]
    for A in A0:
        A[:, 0] = 0.0
    o.set_source_terms(list((a_, b_, A) for (a_, b_), A in zip(specs, A0)))
    o.set_initial()
    o.step(1)
    _, _, pi_re, pi_im = o.get_state()
    assert np.allclose((pi_re + 1j * pi_im)[0][1:-1], cfg.dt * both[1:-1], rtol=1e-13, atol=1e-13 * cfg.dt * np.abs(both).max())
    o.set_source_terms([])
    assert np.array_equal(o.source_field(0, 1, False), mono)
    # the (0, 0) term with the trajectory's own amplitude IS the monopole
    o.set_source_terms([(0, 0, orb["amp_re"] + 1j * orb["amp_im"])])
    assert np.allclose(o.source_field(0, 1, False), mono, rtol=1e-15, atol=0)
    with pytest.raises(ValueError):
        o.set_source_terms([(3, 0, amps[0])])
    o.close()
