#!/usr/bin/env python
"""Writes tests/golden/source_amplitude.txt: the source amplitude A'_m of SURVEY.md 8(c) C.6 (reading A7;
PAPER.md:76 right-hand side of Eq. (1)) at two hand-workable points, evaluated with mpmath at 40
digits directly from the printed expression.  Calls nothing from this repository."""
import os

import mpmath as mp

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def amplitude(a, r0, m, t):
    M = mp.mpf(1)
    a, r0, t = mp.mpf(a), mp.mpf(r0), mp.mpf(t)
    v = a * mp.sqrt(M) / r0 ** mp.mpf("1.5")
    ut = (1 + v) / mp.sqrt(1 - 3 * M / r0 + 2 * v)                      # circular equatorial prograde [textbook]
    Om = mp.sqrt(M) / (r0 ** mp.mpf("1.5") + a * mp.sqrt(M))
    rp, rm = M + mp.sqrt(M * M - a * a), M - mp.sqrt(M * M - a * a)
    Delta = r0 * r0 - 2 * M * r0 + a * a
    R2 = r0 * r0 + a * a
    Sig2 = R2 * R2 - a * a * Delta                                      # theta = pi/2
    mag = (2 / ut) * R2 / (Sig2 * r0 ** 3)
    shift = 0 if a == 0 else a / (rp - rm) * mp.log((r0 - rp) / (r0 - rm))
    phase = -m * (Om * t + shift)                                       # arg A' = -m phi~_p
    return mag, phase


LINES = """# Source amplitude A'_m(t) = (2 mu / u^t) R2_p / (Sigma_p^2 r_p^3 sin theta_p) exp(-i m phi~_p), mu = 1
# (SURVEY.md 8(c) C.6; from the right-hand side -4 pi (r^2 + a^2 cos^2 theta) T of PAPER.md:76 with the scalar
# point-particle density, PAPER.md:114), for the circular equatorial prograde orbit r0 = 10 M, theta_p = pi/2:
#   u^t = (1 + v)/sqrt(1 - 3M/r0 + 2v), v = a sqrt(M)/r0^1.5;  Omega = sqrt(M)/(r0^1.5 + a sqrt(M));
#   phi~_p = Omega t + a/(r+ - r-) ln((r0 - r+)/(r0 - r-)).
# Worked by hand for a = 0: u^t = 1/sqrt(0.7), R2 = 100, Sigma^2 = 10^4, so |A'| = 2 sqrt(0.7) 100/(10^4 10^3)
#   = 2 sqrt(0.7) 1e-5 = 1.6733200530681511e-05 and arg A' = -m t/10^1.5.
# For a = 0.9: v = 0.9/10^1.5 = 0.0284604989..., u^t = 1.0284604989.../sqrt(0.7569209978...) = 1.18212...,
#   Delta = 80.81, R2 = 100.81, Sigma^2 = 100.81^2 - 0.81*80.81 = 10097.2 ; evaluated with mpmath at 40 digits by
#   tests/golden/make_source_amplitude.py (this file's generator; it calls nothing from the repository).
# columns: a r0 m t | |A'| arg(A') (radians, not reduced)
"""

if __name__ == "__main__":
    out = LINES
    for a, r0, m, t in (("0", "10", 2, "7.5"), ("0.9", "10", 2, "7.5"), ("0.9", "10", 3, "2.5")):
        mag, phase = amplitude(a, r0, m, t)
        out += "%s %s %d %s | %s %s\n" % (a, r0, m, t, mp.nstr(mag, 20), mp.nstr(phase, 20))
    open(os.path.join(HERE, "source_amplitude.txt"), "w").write(out)
    print(out)
