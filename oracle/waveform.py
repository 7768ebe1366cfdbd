"""CPU ORACLE of the template generator ("generate the GB waveform ... from the
parameters"): the Galactic-binary waveform of PAPER.md eqs. 5-9.
TEST INFRASTRUCTURE — imported only by tests/ (never by paper_2204_06633_b200).

What is computed, in the paper's notation (eq. 5, with the polarisation amplitudes of eq. 9 factored out):

    cycles(t) = f0 t + 1/2 fdot t^2 + 1/6 fddot t^3                                   (argument of eq. 5 / 2 pi)
    h+(t) = a+ cos(2 pi cycles(t) + phi0),    hx(t) = ax sin(2 pi cycles(t) + phi0)   (eqs. 5a, 5b)

at the sample times t_n = t0 + n dt.  Eq. 9's inclination factors and signs are the amplitudes
    a+ = -A (1 + cos^2 iota),   ax = -2 A cos(iota)                                   (`amplitudes_paper`)
and its rotation by 2 psi is applied by the projection to the basis (u, v) instead (reading A4), so
psi does not appear here.  Eq. 8 closes the frequency evolution: fddot = 11/3 fdot^2 / f0 (`fddot_eq8`).
BASELINE.json's configs use a+ = +A (1 + cos^2 iota), ax = -2 A cos(iota), fddot = 0 (`amplitudes_config`).

How: the inputs are doubles, i.e. exact rationals, so cycles(t_n) is evaluated EXACTLY with Python fractions,
reduced modulo one exactly, and only then turned into an angle and passed to the long-double cos / sin.  (A
product f0 * t rounded to fp64 would already be wrong by 1e-10 cycles after a year at a few mHz.)
`gb_waveform_ld` is the same formula in vectorised long-double arithmetic for long series; the two agree to
1e-12 of the amplitude (tests/test_oracle_waveform.py), which is the long-double rounding of f0 * t.

Pins (tests/test_oracle_waveform.py): a frequency of exactly 1/16 cycle per sample repeats with period 16 and
hits 0 and +-a at the quarter periods; (h+/a+)^2 + (hx/ax)^2 = 1; a chirp whose phase at t = 2^12 s is 32 +
1/128 cycles by integer arithmetic; the central difference of cycles(t) is f0 + fdot t + fddot t^2 / 2 +
fddot delta^2 / 6 exactly (every coefficient of the cubic); face-on and edge-on limits of eq. 9; eq. 8 against
eq. 7 differentiated by hand.
"""
from fractions import Fraction
import math

import numpy as np

LD = np.longdouble
NPAR = 6   # a_plus, a_cross, f0, fdot, fddot, phi0


def fddot_eq8(f0, fdot):
    """eq. 8: second frequency derivative of a binary driven by gravitational radiation."""
    return 11.0 / 3.0 * fdot * fdot / f0


def amplitudes_paper(A, iota):
    """(a+, ax) of eq. 9 without the 2 psi rotation (which the projection applies)."""
    ci = math.cos(iota)
    return -A * (1.0 + ci * ci), -2.0 * A * ci


def amplitudes_config(A, iota):
    """(a+, ax) of BASELINE.json's configs ("opposite h+ sign")."""
    ci = math.cos(iota)
    return A * (1.0 + ci * ci), -2.0 * A * ci


def cycles_exact(f0, fdot, fddot, t):
    """f0 t + fdot t^2 / 2 + fddot t^3 / 6 as an exact rational; t may be a Fraction."""
    t = Fraction(t)
    return Fraction(f0) * t + Fraction(fdot) * t * t / 2 + Fraction(fddot) * t * t * t / 6


def _to_ld(q):
    """A rational |q| <= 1/2 as a long double, correct to 2^-64: q 2^80 rounded to an integer, split in two
    40-bit halves (each exact in a float, which is how numpy builds a long double from a Python int)."""
    k = (q.numerator << 80) // q.denominator
    hi, lo = k >> 40, k & ((1 << 40) - 1)
    return (LD(float(hi)) * LD(2.0 ** 40) + LD(float(lo))) * LD(2.0 ** -80)


def gb_waveform(par, t0, dt, n, first=0):
    """h+, hx (float64 arrays of length n) at t = t0 + (first + i) dt, i = 0..n-1, for one template
    par = (a_plus, a_cross, f0, fdot, fddot, phi0); exact phase reduction, long-double trigonometry."""
    ap, ac, f0, fdot, fddot, phi0 = (float(v) for v in par)
    two_pi = LD(2) * np.arccos(LD(-1))
    hp = np.empty(n)
    hc = np.empty(n)
    T0, DT = Fraction(t0), Fraction(dt)
    for i in range(n):
        c = cycles_exact(f0, fdot, fddot, T0 + (first + i) * DT)
        frac = c - math.floor(c + Fraction(1, 2))                  # in [-1/2, 1/2), exact
        ang = two_pi * _to_ld(frac) + LD(phi0)
        hp[i] = float(LD(ap) * np.cos(ang))
        hc[i] = float(LD(ac) * np.sin(ang))
    return hp, hc


def gb_waveform_ld(par, t0, dt, n, first=0):
    """Same formula, vectorised long double (phase good to ~1e-13 cycles per 1e6 cycles): for long series."""
    ap, ac, f0, fdot, fddot, phi0 = (LD(float(v)) for v in par)
    t = LD(t0) + LD(dt) * np.arange(first, first + n).astype(LD)
    c = f0 * t + fdot * t * t / LD(2) + fddot * t * t * t / LD(6)
    frac = c - np.floor(c + LD(0.5))
    ang = LD(2) * np.arccos(LD(-1)) * frac + phi0
    return (ap * np.cos(ang)).astype(np.float64), (ac * np.sin(ang)).astype(np.float64)
