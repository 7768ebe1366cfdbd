"""Pins of oracle/waveform.py (eqs. 5-9) against things the oracle does not compute itself."""
from fractions import Fraction
import math

import numpy as np
import pytest

from oracle import waveform as wf


def test_sixteen_samples_per_cycle_closed_form():
    """f0 = 2^-7 Hz sampled every 8 s is exactly 1/16 cycle per sample: the series has period 16 and takes the
    values a cos(2 pi n / 16), a sin(2 pi n / 16) (eq. 5 with fdot = 0, phi0 = 0)."""
    ap, ac = 3.0e-22, -1.25e-22
    hp, hc = wf.gb_waveform((ap, ac, 2.0 ** -7, 0.0, 0.0, 0.0), 0.0, 8.0, 64)
    for n in range(64):
        assert hp[n] == pytest.approx(ap * math.cos(2 * math.pi * (n % 16) / 16), abs=1e-15 * abs(ap))
        assert hc[n] == pytest.approx(ac * math.sin(2 * math.pi * (n % 16) / 16), abs=1e-15 * abs(ac))
    assert np.array_equal(hp[:48], hp[16:]) and np.array_equal(hc[:48], hc[16:])
    assert hp[0] == ap and hp[8] == -ap and abs(hp[4]) < 1e-19 * abs(ap)
    assert hc[4] == ac and hc[12] == -ac and abs(hc[8]) < 1e-19 * abs(ac)


def test_late_start_keeps_the_phase():
    """The same signal started 2^40 s later (2^33 whole cycles): identical samples — the phase is reduced
    exactly, not in floating point (fp64 would be off by 1e-6 cycles there)."""
    par = (1.0, 1.0, 2.0 ** -7, 0.0, 0.0, 0.3)
    a = wf.gb_waveform(par, 0.0, 8.0, 32)
    b = wf.gb_waveform(par, 2.0 ** 40, 8.0, 32)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_unit_circle():
    par = (2.0e-22, -0.7e-22, 3.1234e-3, 1.7e-16, wf.fddot_eq8(3.1234e-3, 1.7e-16), 1.1)
    hp, hc = wf.gb_waveform(par, 2.5e7, 10.0, 500)
    assert np.abs((hp / par[0]) ** 2 + (hc / par[1]) ** 2 - 1.0).max() < 5e-16


def test_chirp_phase_by_integer_arithmetic():
    """f0 = 2^-7, fdot = 2^-30, t = 2^12 s: f0 t = 32 cycles, fdot t^2 / 2 = 2^-7 cycles -> phase 2 pi / 128."""
    hp, hc = wf.gb_waveform((1.0, 1.0, 2.0 ** -7, 2.0 ** -30, 0.0, 0.0), 2.0 ** 12, 1.0, 1)
    assert hp[0] == pytest.approx(math.cos(2 * math.pi / 128), abs=1e-15)
    assert hc[0] == pytest.approx(math.sin(2 * math.pi / 128), abs=1e-15)
    # with the cubic term: fddot = 3 * 2^-40 adds fddot t^3 / 6 = 2^-5 cycles
    hp, hc = wf.gb_waveform((1.0, 1.0, 2.0 ** -7, 2.0 ** -30, 3 * 2.0 ** -40, 0.0), 2.0 ** 12, 1.0, 1)
    assert hp[0] == pytest.approx(math.cos(2 * math.pi * (1 / 128 + 1 / 32)), abs=1e-15)
    assert hc[0] == pytest.approx(math.sin(2 * math.pi * (1 / 128 + 1 / 32)), abs=1e-15)


def test_instantaneous_frequency_exact():
    """Central difference of the cubic phase: [c(t + d) - c(t - d)] / (2 d) = f0 + fdot t + fddot t^2 / 2 +
    fddot d^2 / 6, exactly — fixes each coefficient (1, 1/2, 1/6) of eq. 5's argument."""
    f0, fdot, fddot = 3.3e-3, 4.1e-15, 2.9e-26
    for t, d in ((12345.0, 7.0), (9.1e7, 0.5), (-3.0e6, 1000.0)):
        lhs = (wf.cycles_exact(f0, fdot, fddot, Fraction(t) + Fraction(d)) -
               wf.cycles_exact(f0, fdot, fddot, Fraction(t) - Fraction(d))) / (2 * Fraction(d))
        rhs = (Fraction(f0) + Fraction(fdot) * Fraction(t) + Fraction(fddot) * Fraction(t) ** 2 / 2 +
               Fraction(fddot) * Fraction(d) ** 2 / 6)
        assert lhs == rhs


def test_phi0_is_a_phase_shift():
    """phi0 = pi/2 turns cos into -sin and sin into cos (eq. 5: phi0 is added to the argument)."""
    base = wf.gb_waveform((1.0, 1.0, 1.7e-3, 0.0, 0.0, 0.0), 100.0, 10.0, 200)
    quarter = wf.gb_waveform((1.0, 1.0, 1.7e-3, 0.0, 0.0, math.pi / 2), 100.0, 10.0, 200)
    assert np.abs(quarter[0] + base[1]).max() < 2e-16
    assert np.abs(quarter[1] - base[0]).max() < 2e-16


def test_eq9_limits_and_eq8():
    """eq. 9: face-on (iota = 0) is circular, |a+| = |ax| = 2A; edge-on (iota = pi/2) is linear, ax = 0, |a+| =
    A.  eq. 8 is d/dt of eq. 7: fdot = K f^(11/3)  =>  fddot = 11/3 K f^(8/3) fdot = 11/3 fdot^2 / f."""
    ap, ac = wf.amplitudes_paper(1e-22, 0.0)
    assert ap == -2e-22 and ac == -2e-22
    ap, ac = wf.amplitudes_paper(1e-22, math.pi / 2)
    assert ap == pytest.approx(-1e-22, rel=1e-15) and abs(ac) < 2e-38
    cp, cc = wf.amplitudes_config(1e-22, 0.4)
    pp, pc = wf.amplitudes_paper(1e-22, 0.4)
    assert cp == -pp and cc == pc
    K, f = 3.7e-7, 4.0e-3                      # any K: fdot = K f^(11/3)
    fdot = K * f ** (11.0 / 3.0)
    h = 1e-9                                   # d(fdot)/dt = (dfdot/df) fdot, central difference in f
    dfdot_df = (K * (f + h) ** (11.0 / 3.0) - K * (f - h) ** (11.0 / 3.0)) / (2 * h)
    assert wf.fddot_eq8(f, fdot) == pytest.approx(dfdot_df * fdot, rel=1e-6)


def test_long_double_variant_agrees():
    """The vectorised long-double form against the exact-phase form after a year at 5 mHz (1.6e5 cycles)."""
    par = (1.0e-22, -0.8e-22, 5.0e-3, 2.0e-16, wf.fddot_eq8(5.0e-3, 2.0e-16), 0.7)
    a = wf.gb_waveform(par, 3.0e7, 10.0, 300, first=150000)
    b = wf.gb_waveform_ld(par, 3.0e7, 10.0, 300, first=150000)
    assert np.abs(a[0] - b[0]).max() < 1e-12 * abs(par[0])
    assert np.abs(a[1] - b[1]).max() < 1e-12 * abs(par[1])
