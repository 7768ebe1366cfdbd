"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formula: they are closed forms (phasor TDI on a static
constellation), invariants (relabelling, orthogonality, partition of unity), reductions to
library routines (scipy CubicSpline / BarycentricInterpolator), continuous-time brute force
with mpmath, and printed worked-example values (tests/golden/worked_example_p2.json).
"""
import json
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator, CubicSpline

from oracle import oracle as O
from harness import inputs as I

LD = np.longdouble
C = I.C_LIGHT


def mp2ld(v):
    """mpmath -> long double (two-term split, exact to 2^-64)."""
    hi = float(v)
    return LD(hi) + LD(float(v - hi))


def ld2mp(x):
    hi = float(x)
    return mp.mpf(hi) + mp.mpf(float(LD(x) - LD(hi)))


def rel(a, b):
    a = np.asarray(a, dtype=LD)
    b = np.asarray(b, dtype=LD)
    return float(np.sqrt(np.sum((a - b) ** 2)) / np.sqrt(np.sum(b ** 2)))


# ------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("order", [1, 3, 9, 25, 41])
def test_p1_lagrange_exact_on_polynomials(order):
    """Exact for degree <= order, NOT for degree order+1 (reading A5)."""
    rng = np.random.default_rng(order)
    T = order + 1
    n_len = 4 * T + 40
    idx = np.arange(n_len)
    mp.mp.dps = 50
    for trial in range(5):
        coef = [mp.mpf(float(c)) for c in rng.normal(size=order + 1)]
        scale = mp.mpf(n_len)

        def poly(x, extra=0):
            z = (mp.mpf(x) - n_len / 2) / scale
            return sum(c * z ** k for k, c in enumerate(coef)) + extra * z ** (order + 1)

        n = int(rng.integers(2 * T, n_len - 2 * T))
        D = float(rng.uniform(-T / 2, T / 2))
        x = np.array([mp2ld(poly(int(i))) for i in idx], dtype=LD)
        want = poly(mp.mpf(n) - mp.mpf(D))
        assert abs(ld2mp(O.interp(x, n, LD(D), order)) - want) < 3e-18 * (1 + abs(want)) * (1 + order)
        # degree order+1 is NOT reproduced: the error is the node polynomial prod(eps - m) / scale^(order+1)
        x2 = np.array([mp2ld(poly(int(i), 1)) for i in idx], dtype=LD)
        err2 = ld2mp(O.interp(x2, n, LD(D), order)) - poly(mp.mpf(n) - mp.mpf(D), 1)
        p = T // 2
        eps = mp.ceil(mp.mpf(D)) - mp.mpf(D)
        node = mp.mpf(1)
        for m in range(-p + 1, p + 1):
            node *= (eps - m)
        node /= scale ** (order + 1)
        assert abs(err2 + node) < 1e-3 * abs(node) + 1e-18


@pytest.mark.parametrize("order", [1, 9, 25, 41])
def test_p1_weight_identities(order):
    p = (order + 1) // 2
    j = np.arange(-p + 1, p + 1).astype(LD)
    for eps in [LD(0.0), LD(0.123456789), LD(0.5), LD(0.999)]:
        w = O.lagrange_weights(order, eps)
        assert abs(float(w.sum() - 1)) < 1e-17                      # partition of unity
        assert abs(float((w * j).sum() - eps)) < 1e-16              # reproduces the position
        w_m = O.lagrange_weights(order, LD(1) - eps)                # mirror symmetry w_j(e) = w_{1-j}(1-e)
        assert np.max(np.abs(w - w_m[::-1])) < 1e-17
    w0 = O.lagrange_weights(order, LD(0))
    assert w0[p - 1] == 1 and np.all(np.delete(w0, p - 1) == 0)     # exact sample pass-through


def test_p1_lebesgue_constants():
    """Max over eps of sum |w_j| for the centred stencil: 1.00, 1.56, 1.88, 2.03."""
    want = {1: 1.00, 9: 1.56, 25: 1.88, 41: 2.03}
    for order, val in want.items():
        leb = max(float(np.abs(O.lagrange_weights(order, LD(e))).sum()) for e in np.linspace(0, 1, 201))
        assert abs(leb - val) < 0.006, (order, leb)


@pytest.mark.parametrize("order", [1, 5, 25])
def test_p1_stencil_placement_vs_scipy(order):
    """interp(x, n, D) equals the polynomial through samples q-p+1..q+p evaluated at n-D,
    q = n - ceil(D): the library routine is scipy's BarycentricInterpolator."""
    rng = np.random.default_rng(7 + order)
    p = (order + 1) // 2
    x = rng.normal(size=200)
    for D in [0.0, 0.25, 3.0, 3.75, -2.5, -0.999, 17.31]:
        n = 100
        q = n - int(np.ceil(D))
        nodes = np.arange(q - p + 1, q + p + 1)
        want = BarycentricInterpolator(nodes.astype(float), x[nodes])(n - D)
        got = float(O.interp(x.astype(LD), n, LD(D), order))
        assert abs(got - want) < 1e-11 * np.abs(x[nodes]).max() * (1 + order)
    # a linear ramp x[i] = i returns the target position n - D exactly: pins sign of D, ceil and eps
    ramp = np.arange(200).astype(LD)
    for D in [0.0, 0.3, 5.9, -4.2]:
        assert abs(float(O.interp(ramp, 100, LD(D), order) - (LD(100) - LD(D)))) < 1e-15


def test_p1_sinusoid_error_table():
    """Interpolation error on a unit sinusoid, max over eps."""
    want = {(1, 0.314): 1.1e-2, (9, 0.314): 1.9e-9, (9, 0.628): 1.7e-6, (25, 0.628): 7e-15}
    for (order, wdt), val in want.items():
        i = np.arange(120).astype(LD)
        x = np.sin(LD(wdt) * i)
        err = 0.0
        for e in np.linspace(0.0, 0.98, 25):
            for n in range(50, 72):        # scan the phase as well
                got = O.interp(x, n, LD(e), order)
                err = max(err, abs(float(got - np.sin(LD(wdt) * (LD(n) - LD(e))))))
        assert 0.3 * val < err < 3 * val, (order, wdt, err)


# ------------------------------------------------------------------------------ P9
def _poly_table(nk, knot_dt, cx, cl, t_start=0.0):
    """Orbit table whose 15 channels are cubic polynomials of t (exactly splinable)."""
    tk = t_start + knot_dt * np.arange(nk)
    x = np.empty((3, 3, nk))
    for i in range(3):
        for a in range(3):
            x[i, a] = np.polyval(cx[i][a][::-1], tk)
    ltt = np.stack([np.polyval(cl[s][::-1], tk) for s in range(6)])
    return I.OrbitTable(t_start, knot_dt, x, ltt)


def test_p9_spline_vs_scipy_and_cubics():
    tb = I.orbit_table("kepler", 0.0, 40 * I.DAY)
    orc = O.Oracle(tb, 10.0, 0.0, 25)
    tk = tb.t_start + tb.knot_dt * np.arange(tb.n_knots)
    tq = np.random.default_rng(1).uniform(tk[0], tk[-1], size=500)
    for ch in [0, 4, 8, 9, 14]:
        tab = tb.x.reshape(9, -1)[ch] if ch < 9 else tb.ltt[ch - 9]
        want = CubicSpline(tk, tab, bc_type="not-a-knot")(tq)
        got = orc.spline(ch, tq).astype(float)
        assert np.max(np.abs(got - want)) < 2e-14 * np.abs(tab).max()
    # a cubic is reproduced exactly (long double); integer coefficients and knots keep the table exact in fp64
    rng = np.random.default_rng(2)
    cx = [[[float(v) for v in rng.integers(-9, 10, size=4) * [100000, 100, 3, 1]] for _ in range(3)] for _ in range(3)]
    cl = [[float(v) for v in rng.integers(-9, 10, size=4)] for _ in range(6)]
    tp = _poly_table(12, 8.0, cx, cl)
    orc = O.Oracle(tp, 1.0, 0.0, 25)
    tq = rng.uniform(0, 88.0, size=100).astype(LD)
    mp.mp.dps = 40
    for ch, co in [(0, cx[0][0]), (5, cx[1][2]), (9, cl[0]), (14, cl[5])]:
        got = orc.spline(ch, tq)
        scale = max(abs(sum(mp.mpf(c) * mp.mpf(t) ** k for k, c in enumerate(co))) for t in (0, 44, 88)) + 1
        for tt, g in zip(tq, got):
            want = sum(mp.mpf(c) * ld2mp(tt) ** k for k, c in enumerate(co))
            assert abs(ld2mp(g) - want) < 2e-18 * scale


# ------------------------------------------------------------------------------ P2
def _phasor_reference(beta, lam, psi, iota, A, f, L, x):
    """Closed-form phasors on a static equal-arm constellation (mpmath), eqs. 9-12, 16-18."""
    mp.mp.dps = 40
    w = 2 * mp.pi * mp.mpf(f)
    cb, sb, cl, sl = mp.cos(beta), mp.sin(beta), mp.cos(lam), mp.sin(lam)
    k = [-cb * cl, -cb * sl, -sb]
    u0 = [sl, -cl, mp.mpf(0)]
    v0 = [-sb * cl, -sb * sl, cb]
    ap = mp.mpf(A) * (1 + mp.cos(iota) ** 2)
    ac = 2 * mp.mpf(A) * mp.cos(iota) * 1j
    c2, s2 = mp.cos(2 * psi), mp.sin(2 * psi)
    apR, acR = c2 * ap - s2 * ac, s2 * ap + c2 * ac           # eq. 9 rotation
    X = [[mp.mpf(float(x[i, a])) for a in range(3)] for i in range(3)]
    dot = lambda a, b: sum(p * q for p, q in zip(a, b))
    Y = {}
    for (i, j) in I.LINKS:
        d = [X[i - 1][a] - X[j - 1][a] for a in range(3)]
        nrm = mp.sqrt(dot(d, d))
        n = [q / nrm for q in d]
        xp = dot(u0, n) ** 2 - dot(v0, n) ** 2
        xc = 2 * dot(u0, n) * dot(v0, n)
        G = xp * apR + xc * acR
        te = mp.mpf(L) + dot(k, X[j - 1]) / C
        tr = dot(k, X[i - 1]) / C
        Y[(i, j)] = G * (mp.e ** (-1j * w * te) - mp.e ** (-1j * w * tr)) / (2 * (1 - dot(k, n)))
    D = mp.e ** (-1j * w * mp.mpf(L))
    out = {}
    for ch, name in enumerate("XYZ"):
        r = lambda i: (i - 1 + ch) % 3 + 1
        y13, y31, y12, y21 = Y[(r(1), r(3))], Y[(r(3), r(1))], Y[(r(1), r(2))], Y[(r(2), r(1))]
        X1 = (1 - D ** 2) * ((y13 + D * y31) - (y12 + D * y21))
        out[name] = (X1, (1 - D ** 4) * X1)
    return Y, out, w


def _series(ph, w, t):
    """Re[ph exp(i w t)] in long double."""
    wt = LD(float(w)) * t + (LD(float(w - float(w)))) * t
    return LD(float(ph.real)) * np.cos(wt) - LD(float(ph.imag)) * np.sin(wt)


@pytest.mark.parametrize("order,dt,tol", [(25, 10.0, 1e-13), (41, 5.0, 1e-13), (9, 10.0, 1e-10)])
def test_p2_closed_form_static(order, dt, tol, golden_dir):
    g = json.load(open(os.path.join(golden_dir, "worked_example_p2.json")))
    beta, lam, psi, iota, A, f = 0.2, 1.0, 0.3, 0.5, 1e-22, 2e-3
    L = I.ARM / C
    n, t0 = 3000, 5.0
    tb = I.orbit_table("static", t0, t0 + n * dt, const_ltt=L)
    Y, XYZ, w = _phasor_reference(beta, lam, psi, iota, A, f, L, tb.x[:, :, 0])
    # the closed form itself against the printed worked example (independent of the oracle)
    for name, v in g["links"].items():
        ph = Y[(int(name[0]), int(name[1]))]
        assert abs(float(ph.real) - v["re"]) < 2e-9 * abs(ph) and abs(float(ph.imag) - v["im"]) < 2e-9 * abs(ph)
    for name, v in g["tdi"].items():
        for gi, key in enumerate(("gen1", "gen2")):
            ph = XYZ[name][gi]
            assert abs(float(ph.real) - v[key][0]) < 2e-9 * abs(ph) and abs(float(ph.imag) - v[key][1]) < 2e-9 * abs(ph)
    # the discrete oracle against the closed form
    t = LD(t0) + LD(dt) * np.arange(n).astype(LD)
    wt = LD(2) * np.arccos(LD(-1)) * LD(f) * t
    hp = LD(A) * (1 + np.cos(LD(iota)) ** 2) * np.cos(wt)
    hc = -2 * LD(A) * np.cos(LD(iota)) * np.sin(wt)
    orc = O.Oracle(tb, dt, t0, order)
    y = orc.project(hp, hc, beta, lam, psi)
    mpj, mf1, mb1 = orc.margins(1)
    _, mf2, mb2 = orc.margins(2)
    for s, lk in enumerate(I.LINKS):
        want = _series(Y[lk], w, t)
        assert rel(y[s, mpj:n - mpj], want[mpj:n - mpj]) < tol
        assert np.all(y[s, :mpj] == 0) and np.all(y[s, n - mpj:] == 0)
    for gen, mf, mb in ((1, mf1, mb1), (2, mf2, mb2)):
        for nested in (True, False):
            out = orc.tdi(y, gen, nested=nested, channels=O.CH_XYZ_AET)
            for ch, name in enumerate("XYZ"):
                want = _series(XYZ[name][gen - 1], w, t)
                assert rel(out[ch, mf:n - mb], want[mf:n - mb]) < 10 * tol, (gen, nested, name)
                assert np.all(out[ch, :mf] == 0) and np.all(out[ch, n - mb:] == 0)
            # eq. 21 on the phasors; |A|, |E|, |T| against the printed values, series against the oracle
            Xp, Yp, Zp = (XYZ[c][gen - 1] for c in "XYZ")
            aet = [(Zp - Xp) / mp.sqrt(2), (Xp - 2 * Yp + Zp) / mp.sqrt(6), (Xp + Yp + Zp) / mp.sqrt(3)]
            for c in range(3):
                printed = g["aet_abs"][f"gen{gen}"][c]
                assert abs(float(abs(aet[c])) - printed) < 1e-8 * printed
            for c in range(2):   # T is 3e-5 of A in this exactly-equal-arm case: not a parity case
                assert rel(out[3 + c, mf:n - mb], _series(aet[c], w, t)[mf:n - mb]) < 10 * tol
    if order == 25:   # printed spot values at t = 12345 s = t0 + 1234 dt
        ns = 1234
        X1 = orc.tdi(y, 1)[0, ns]
        X2 = orc.tdi(y, 2)[0, ns]
        assert abs(float(y[0, ns]) - g["spot"]["y12"]) < 1e-10 * abs(g["spot"]["y12"])
        assert abs(float(X1) - g["spot"]["X1"]) < 1e-10 * abs(g["spot"]["X1"])
        assert abs(float(X2) - g["spot"]["X2"]) < 1e-10 * abs(g["spot"]["X2"])


# ------------------------------------------------------------------------------ P5
def _gb_mp(t, A, f0, fdot, iota, phi0):
    ph = mp.mpf(phi0) + 2 * mp.pi * (mp.mpf(f0) * t + mp.mpf(fdot) * t * t / 2)
    return (mp.mpf(A) * (1 + mp.cos(iota) ** 2) * mp.cos(ph), -2 * mp.mpf(A) * mp.cos(iota) * mp.sin(ph))


def test_p5_brute_force_continuous_time():
    """Direct evaluation of eq. 16 and eqs. 17-20 at exact delayed times (no interpolation, no
    spline: the orbit channels are cubics) against the discrete oracle on a tiny input."""
    mp.mp.dps = 40
    rng = np.random.default_rng(5)
    static = I.static_positions([0.0])[:, :, 0]
    # slowly moving spacecraft and strongly drifting light times (so NESTED != SUM visibly)
    cx = [[[float(static[i, a]), 30.0 * rng.normal(), 1e-5 * rng.normal(), 1e-11 * rng.normal()] for a in range(3)]
          for i in range(3)]
    cl = [[8.3 + 0.05 * rng.normal(), 3e-6 * rng.normal(), 1e-11 * rng.normal(), 1e-17 * rng.normal()]
          for _ in range(6)]
    dt, t0, n, order = 10.0, 20000.0, 700, 25
    tb = _poly_table(14, 4000.0, cx, cl)
    src = I.Source(A=1e-22, f0=2e-3, fdot=3e-9, iota=0.5, phi0=0.7, psi=0.3, beta=0.2, lam=1.0)
    hp = np.empty(n, dtype=LD)
    hc = np.empty(n, dtype=LD)
    for i in range(n):
        a, b = _gb_mp(mp.mpf(t0) + mp.mpf(dt) * i, src.A, src.f0, src.fdot, src.iota, src.phi0)
        hp[i], hc[i] = mp2ld(a), mp2ld(b)
    orc = O.Oracle(tb, dt, t0, order)
    y = orc.project(hp, hc, src.beta, src.lam, src.psi)

    polyv = lambda co, t: sum(mp.mpf(c) * t ** k for k, c in enumerate(co))
    cb, sb, cl_, sl = mp.cos(src.beta), mp.sin(src.beta), mp.cos(src.lam), mp.sin(src.lam)
    k = [-cb * cl_, -cb * sl, -sb]
    u = [sl, -cl_, mp.mpf(0)]
    v = [-sb * cl_, -sb * sl, cb]
    dot = lambda a, b: sum(p * q for p, q in zip(a, b))
    c2, s2 = mp.cos(2 * mp.mpf(src.psi)), mp.sin(2 * mp.mpf(src.psi))

    def H(t, xp, xc):      # eq. 11 with the eq. 9 rotation
        a, b = _gb_mp(t, src.A, src.f0, src.fdot, src.iota, src.phi0)
        return xp * (c2 * a - s2 * b) + xc * (s2 * a + c2 * b)

    def y_direct(i, j, t):  # eq. 16, all orbit quantities at reception time t
        xi = [polyv(cx[i - 1][a], t) for a in range(3)]
        xj = [polyv(cx[j - 1][a], t) for a in range(3)]
        d = [p - q for p, q in zip(xi, xj)]
        nrm = mp.sqrt(dot(d, d))
        nv = [q / nrm for q in d]
        xp = dot(u, nv) ** 2 - dot(v, nv) ** 2
        xc = 2 * dot(u, nv) * dot(v, nv)
        Lij = polyv(cl[I.LINKS.index((i, j))], t)
        return (H(t - Lij - dot(k, xj) / C, xp, xc) - H(t - dot(k, xi) / C, xp, xc)) / (2 * (1 - dot(k, nv)))

    mpj, mf, mb = orc.margins(2)
    picks = [mf, mf + 1, n // 2, n - mb - 1]
    ymax = float(np.abs(y).max())
    for nn in picks:
        t = mp.mpf(t0) + mp.mpf(dt) * nn
        for s, (i, j) in enumerate(I.LINKS):
            assert abs(ld2mp(y[s, nn]) - y_direct(i, j, t)) < 1e-13 * ymax

    terms = [(+1, "", 13), (+1, "13", 31), (+1, "131", 12), (+1, "1312", 21),
             (-1, "", 12), (-1, "12", 21), (-1, "121", 13), (-1, "1213", 31),
             (+1, "13121", 12), (+1, "131212", 21), (+1, "1312121", 13), (+1, "13121213", 31),
             (-1, "12131", 13), (-1, "121313", 31), (-1, "1213131", 12), (-1, "12131312", 21)]

    def tdi_direct(ch, gen, nested, t):
        r = lambda i: (i - 1 + ch) % 3 + 1
        acc = mp.mpf(0)
        for sign, chain, ser in terms[:8 * gen]:
            d = mp.mpf(0)
            for a in range(len(chain) - 1):
                sl_ = I.LINKS.index((r(int(chain[a])), r(int(chain[a + 1]))))
                d += polyv(cl[sl_], t - d) if nested else polyv(cl[sl_], t)
            acc += sign * y_direct(r(ser // 10), r(ser % 10), t - d)
        return acc

    results = {}
    for gen in (1, 2):
        for nested in (True, False):
            out = orc.tdi(y, gen, nested=nested)
            results[(gen, nested)] = out
            xmax = float(np.abs(out).max())
            for nn in picks[1:3]:
                t = mp.mpf(t0) + mp.mpf(dt) * nn
                for ch in range(3):
                    # analytic y at the delayed time differs from the interpolated discrete y by
                    # interpolation error only (< 1e-14 at order 25, w dt = 0.13)
                    assert abs(ld2mp(out[ch, nn]) - tdi_direct(ch, gen, nested, t)) < 3e-12 * xmax
    # with 3e-6 drift the two chain modes are different definitions (A15): the pin above separates them
    assert rel(results[(2, True)][0, mf:n - mb], results[(2, False)][0, mf:n - mb]) > 1e-7


# ------------------------------------------------------------------------------ P3
def test_p3_laser_noise_suppression():
    """y_ij = p_j(t - L_ij(t)) - p_i(t) from three analytic band-limited series: TDI-2 with NESTED
    delays cancels it to interpolation level; SUM (eq. 20) and TDI-1 do not."""
    dt, order, n = 10.0, 25, 3000
    t0 = 3.0e7
    tb = I.orbit_table("kepler", t0, t0 + n * dt)
    orc = O.Oracle(tb, dt, t0, order)
    par = I.band_limited_noise(3)
    tau = LD(dt) * np.arange(n).astype(LD)               # time since t0, exact
    y = np.zeros((6, n), dtype=LD)
    for s, (i, j) in enumerate(I.LINKS):
        Lij = orc.spline(9 + s, LD(t0) + tau)
        y[s] = I.eval_tones(par, j - 1, tau - Lij) - I.eval_tones(par, i - 1, tau)
    rms_p = float(np.sqrt(np.mean(I.eval_tones(par, 0, tau) ** 2)))
    res = {}
    for gen in (1, 2):
        mpj, mf, mb = orc.margins(gen)
        for nested in (True, False):
            out = orc.tdi(y, gen, nested=nested)
            res[(gen, nested)] = float(np.sqrt(np.mean(out[:, mf:n - mb] ** 2))) / rms_p
    assert res[(2, True)] < 1e-12, res
    assert res[(2, False)] > 1e-10 and res[(1, True)] > 1e-10 and res[(1, False)] > 1e-10, res


# ------------------------------------------------------------------------ P4, P6, P7, P10
@pytest.fixture(scope="module")
def kepler_case():
    w = I.config(2, n=2400, f0=3e-3)
    tb = w.table()
    hp, hc = w.waveform()
    return w, tb, hp, hc


def test_p4_relabelling(kepler_case):
    w, tb, hp, hc = kepler_case
    s = w.sources[0]
    base = O.Oracle(tb, w.dt, w.t0, w.order)
    y0 = base.project(hp, hc, s.beta, s.lam, s.psi)
    x0 = base.tdi(y0, 2)
    mpj, mf, mb = base.margins(2)
    sl = slice(mf, w.n - mb)
    # cyclic: new 1 = old 2, new 2 = old 3, new 3 = old 1  =>  (X, Y, Z)_new = (Y, Z, X)_old
    perm = {1: 2, 2: 3, 3: 1}
    orc = O.Oracle(tb.relabel(perm), w.dt, w.t0, w.order)
    y1 = orc.project(hp, hc, s.beta, s.lam, s.psi)
    for sl_new, (i, j) in enumerate(I.LINKS):
        assert rel(y1[sl_new, sl], y0[I.LINKS.index((perm[i], perm[j])), sl]) < 1e-17
    x1 = orc.tdi(y1, 2)
    for c_new, c_old in ((0, 1), (1, 2), (2, 0)):
        assert rel(x1[c_new, sl], x0[c_old, sl]) < 1e-15
    # reflection 2 <-> 3: X -> -X, Y -> -Z, Z -> -Y  ("up to a sign")
    perm = {1: 1, 2: 3, 3: 2}
    orc = O.Oracle(tb.relabel(perm), w.dt, w.t0, w.order)
    x2 = orc.tdi(orc.project(hp, hc, s.beta, s.lam, s.psi), 2)
    for c_new, c_old in ((0, 0), (1, 2), (2, 1)):
        assert rel(x2[c_new, sl], -x0[c_old, sl]) < 1e-15


def test_p6_aet_orthonormal(kepler_case):
    w, tb, hp, hc = kepler_case
    s = w.sources[0]
    orc = O.Oracle(tb, w.dt, w.t0, w.order)
    out = orc.tdi(orc.project(hp, hc, s.beta, s.lam, s.psi), 2, channels=O.CH_XYZ_AET)
    a = (out[:3] ** 2).sum(axis=0)
    b = (out[3:] ** 2).sum(axis=0)
    assert np.max(np.abs(a - b)) < 1e-17 * a.max()
    # explicit eq. 21 on one sample
    X, Y, Z = out[0], out[1], out[2]
    assert rel(out[3], (Z - X) / np.sqrt(LD(2))) < 1e-17
    assert rel(out[4], (X - 2 * Y + Z) / np.sqrt(LD(6))) < 1e-17
    assert rel(out[5], (X + Y + Z) / np.sqrt(LD(3))) < 1e-15
    only_aet = orc.tdi(orc.project(hp, hc, s.beta, s.lam, s.psi), 2, channels=O.CH_AET)
    assert np.array_equal(only_aet, out[3:])


def test_p7_p10_generation_structure_and_mode_equivalence():
    w = I.config(1, n=2000)                       # EQ orbits, constant equal light times
    tb = w.table()
    s = w.sources[0]
    # smooth long-double waveform: an fp64 phase carries ~1e-11 of broadband rounding noise, on which
    # a cascade of two interpolations legitimately differs from one interpolation by the total delay
    t = LD(w.t0) + LD(w.dt) * np.arange(w.n).astype(LD)
    ph = LD(s.phi0) + 2 * np.arccos(LD(-1)) * (LD(s.f0) * t + LD(s.fdot) * t * t / 2)
    hp = LD(s.A) * (1 + np.cos(LD(s.iota)) ** 2) * np.cos(ph)
    hc = -2 * LD(s.A) * np.cos(LD(s.iota)) * np.sin(ph)
    orc = O.Oracle(tb, w.dt, w.t0, w.order)
    y = orc.project(hp, hc, s.beta, s.lam, s.psi)
    mpj, mf, mb = orc.margins(2)
    sl = slice(mf + 40, w.n - mb - 20)     # the cascade's stencil must stay inside the valid X1
    x1 = orc.tdi(y, 1)
    x2 = orc.tdi(y, 2)
    x2s = orc.tdi(y, 2, nested=False)
    assert rel(x2s[:, sl], x2[:, sl]) < 1e-16                       # P10
    # P7: X2 = X1 - D^4 X1 for constant equal delays (up to interpolation error of the cascade)
    L = tb.ltt[0, 0]
    for ch in range(3):
        delayed = np.array([O.interp(x1[ch], nn, LD(4 * L / w.dt), w.order) for nn in range(sl.start, sl.stop)])
        assert rel(x2[ch, sl], x1[ch, sl] - delayed) < 1e-12
    # gen 1 = first 8 terms of gen 2: remove the 8 extra terms by hand from y
    extra = np.zeros(w.n, dtype=LD)
    chains = [(+1, 4, 0), (+1, 5, 5), (+1, 6, 3), (+1, 7, 2), (-1, 4, 3), (-1, 5, 2), (-1, 6, 0), (-1, 7, 5)]
    for nn in range(sl.start, sl.stop):
        extra[nn] = sum(sg * O.interp(y[slot], nn, LD(k * L / w.dt), w.order) for sg, k, slot in chains)
    assert rel(x2[0, sl] - extra[sl], x1[0, sl]) < 1e-15


# ------------------------------------------------------------------------------ P8
def test_p8_long_wavelength_limit():
    """For wL << 1:  y_ij -> -(L_ij/2) d/dt[xi+ h+ + xix hx](t - k.x_i/c), independent of k.n_ij.
    A flipped n_ij or a swapped difference in eq. 16 breaks this at O(1)."""
    f0 = 1e-5
    w = I.config(2, n=1500, f0=f0)
    src = I.Source(A=1e-22, f0=f0, fdot=0.0, iota=0.8, phi0=0.3, psi=0.4, beta=0.35, lam=2.2)
    tb = w.table()
    hp, hc = I.gb_waveform(w.n, w.dt, w.t0, src.A, src.f0, src.fdot, src.iota, src.phi0)
    orc = O.Oracle(tb, w.dt, w.t0, w.order)
    y = orc.project(hp, hc, src.beta, src.lam, src.psi).astype(float)
    mpj = orc.margins(1)[0]
    nn = np.arange(mpj, w.n - mpj)
    t = w.t0 + w.dt * nn
    x = I.kepler_positions(t)
    cb, sb, cl, sl = np.cos(src.beta), np.sin(src.beta), np.cos(src.lam), np.sin(src.lam)
    k = np.array([-cb * cl, -cb * sl, -sb])
    u0 = np.array([sl, -cl, 0.0])
    v0 = np.array([-sb * cl, -sb * sl, cb])
    c2, s2 = np.cos(2 * src.psi), np.sin(2 * src.psi)
    ci = np.cos(src.iota)
    for s, (i, j) in enumerate(I.LINKS):
        d = x[i - 1] - x[j - 1]
        n_ij = d / np.linalg.norm(d, axis=0)
        xp = (u0 @ n_ij) ** 2 - (v0 @ n_ij) ** 2
        xc = 2 * (u0 @ n_ij) * (v0 @ n_ij)
        tr = t - (k @ x[i - 1]) / C
        ph = src.phi0 + 2 * np.pi * f0 * tr
        dhp = -src.A * (1 + ci * ci) * np.sin(ph) * 2 * np.pi * f0       # analytic time derivatives
        dhc = -2 * src.A * ci * np.cos(ph) * 2 * np.pi * f0
        dH = xp * (c2 * dhp - s2 * dhc) + xc * (s2 * dhp + c2 * dhc)
        Lij = np.linalg.norm(d, axis=0) / C
        want = -0.5 * Lij * dH
        assert rel(y[s, nn], want) < 2e-3, s


# ------------------------------------------------------------------------------ margins
def test_margins_cover_every_stencil():
    """Reading A8: for every valid sample, every tap index of every interpolation lies in [0, n)."""
    for cfg, kw in ((1, {}), (2, {"n": 4000}), (4, {"n": 4000})):
        w = I.config(cfg, **kw)
        tb = w.table()
        orc = O.Oracle(tb, w.dt, w.t0, w.order)
        p = (w.order + 1) // 2
        tq = np.linspace(w.t0, w.t0 + w.n * w.dt, 400)
        r_max = max(float(np.sqrt(sum(orc.spline(3 * i + a, tq) ** 2 for a in range(3))).max()) for i in range(3))
        l_max = max(float(orc.spline(9 + s, tq).max()) for s in range(6))
        mpj, mf, mb = orc.margins(w.tdi_gen)
        reach_proj = int(np.ceil((r_max / C + l_max) / w.dt)) + p
        assert mpj >= reach_proj
        nl = 3 if w.tdi_gen == 1 else 7
        assert mf >= mpj + int(np.ceil(nl * l_max / w.dt)) + p     # TDI reads only valid y
        assert mb >= mpj + p


def test_margins_are_reading_a8():
    """Reading A8 itself (the paper is silent on edges): from the TABLE maxima
    R_max = max |x_i| and L_max = max L_ij over the knots,
        M_proj = ceil((1.001 R_max/c + 1.001 L_max)/dt) + p + 2,
        M_front = M_proj + ceil(G 1.001 L_max/dt) + p + 2 (G = 4 | 8),  M_back = M_proj + p + 2,
    so a joint drift of the 1.001 factors or of the `+ p + 2` on both sides (oracle and library assert equality with
    each other on the GPU) cannot go unnoticed.  The survey prints M_proj = 67 for Keplerian orbits at dt = 10 s,
    order 25 (R_max/c = 501.4 s, L_max = 8.34 s)."""
    for cfg, kw in ((1, {}), (2, {"n": 4000}), (3, {"n": 4000, "batch": 1}), (4, {"n": 4000}), (5, {"n": 4000})):
        w = I.config(cfg, **kw)
        tb = w.table()
        orc = O.Oracle(tb, w.dt, w.t0, w.order)
        p = (w.order + 1) // 2
        x = np.asarray(tb.x, dtype=np.float64).reshape(3, 3, -1)
        r_max = float(np.sqrt((x ** 2).sum(axis=1)).max())
        l_max = float(np.asarray(tb.ltt).max())
        m_proj = math.ceil((1.001 * r_max / C + 1.001 * l_max) / w.dt) + p + 2
        for gen, G in ((1, 4), (2, 8)):
            want = (m_proj, m_proj + math.ceil(G * 1.001 * l_max / w.dt) + p + 2, m_proj + p + 2)
            assert orc.margins(gen) == want, (cfg, gen)
    w = I.config(2)     # the whole year of knots: R_max reaches the aphelion
    assert O.Oracle(w.table(), w.dt, w.t0, w.order).margins(2)[0] == 67
