"""Seeded synthetic input generators (orbit tables, waveforms, config descriptors).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none
of the method's arithmetic: no Lagrange weights, no spline fit, no projection, no
TDI.  It only manufactures the *inputs* of `lr_create / lr_project / lr_tdi`:

* orbit tables (spacecraft positions and the six light travel times on uniform
  knots) standing in for the paper's "LISA Orbits" products, which are not in the
  container (§IV.D);
* Galactic-binary and chirp strain series h+(t), h×(t) sampled at the SSB
  (eqs. 5-9; BASELINE.json `configs`);
* the five workload descriptors of BASELINE.json `configs`.

Everything is numpy fp64 and deterministic from a seed.  The recipe is restated in
DESIGN.md ("Input recipe").  Link order everywhere: [12, 23, 31, 13, 32, 21]; link
ij is received on spacecraft i and emitted by spacecraft j.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

C_LIGHT = 299792458.0            # m/s, exact
AU = 149597870700.0              # m
YEAR = 365.25 * 86400.0          # s
DAY = 86400.0
ARM = 2.5e9                      # nominal armlength, m
MSUN_S = 4.925490947641267e-06   # G*Msun/c^3 in seconds

# (receiver i, emitter j), 1-based, in slot order [12, 23, 31, 13, 32, 21]
LINKS = ((1, 2), (2, 3), (3, 1), (1, 3), (3, 2), (2, 1))


# --------------------------------------------------------------------------- orbits
def eq_positions(t):
    """Equal-armlength analytic orbits, first order in e.

    Returns x[3 spacecraft, 3 xyz, len(t)] in metres.  Spacecraft are indexed
    clockwise seen from +z, hence the minus sign in `b`.
    """
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    om = 2.0 * np.pi / YEAR
    e = ARM / (2.0 * np.sqrt(3.0) * AU)
    a = om * t
    out = np.empty((3, 3, t.size))
    for n in range(3):
        b = -2.0 * np.pi * n / 3.0
        out[n, 0] = AU * np.cos(a) + 0.5 * e * AU * (np.cos(2 * a - b) - 3.0 * np.cos(b))
        out[n, 1] = AU * np.sin(a) + 0.5 * e * AU * (np.sin(2 * a - b) - 3.0 * np.sin(b))
        out[n, 2] = -np.sqrt(3.0) * e * AU * np.cos(a - b)
    return out


def kepler_positions(t):
    """Eccentric Keplerian orbits, three spacecraft, one-year period.

    e ~ 0.0048, armlength breathing of a fraction of a percent.
    """
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    om = 2.0 * np.pi / YEAR
    alpha = ARM / (2.0 * AU)
    nu = np.pi / 3.0 + 0.625 * alpha
    e = np.sqrt(1.0 + (4.0 / np.sqrt(3.0)) * alpha * np.cos(nu) + (4.0 / 3.0) * alpha**2) - 1.0
    tan_i = (2.0 / np.sqrt(3.0)) * alpha * np.sin(nu) / (1.0 + (2.0 / np.sqrt(3.0)) * alpha * np.cos(nu))
    inc = np.arctan(tan_i)
    out = np.empty((3, 3, t.size))
    for n in range(3):
        sig = -2.0 * np.pi * n / 3.0
        m = om * t - sig
        psi = m.copy()
        for _ in range(12):  # Newton on psi + e sin(psi) = m
            psi = psi - (psi + e * np.sin(psi) - m) / (1.0 + e * np.cos(psi))
        xo = AU * (np.cos(psi) + e) * np.cos(inc)
        yo = AU * np.sqrt(1.0 - e * e) * np.sin(psi)
        zo = AU * (np.cos(psi) + e) * np.sin(inc)
        out[n, 0] = np.cos(sig) * xo - np.sin(sig) * yo
        out[n, 1] = np.sin(sig) * xo + np.cos(sig) * yo
        out[n, 2] = zo
    return out


def make_perturbed_positions(seed):
    """Keplerian orbits plus seeded low-frequency perturbations (BASELINE.json config 4).

    A common-mode term of relative amplitude 1e-3 au and a per-spacecraft term of
    2e-4 au, each a sum of five sinusoids with periods in [0.3, 3] years.
    Returns a function t -> x[3,3,len(t)].
    """
    rng = np.random.default_rng(seed)

    def draw():
        return (rng.uniform(0.3, 3.0, size=(3, 5)) * YEAR,          # periods per axis
                rng.normal(size=(3, 5)) / np.sqrt(5.0),             # amplitudes
                rng.uniform(0.0, 2.0 * np.pi, size=(3, 5)))         # phases

    common = draw()
    per_sc = [draw() for _ in range(3)]

    def series(par, t):
        per, amp, ph = par
        arg = 2.0 * np.pi * t[None, None, :] / per[:, :, None] + ph[:, :, None]
        return (amp[:, :, None] * np.sin(arg)).sum(axis=1)           # [3 xyz, len(t)]

    def fn(t):
        t = np.atleast_1d(np.asarray(t, dtype=np.float64))
        x = kepler_positions(t)
        cm = 1e-3 * AU * series(common, t)
        for n in range(3):
            x[n] += cm + 2e-4 * AU * series(per_sc[n], t)
        return x

    return fn


def static_positions(t):
    """Static equilateral triangle of SURVEY.md's worked example (pin P2)."""
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    r = ARM / np.sqrt(3.0)
    e1 = np.array([0.0, 1.0, 0.0])
    e2 = np.array([-0.5, 0.0, np.sqrt(3.0) / 2.0])
    centre = np.array([AU, 0.0, 0.0])
    out = np.empty((3, 3, t.size))
    for n in range(3):
        th = -2.0 * np.pi * n / 3.0
        out[n] = (centre + r * (np.cos(th) * e1 + np.sin(th) * e2))[:, None]
    return out


def light_times(pos_fn, t, iters=4):
    """Flat-space light travel times L_ij(t) = |x_i(t) - x_j(t - L_ij)|/c by fixed point.

    Stand-in for the post-Minkowskian light times of PAPER.md:240; gives L_ij != L_ji.
    Returns ltt[6, len(t)] in seconds, link order LINKS.
    """
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    xr = pos_fn(t)
    out = np.empty((6, t.size))
    for s, (i, j) in enumerate(LINKS):
        L = np.full(t.size, ARM / C_LIGHT)
        for _ in range(iters):
            xe = pos_fn(t - L)[j - 1]
            L = np.linalg.norm(xr[i - 1] - xe, axis=0) / C_LIGHT
        out[s] = L
    return out


@dataclasses.dataclass
class OrbitTable:
    """Host-side orbit table handed to `lr_create` (include/lr.h `lr_orbits`)."""
    t_start: float
    knot_dt: float
    x: np.ndarray      # [3, 3, n_knots] metres
    ltt: np.ndarray    # [6, n_knots] seconds

    @property
    def n_knots(self):
        return self.x.shape[-1]

    def relabel(self, perm):
        """Table with spacecraft relabelled: new spacecraft a is old spacecraft perm[a] (1-based)."""
        x = np.stack([self.x[perm[a] - 1] for a in (1, 2, 3)])
        ltt = np.empty_like(self.ltt)
        for s, (i, j) in enumerate(LINKS):
            ltt[s] = self.ltt[LINKS.index((perm[i], perm[j]))]
        return OrbitTable(self.t_start, self.knot_dt, np.ascontiguousarray(x), ltt)


_POS = {"eq": eq_positions, "kepler": kepler_positions, "static": static_positions}


def orbit_table(kind, t_begin, t_end, knot_dt=DAY, pad=2 * DAY, seed=0, const_ltt=None):
    """Orbit table on uniform knots covering [t_begin - pad, t_end + pad].

    kind: "eq" | "kepler" | "static" | "perturbed".  `const_ltt` (seconds) replaces the
    fixed-point light times by one constant for all six links.
    """
    pos_fn = make_perturbed_positions(seed) if kind == "perturbed" else _POS[kind]
    k0 = math.floor((t_begin - pad) / knot_dt)
    k1 = math.ceil((t_end + pad) / knot_dt)
    tk = np.arange(k0, k1 + 1, dtype=np.float64) * knot_dt
    x = np.ascontiguousarray(pos_fn(tk))
    if const_ltt is not None:
        ltt = np.full((6, tk.size), float(const_ltt))
    else:
        ltt = light_times(pos_fn, tk)
    return OrbitTable(float(tk[0]), float(knot_dt), x, np.ascontiguousarray(ltt))


# ------------------------------------------------------------------------ waveforms
def gb_waveform(n, dt, t0, A, f0, fdot, iota, phi0):
    """Galactic binary of BASELINE.json configs: Phi = phi0 + 2 pi (f0 t + fdot t^2 / 2),
    h+ = A (1 + cos^2 iota) cos Phi, hx = -2 A cos(iota) sin Phi."""
    t = t0 + dt * np.arange(n, dtype=np.float64)
    phase = phi0 + 2.0 * np.pi * (f0 * t + 0.5 * fdot * t * t)
    ci = np.cos(iota)
    return A * (1.0 + ci * ci) * np.cos(phase), -2.0 * A * ci * np.sin(phase)


def tukey(n, frac):
    w = np.ones(n)
    m = int(frac * n)
    if m > 0:
        ramp = 0.5 * (1.0 - np.cos(np.pi * np.arange(m) / m))
        w[:m] = ramp
        w[n - m:] = ramp[::-1]
    return w


def chirp_waveform(n, dt, t0, mchirp_msun, iota, phi_c, f_end=1e-2, f_lo=1e-4, amp_end=1e-21):
    """Leading-order post-Newtonian inspiral (BASELINE.json config 5).

    t_c is chosen so that f(t_end) = f_end; amplitude ~ f^(2/3) normalised to `amp_end`
    at the end; 5 % Tukey tapers, the leading one starting where f crosses `f_lo`.
    """
    M = mchirp_msun * MSUN_S
    t = t0 + dt * np.arange(n, dtype=np.float64)
    tau_end = 5.0 / 256.0 * M ** (-5.0 / 3.0) * (np.pi * f_end) ** (-8.0 / 3.0)
    tau = tau_end + (t[-1] - t)
    f = (1.0 / np.pi) * (5.0 / (256.0 * tau)) ** 0.375 * M ** (-0.625)
    phase = phi_c - 2.0 * (tau / (5.0 * M)) ** 0.625
    amp = amp_end * (f / f_end) ** (2.0 / 3.0)
    i0 = int(np.argmax(f >= f_lo))
    win = np.zeros(n)
    win[i0:] = tukey(n - i0, 0.05)
    ci = np.cos(iota)
    return amp * win * (1.0 + ci * ci) * np.cos(phase), -2.0 * amp * win * ci * np.sin(phase)


def gb_waveform_device(srcs, n, dt, t0, device):
    """The configs' GB waveform family for a list of sources, evaluated with torch ON THE DEVICE (input generation
    only: config 3's chunks of 64 templates x 1.58e6 samples are made here instead of on the host).  Returns
    (h_plus, h_cross), CUDA float64 [len(srcs), n].  Rounding differs from `gb_waveform` (torch vs numpy cos):
    whoever needs the oracle's view of these inputs copies THESE arrays back."""
    import torch
    t = t0 + dt * torch.arange(n, dtype=torch.float64, device=device)
    hp = torch.empty((len(srcs), n), dtype=torch.float64, device=device)
    hc = torch.empty_like(hp)
    for b, s in enumerate(srcs):
        ph = s.phi0 + 2.0 * np.pi * (s.f0 * t + 0.5 * s.fdot * t * t)
        ci = np.cos(s.iota)
        hp[b] = s.A * (1.0 + ci * ci) * torch.cos(ph)
        hc[b] = -2.0 * s.A * ci * torch.sin(ph)
    return hp, hc


def band_limited_noise(seed, n_series=3, n_tones=40, f_max=5e-3):
    """Parameters of `n_series` independent sums of sinusoids (laser-noise pin P3).

    Returns (freq, amp, phase) each [n_series, n_tones]; evaluate analytically with
    `eval_tones` at arbitrary (also extended-precision) times."""
    rng = np.random.default_rng(seed)
    return (rng.uniform(0.02 * f_max, f_max, size=(n_series, n_tones)),
            rng.normal(size=(n_series, n_tones)) / np.sqrt(n_tones),
            rng.uniform(0.0, 2.0 * np.pi, size=(n_series, n_tones)))


# -------------------------------------------------------------------- workload configs
@dataclasses.dataclass
class Source:
    """One template: waveform parameters and sky angles."""
    beta: float
    lam: float
    psi: float
    A: float = 0.0
    f0: float = 0.0
    fdot: float = 0.0
    iota: float = 0.0
    phi0: float = 0.0
    mchirp: float = 0.0      # chirp only


@dataclasses.dataclass
class Workload:
    name: str
    n: int
    dt: float
    t0: float
    order: int
    tdi_gen: int
    orbit_kind: str
    orbit_seed: int
    const_ltt: float | None
    sources: list
    kind: str = "gb"         # "gb" | "chirp"
    channels: str = "XYZ"

    def table(self):
        return orbit_table(self.orbit_kind, self.t0, self.t0 + self.n * self.dt,
                           seed=self.orbit_seed, const_ltt=self.const_ltt)

    def waveform(self, b=0):
        s = self.sources[b]
        if self.kind == "chirp":
            return chirp_waveform(self.n, self.dt, self.t0, s.mchirp, s.iota, s.phi0)
        return gb_waveform(self.n, self.dt, self.t0, s.A, s.f0, s.fdot, s.iota, s.phi0)


def draw_gb(rng, f0=None):
    """One GB with the prior shapes of PAPER.md:291-300 (Table I) on BASELINE.json's ranges."""
    lf = rng.uniform(-4.0, -2.0)
    s = Source(
        f0=10.0 ** lf if f0 is None else f0,
        fdot=10.0 ** rng.uniform(-19.0, -15.0),
        A=10.0 ** rng.uniform(-23.0, -21.0),
        iota=float(np.arccos(rng.uniform(-1.0, 1.0))),
        beta=float(np.arcsin(rng.uniform(-1.0, 1.0))),
        lam=rng.uniform(0.0, 2.0 * np.pi),
        phi0=rng.uniform(0.0, 2.0 * np.pi),
        psi=rng.uniform(0.0, np.pi),
    )
    return s


FIG3_SOURCE = Source(A=1e-22, f0=1e-2, fdot=1.4e-14, iota=1.11, phi0=4.58, psi=0.45, lam=5.23, beta=1.23)
TINY_SOURCE = Source(A=1e-22, f0=2e-3, fdot=1e-17, iota=0.5, phi0=0.7, psi=0.3, beta=0.2, lam=1.0)


def config(i, *, batch=None, n=None, f0=None, t0=3.0e6):
    """Workload descriptor for BASELINE.json `configs[i-1]`, i in 1..5.

    `n`, `batch` shrink the case for parity tests; `f0` pins the GB frequency (the
    1e-4 / 1e-3 / 1e-2 Hz strata).  t0 is the time of sample 0.
    """
    if i == 1:   # Tiny: EQ orbits, constant equal light times, TDI-1
        return Workload("tiny", n or 10640, 10.0, t0, 25, 1, "eq", 0, ARM / C_LIGHT, [TINY_SOURCE])
    if i == 2:   # one year, Keplerian, TDI-2 XYZ+AET
        rng = np.random.default_rng(2204)
        return Workload("year", n or 3153600, 10.0, t0, 25, 2, "kepler", 0, None,
                        [draw_gb(rng, f0)], channels="XYZ_AET")
    if i == 3:   # MCMC batch around the Fig. 3 source
        rng = np.random.default_rng(633)
        B = batch or 1024
        fid = FIG3_SOURCE
        srcs = []
        for _ in range(B):
            g = 1.0 + 1e-4 * rng.normal(size=8)
            srcs.append(Source(A=fid.A * g[0], f0=(f0 or fid.f0) * g[1], fdot=fid.fdot * g[2], iota=fid.iota * g[3],
                               phi0=fid.phi0 * g[4], psi=fid.psi * g[5], lam=fid.lam * g[6], beta=fid.beta * g[7]))
        return Workload("batch", n or 1576800, 10.0, t0, 25, 2, "kepler", 0, None, srcs, channels="AET")
    if i == 4:   # numerical-style orbits, 4 years at 5 s, order 41
        src = Source(A=1e-22, f0=f0 or 2e-3, fdot=1.2e-17, iota=1.11, phi0=4.58, psi=0.45, lam=5.23, beta=1.2)
        # seed 45 drew an L12 range of 0.497 s, outside the paper's ESA-like 0.1-0.4 s window
        # (PAPER.md:249 quotes 0.232 s); the recipe redraws with the next seed: 46 gives 0.320 s.
        return Workload("4yr", n or 25228800, 5.0, t0, 41, 2, "perturbed", 46, None, [src])
    if i == 5:   # chirp
        rng = np.random.default_rng(9)
        mc = 10.0 ** rng.uniform(5.0, 6.0)
        src = Source(beta=float(np.arcsin(rng.uniform(-1, 1))), lam=rng.uniform(0, 2 * np.pi),
                     psi=rng.uniform(0, np.pi), iota=float(np.arccos(rng.uniform(-1, 1))),
                     phi0=rng.uniform(0, 2 * np.pi), mchirp=mc)
        return Workload("chirp", n or 1555200, 5.0, t0, 25, 2, "kepler", 0, None, [src], kind="chirp")
    raise ValueError(i)


def eval_tones(par, k, t):
    """Series k of `band_limited_noise` at times t (any float dtype, e.g. np.longdouble)."""
    freq, amp, ph = par
    t = np.asarray(t)
    two_pi = 2 * np.arccos(t.dtype.type(-1)) if t.dtype == np.longdouble else 2.0 * np.pi
    out = np.zeros_like(t)
    for f, a, p in zip(freq[k], amp[k], ph[k]):
        out = out + t.dtype.type(a) * np.sin(two_pi * t.dtype.type(f) * t + t.dtype.type(p))
    return out


# ------------------------------------------------------------------------------- noise PSD (stand-in)
def psd_standin(f, tdi_gen=2, arm_s=ARM / C_LIGHT):
    """One-sided noise PSD S_n(f) of the TDI channels A, E, T as [3, len(f)] — a smooth analytic STAND-IN for
    the "SciRDv1" curve of the LDC `tdi` package, which is not in the container.  Shape: test-mass
    acceleration noise (3e-15 m/s^2/rtHz, reddened below 0.4 mHz) and optical-metrology noise (15 pm/rtHz,
    reddened below 2 mHz) in relative-frequency units, through the equal-arm Michelson transfer
    16 sin^2(w L) [S_oms + (3 + cos 2wL) S_acc] (x 4 sin^2(2 w L) for generation 2), with T less sensitive
    than A, E at low frequency.  Only its smoothness and dynamic range matter for the tests; entry f = 0 is inf."""
    f = np.asarray(f, dtype=np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        w = 2.0 * np.pi * f
        s_acc = (3e-15 / (w * C_LIGHT)) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
        s_oms = (15e-12 * w / C_LIGHT) ** 2 * (1.0 + (2e-3 / f) ** 4)
        x = w * arm_s
        gen = 4.0 * np.sin(2.0 * x) ** 2 if tdi_gen == 2 else 1.0
        floor = 1e-6   # keeps the zeros of the transfer function (f = k / 2L) finite
        tr = 16.0 * (np.sin(x) ** 2 + floor) * (gen + floor if tdi_gen == 2 else 1.0)
        ae = tr * (s_oms + (3.0 + np.cos(2.0 * x)) * s_acc)
        tt = tr * (s_oms + 8.0 * (np.sin(0.5 * x) ** 2 + floor) * s_acc) * (2.0 + np.cos(x))
    out = np.stack([ae, ae, tt])
    out[:, f == 0] = np.inf
    return out
