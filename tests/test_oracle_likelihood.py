"""Pins of the likelihood oracle (oracle/likelihood.py; eqs. 2-4, 22) against what the mathematics
fixes — none of them re-types the oracle's formula."""
import numpy as np

from oracle import likelihood as lk
from harness import inputs

LD = np.longdouble


def _setup(n=8192, dt=10.0):
    f = np.fft.rfftfreq(n, dt)
    return n, dt, f, inputs.psd_standin(f), dt * np.arange(n)


def test_monochromatic_snr_closed_form():
    """A sinusoid on a bin centre: <a|a> = A^2 T / S_n(f) (textbook SNR of a monochromatic source); a wrong
    factor (2 vs 4), a wrong df or dt, or a two-sided PSD would all miss it."""
    n, dt, f, psd, t = _setup()
    for k, ch, A, ph in ((37, 0, 1e-21, 0.3), (1500, 1, 3e-22, 2.0), (4000, 2, 5e-21, -1.0)):
        x = np.zeros((3, n))
        x[ch] = A * np.cos(2 * np.pi * f[k] * t + ph)
        fa = lk.to_frequency(x, dt)
        want = LD(A) ** 2 * n * dt / LD(psd[ch, k])
        got = lk.inner_product(fa, fa, psd, dt, n)
        assert abs(got - want) < 1e-10 * want


def test_parseval_with_flat_psd():
    """S_n = 1 on every bin: <a|a> = 2 dt sum a[n]^2 up to the DC and Nyquist bins (removed from the signal)."""
    n, dt, f, _, t = _setup(4096)
    rng = np.random.default_rng(0)
    x = rng.normal(size=(3, n))
    X = np.fft.rfft(x, axis=-1)
    X[:, 0] = 0
    X[:, -1] = 0
    x = np.fft.irfft(X, n=n, axis=-1)
    fa = lk.to_frequency(x, dt)
    got = lk.inner_product(fa, fa, np.ones((3, f.size)), dt, n)
    want = 2 * dt * (x.astype(LD) ** 2).sum()
    assert abs(got - want) < 1e-12 * want


def test_bilinear_symmetric_and_channel_sum():
    n, dt, f, psd, t = _setup(2048)
    rng = np.random.default_rng(1)
    a, b, c = (lk.to_frequency(rng.normal(size=(3, n)), dt) for _ in range(3))
    ip = lambda u, v: lk.inner_product(u, v, psd, dt, n)
    assert abs(ip(a, b) - ip(b, a)) < 1e-14 * abs(ip(a, a))
    assert abs(ip(a + 2 * c, b) - (ip(a, b) + 2 * ip(c, b))) < 1e-12 * abs(ip(a, a))
    per_channel = sum(lk.inner_product(a[i:i + 1], b[i:i + 1], psd[i:i + 1], dt, n) for i in range(3))
    assert abs(ip(a, b) - per_channel) < 1e-14 * abs(ip(a, a))      # eq. 22


def test_loglikelihood_snr_overlap():
    """eq. 3: log L = -(<d|d> + <h|h> - 2 <d|h>)/2, zero iff h = d; eq. 4: rho_ex = rho_opt when h = d, overlap
    of a signal with itself is 1 and with an orthogonal one (another bin) is 0."""
    n, dt, f, psd, t = _setup(4096)
    mk = lambda k, A: lk.to_frequency(np.stack([A * np.cos(2 * np.pi * f[k] * t)] * 3), dt)
    d, h = mk(100, 1e-21), mk(100, 1.1e-21)
    ll = lk.log_likelihood(d, h, psd, dt, n)
    ip = lambda u, v: lk.inner_product(u, v, psd, dt, n)
    assert abs(ll + (ip(d, d) + ip(h, h) - 2 * ip(d, h)) / 2) < 1e-12 * abs(ip(d, d))
    assert lk.log_likelihood(d, d, psd, dt, n) == 0
    assert ll < 0
    assert abs(lk.overlap(d, d, psd, dt, n) - 1) < 1e-15
    assert abs(lk.overlap(d, h, psd, dt, n) - 1) < 1e-12         # same shape, other amplitude
    assert abs(lk.overlap(d, mk(200, 1e-21), psd, dt, n)) < 1e-10
    assert abs(lk.snr_opt(d, psd, dt, n) ** 2 - ip(d, d)) < 1e-12 * ip(d, d)
