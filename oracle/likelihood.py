"""CPU ORACLE of the likelihood stage: noise-weighted inner product, log-likelihood,
SNR, overlap.  TEST INFRASTRUCTURE — imported only by tests/ (never by paper_2204_06633_b200).

Plain statement of PAPER.md eqs. 2-4 and 22:

    <a|b> = 4 Re int_0^inf a~(f)^* b~(f) / S_n(f) df          summed over the channels A, E, T       (2), (22)
    log L = -1/2 <d - h | d - h>                                                                      (3)
    rho_opt = sqrt(<h|h>),  rho_ex = <d|h> / sqrt(<h|h>),  overlap = rho_ex / sqrt(<s|s>)             (4)

Discretisation (the paper does not print one; DESIGN.md §3 reading A17): a~(f_k) = dt * sum_n a[n] exp(-2 pi i k n
/ N), f_k = k / (N dt), df = 1 / (N dt), the integral is the sum over k = 1 .. N/2 (the DC bin, where S_n
diverges, is left out).  The FFT is numpy's (a library routine used as one step, fp64); the weighted sum is
accumulated in long double.

Pins (tests/test_oracle_likelihood.py): a sinusoid on a bin centre has <a|a> = A^2 T / S_n(f) (textbook
monochromatic SNR); bilinearity and symmetry; <a|a> with a flat PSD equals the time-domain Parseval sum;
log L = 0 iff d = h; overlap of a signal with itself is 1.
"""
import numpy as np

LD = np.longdouble


def to_frequency(x, dt):
    """a~(f_k) for k = 0 .. N/2 along the last axis (library FFT), in the convention above."""
    return dt * np.fft.rfft(np.asarray(x, dtype=np.float64), axis=-1)


def inner_product(fa, fb, psd, dt, n):
    """<a|b> of eq. 2 summed over channels (eq. 22).  fa, fb: [..., n_ch, nf] complex from `to_frequency`;
    psd: [n_ch, nf] one-sided S_n(f_k) (entry 0 unused); n = number of time samples."""
    df = LD(1) / (LD(n) * LD(dt))
    re = fa.real.astype(LD) * fb.real.astype(LD) + fa.imag.astype(LD) * fb.imag.astype(LD)   # Re(a^* b)
    w = re[..., 1:] / np.asarray(psd, dtype=LD)[..., 1:]
    return LD(4) * df * w.sum(axis=(-1, -2))


def log_likelihood(fd, fh, psd, dt, n):
    """eq. 3 with the proportionality constant 1."""
    r = fd - fh
    return -inner_product(r, r, psd, dt, n) / LD(2)


def snr_opt(fh, psd, dt, n):
    return np.sqrt(inner_product(fh, fh, psd, dt, n))


def overlap(fd, fh, psd, dt, n):
    """rho_ex / sqrt(<d|d>) with no additive noise (d = s)."""
    return inner_product(fd, fh, psd, dt, n) / np.sqrt(inner_product(fh, fh, psd, dt, n) *
                                                       inner_product(fd, fd, psd, dt, n))
