"""GPU parity of the template generator (lr_gb_waveform, lr_response_gb, PAPER.md
eqs. 5-9) against oracle/waveform.py and against the h -> out path."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from oracle import waveform as owf
from harness import inputs
from parity_util import CH_NAMES, ORC_CH, assert_parity, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lr():
    import paper_2204_06633_b200 as pkg
    return pkg


def _templates():
    """Four binaries: the configs' form (fddot = 0), the paper's form (eqs. 8, 9), a fast chirper, a late phase."""
    out = []
    a = owf.amplitudes_config(1.0e-22, 0.5)
    out.append((a[0], a[1], 3.0e-3, 1.0e-16, 0.0, 0.7))
    a = owf.amplitudes_paper(2.3e-22, 1.1)
    out.append((a[0], a[1], 5.1e-3, 3.0e-15, owf.fddot_eq8(5.1e-3, 3.0e-15), 2.9))
    out.append((1.0e-21, -0.4e-21, 2.0e-2, 7.0e-13, owf.fddot_eq8(2.0e-2, 7.0e-13), -1.3))
    out.append((1.0, 1.0, 1.0e-4, 0.0, 0.0, 6.0))
    return np.array(out)


@pytest.mark.parametrize("t0", [0.0, 3.1e7, 1.2e8 + 0.123])
def test_gb_waveform_against_exact_phase_oracle(lr, t0):
    """Every sample of four templates within 4e-15 of the amplitude (rounding of the angle 2 pi frac + phi0, |angle| < 10, and of sincos) of the exact-phase oracle — after up to
    2.4e6 cycles, where a phase formed in fp64 would be wrong by 1e-9."""
    import torch
    dt, n = 10.0, 3000
    gb = _templates()
    tab = inputs.orbit_table("kepler", t0, t0 + n * dt)
    R = lr.Response(tab, dt, 25, 2, t0=t0)
    hp, hc = R.gb_waveform(gb, n)
    torch.cuda.synchronize()
    hp, hc = hp.cpu().numpy(), hc.cpu().numpy()
    for b in range(gb.shape[0]):
        op, oc = owf.gb_waveform(gb[b], t0, dt, n)
        assert np.abs(hp[b] - op).max() <= 4e-15 * abs(gb[b, 0]), (b, np.abs(hp[b] - op).max() / abs(gb[b, 0]))
        assert np.abs(hc[b] - oc).max() <= 4e-15 * abs(gb[b, 1]), (b, np.abs(hc[b] - oc).max() / abs(gb[b, 1]))


def test_gb_waveform_full_length_windows(lr):
    """One year at 10 s (config 2's length): sampled windows against the exact-phase oracle."""
    import torch
    w = inputs.config(2)
    gb = _templates()[:2]
    R = lr.Response(w.table(), w.dt, w.order, 2, t0=w.t0)
    hp, hc = R.gb_waveform(gb, w.n)
    torch.cuda.synchronize()
    for first in (0, 1234567, w.n - 200):
        for b in range(2):
            op, oc = owf.gb_waveform(gb[b], w.t0, w.dt, 200, first=first)
            assert np.abs(hp[b, first:first + 200].cpu().numpy() - op).max() <= 4e-15 * abs(gb[b, 0])
            assert np.abs(hc[b, first:first + 200].cpu().numpy() - oc).max() <= 4e-15 * abs(gb[b, 1])


@pytest.mark.parametrize("chunk", [0, 1792 * 4])
def test_response_gb_equals_waveform_then_response(lr, chunk):
    """lr_response_gb == lr_response(lr_gb_waveform(...)) bit for bit (whatever the chunking), and both match
    the oracle run on the oracle's own waveform to the per-call bar."""
    import torch
    w = inputs.config(2, n=20011, f0=3e-3, t0=2.0e7)
    tab = w.table()
    gb = _templates()[:3]
    beta, lam, psi = [0.3, -0.8, 1.0], [1.0, 4.0, 5.5], [0.2, 1.0, 2.5]
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    if chunk:
        lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, chunk)
    out = R.response_gb(gb, beta, lam, psi, w.n)
    hp, hc = R.gb_waveform(gb, w.n)
    ref = R.response(hp, hc, beta, lam, psi)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    oh = out.cpu().numpy()
    for b in range(3):
        op, oc = owf.gb_waveform(gb[b], w.t0, w.dt, w.n)
        y = O.project(op, oc, beta[b], lam[b], psi[b], lo=mp, hi=w.n - mp)
        oo = O.tdi(y, 2, nested=True, channels=ORC_CH["XYZ_AET"], lo=mf, hi=w.n - mb)
        assert_parity(oh[b][:, mf:w.n - mb], oo[:, mf:w.n - mb], f"response_gb b={b}", CH_NAMES["XYZ_AET"])


def test_response_gb_errors(lr):
    import torch
    w = inputs.config(1)
    R = lr.Response(w.table(), w.dt, w.order, 1, t0=w.t0)
    out = torch.empty((1, 3, w.n), dtype=torch.float64, device="cuda")
    bad = np.array([[1.0, 1.0, float("nan"), 0.0, 0.0, 0.0]])
    with pytest.raises(lr.LrError):
        R.response_gb(bad, [0.1], [0.2], [0.3], w.n, out=out)
    with pytest.raises(ValueError):
        R.response_gb(np.zeros((1, 5)), [0.1], [0.2], [0.3], w.n, out=out)


def test_loglike_gb_against_oracle_pipeline(lr):
    """Parameters -> log L in one call against the oracle chain: exact-phase waveform, long-double
    projection and TDI (A, E, T), numpy FFT, eq. 3 accumulated in long double.  Data = template 1 (noiseless
    injection), analytic stand-in PSD.  11 templates (two chunks of 8), odd N."""
    import torch
    from oracle import likelihood as lk
    w = inputs.config(2, n=12001, f0=3e-3, t0=2.0e7)
    tab = w.table()
    rng = np.random.default_rng(5)
    nb = 11
    gb = np.empty((nb, 6))
    for b in range(nb):
        a = owf.amplitudes_paper(1e-22 * (1 + 0.1 * b), 0.3 + 0.2 * b)
        f0 = 3e-3 * (1 + 1e-4 * rng.standard_normal())
        gb[b] = (a[0], a[1], f0, 1e-16, owf.fddot_eq8(f0, 1e-16), rng.uniform(0, 2 * math.pi))
    gb[7] = gb[1]                                             # a copy of the data's parameters: log L = 0
    beta, lam, psi = rng.uniform(-1, 1, nb), rng.uniform(0, 6, nb), rng.uniform(0, 3, nb)
    beta[7], lam[7], psi[7] = beta[1], lam[1], psi[1]
    n, dt = w.n, w.dt
    O = orc.Oracle(tab, dt, w.t0, w.order)
    mp, mf, mb = O.margins(2)
    aet = np.zeros((nb, 3, n))
    for b in range(nb):
        op, oc = owf.gb_waveform(gb[b], w.t0, dt, n)
        y = O.project(op, oc, beta[b], lam[b], psi[b], lo=mp, hi=n - mp)
        aet[b] = O.tdi(y, 2, nested=True, channels=ORC_CH["AET"], lo=mf, hi=n - mb)
    f = np.fft.rfftfreq(n, dt)
    psd = inputs.psd_standin(f)
    inv = np.zeros_like(psd)
    inv[:, 1:] = 1.0 / psd[:, 1:]
    fh = lk.to_frequency(aet, dt)
    want = np.array([lk.log_likelihood(fh[1], fh[b], psd, dt, n) for b in range(nb)], dtype=np.float64)

    R = lr.Response(tab, dt, w.order, 2, t0=w.t0, channels="AET")
    data_f = torch.from_numpy(np.ascontiguousarray(np.fft.rfft(aet[1], axis=-1))).cuda()   # unnormalised DFT
    inv_d = to_dev(inv)
    got = R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    assert np.all(got <= 0)
    # the data are the ORACLE's template 1; the GPU's own template 1 differs from it by the path's 1e-13
    assert abs(got[1]) <= 1e-20 * np.abs(want).max() and abs(got[7]) <= 1e-20 * np.abs(want).max()
    others = [b for b in range(nb) if b not in (1, 7)]
    assert np.abs(got[others] - want[others]).max() <= 1e-10 * np.abs(want).max()
    # <h|d> mode, and the same call twice gives the same bits
    cross = R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, 4.0 * dt / n, mode=lr.LR_IP_CROSS).cpu().numpy()
    want_c = lk.inner_product(fh, fh[1:2], psd, dt, n).astype(np.float64)
    assert np.abs(cross - want_c).max() <= 1e-10 * np.abs(want_c).max()
    again = R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n).cpu().numpy()
    assert np.array_equal(got, again)
    # zero-padded transform (LR_OPT_FFT_LENGTH): 12001 -> 12005 = 5 * 7^4; the oracle pads the same series
    m = lr.lr_fft_good_length(n)
    assert m == 12005
    pad = np.concatenate([aet, np.zeros((nb, 3, m - n))], axis=-1)
    fpad = lk.to_frequency(pad, dt)
    psd_m = inputs.psd_standin(np.fft.rfftfreq(m, dt))
    inv_m = np.zeros_like(psd_m)
    inv_m[:, 1:] = 1.0 / psd_m[:, 1:]
    want_m = np.array([lk.log_likelihood(fpad[1], fpad[b], psd_m, dt, m) for b in range(nb)], dtype=np.float64)
    R.set_fft_length(m)
    data_m = torch.from_numpy(np.ascontiguousarray(np.fft.rfft(pad[1], axis=-1))).cuda()
    got_m = R.loglike_gb(gb, beta, lam, psi, n, data_m, to_dev(inv_m), -2.0 * dt / m).cpu().numpy()
    assert np.abs(got_m[others] - want_m[others]).max() <= 1e-10 * np.abs(want_m).max()
    assert np.abs(want_m[others] / want[others] - 1).max() < 0.05      # the same integral on a finer grid
    R.set_fft_length(0)
    assert np.array_equal(R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n).cpu().numpy(), got)
    with pytest.raises(lr.LrError):
        R.set_fft_length(n - 1)
        R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n)
    R.set_fft_length(0)
    R6 = lr.Response(tab, dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    with pytest.raises(lr.LrError):
        R6.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, 1.0)


def test_loglike_gb_pipelined_chunks_bitwise(lr):
    """batch > 8: lr_loglike_gb runs the transforms and the inner product of one chunk of 8 templates on a stream
    of the handle beside the response of the next chunk (two slots, reused from the third chunk on).  The 27
    scalars must equal, bit for bit, those of four separate calls of <= 8 templates (the one-slot path), on the
    default and on a caller's stream, twice in a row."""
    import torch
    w = inputs.config(2, n=9001, f0=4e-3, t0=2.5e7)
    tab = w.table()
    rng = np.random.default_rng(27)
    nb = 27
    gb = np.empty((nb, 6))
    for b in range(nb):
        a = owf.amplitudes_paper(1e-22 * (1 + 0.05 * b), 0.2 + 0.1 * b)
        gb[b] = (a[0], a[1], 4e-3 * (1 + 1e-4 * rng.standard_normal()), 1e-16, 0.0, rng.uniform(0, 2 * math.pi))
    beta, lam, psi = rng.uniform(-1, 1, nb), rng.uniform(0, 6, nb), rng.uniform(0, 3, nb)
    n, dt = w.n, w.dt
    R = lr.Response(tab, dt, w.order, 2, t0=w.t0, channels="AET")
    data_f = torch.fft.rfft(R.response_gb(gb[3:4], beta[3:4], lam[3:4], psi[3:4], n)[0], dim=-1).contiguous()
    inv = np.zeros((3, n // 2 + 1))
    inv[:, 1:] = 1.0 / inputs.psd_standin(np.fft.rfftfreq(n, dt))[:, 1:]
    inv_d = to_dev(inv)
    parts = [R.loglike_gb(gb[lo:lo + 8], beta[lo:lo + 8], lam[lo:lo + 8], psi[lo:lo + 8], n, data_f, inv_d,
                          -2.0 * dt / n).cpu().numpy() for lo in range(0, nb, 8)]
    want = np.concatenate(parts)
    assert want[3] == 0.0 and np.all(want[np.arange(nb) != 3] < 0)
    for _ in range(2):
        got = R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n).cpu().numpy()
        assert np.array_equal(got, want)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        got_s = R.loglike_gb(gb, beta, lam, psi, n, data_f, inv_d, -2.0 * dt / n, stream=s)
        got_s = got_s.cpu().numpy()      # ordered behind the call on s: the side stream is joined before it returns
    assert np.array_equal(got_s, want)
