"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot run 3e6-2.5e7 samples in long double within a test, so each case runs the whole workload on
the GPU and compares sampled windows (the first and last valid samples, plus seeded random windows) that the
oracle computes one by one; outside the margins every output must be exactly 0.  Same bar as the reduced
cases: 1e-10 per channel (parity_util).
"""
import numpy as np
import pytest

from harness import inputs
from parity_util import windows
from test_gpu_parity import check_workload, lr  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def _wins(w, lr_mod, count, width=384, seed=0, gen=None):
    """Windows over the TDI-valid region (the projection is checked on the same windows)."""
    R = lr_mod.Response(w.table(), w.dt, w.order, gen or w.tdi_gen, t0=w.t0)
    mp, mf, mb = R.margins()
    R.close()
    return windows(mf, w.n - mb, width, count, seed)


def test_full_size_config2_year(lr):  # noqa: F811
    """configs[1]: 3,153,600 samples, one launch per stage, XYZ+AET, nested and eq. 20 sums."""
    w = inputs.config(2)
    assert w.n == 3153600
    wins = _wins(w, lr, 8, seed=22)
    check_workload(lr, w, wins=wins)
    check_workload(lr, w, wins=wins[:3], chain="sum", proj=False)


BENCH_CHUNK = 64   # bench.py's --chunk default: templates per launch of the batch leg


def test_full_size_config3_bench_launch_shape(lr):  # noqa: F811
    """configs[2] at the launch shape bench.py times: chunks of 64 templates x 1,576,800 samples (12,319 projection
    tiles x 64 = 788,416 CTAs, 4.8 GB of y per launch), A,E,T.  Compared with the oracle on sampled windows of
    template 0, template 1023 and six seeded picks across the 1,024 ("the first, the last and 6
    seeded picks"); only the chunks that hold a pick are generated and run.  The inputs are made on the device by
    the harness generator bench.py uses, and the oracle reads those same arrays."""
    import bench
    import torch
    from oracle import oracle as orc
    from parity_util import CH_NAMES, LINK_NAMES, ORC_CH, assert_parity
    assert bench.DEFAULT_CHUNK == BENCH_CHUNK
    w = inputs.config(3)
    assert w.n == 1576800 and len(w.sources) == 1024 and w.channels == "AET"
    n = w.n
    picks = sorted({0, 1023} | {int(i) for i in np.random.default_rng(633).choice(np.arange(1, 1023), 6, replace=False)})
    assert len(picks) == 8
    tab = w.table()
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="AET")
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    assert (mp, mf, mb) == O.margins(2)
    wins = _wins(w, lr, 3, seed=35)
    y = torch.empty((BENCH_CHUNK, 6, n), dtype=torch.float64, device="cuda")
    out = torch.empty((BENCH_CHUNK, 3, n), dtype=torch.float64, device="cuda")
    seen = {}
    for lo in sorted({(p // BENCH_CHUNK) * BENCH_CHUNK for p in picks}):
        src = w.sources[lo:lo + BENCH_CHUNK]
        hp, hc = inputs.gb_waveform_device(src, n, w.dt, w.t0, "cuda")
        be, la, ps = ([getattr(s, k) for s in src] for k in ("beta", "lam", "psi"))
        R.project(hp, hc, be, la, ps, y_out=y)
        R.tdi(y, out=out)
        torch.cuda.synchronize()
        for p in (p for p in picks if lo <= p < lo + BENCH_CHUNK):
            k = p - lo
            hpk, hck, yk, ok = (t[k].cpu().numpy() for t in (hp, hc, y, out))
            assert not yk[:, :mp].any() and not yk[:, n - mp:].any()
            assert not ok[:, :mf].any() and not ok[:, n - mb:].any()
            for a, b in wins:
                yo = O.project(hpk, hck, be[k], la[k], ps[k], lo=a, hi=b)
                assert_parity(yk[:, a:b], yo[:, a:b], f"batch project template {p} [{a},{b})", LINK_NAMES)
                oo = O.tdi(yk, 2, nested=True, channels=ORC_CH["AET"], lo=a, hi=b)
                assert_parity(ok[:, a:b], oo[:, a:b], f"batch tdi template {p} [{a},{b})", CH_NAMES["AET"])
            seen[p] = ok[:, wins[0][0]:wins[0][1]].copy()
        del hp, hc
    # templates differ: no two outputs may coincide (batch indexing across and inside chunks)
    vals = list(seen.values())
    assert all(not np.array_equal(vals[i], vals[j]) for i in range(len(vals)) for j in range(i))


def test_full_size_config3_sampled_templates(lr):  # noqa: F811
    """configs[2], three templates in one small launch (host-generated inputs), four windows each."""
    w = inputs.config(3, batch=16)
    wins = _wins(w, lr, 4, seed=34)
    w.sources = [w.sources[i] for i in (0, 7, 15)]
    check_workload(lr, w, idx=(0, 1, 2), wins=wins)


def test_full_size_config4_four_years(lr):  # noqa: F811
    """configs[3]: 25,228,800 samples at dt = 5 s, order 41, perturbed orbits, TDI-2 XYZ (the maximum size of
    the configs: 1.2 GB of y)."""
    w = inputs.config(4)
    assert w.n == 25228800
    check_workload(lr, w, wins=_wins(w, lr, 6, width=256, seed=44))


def test_full_size_config5_chirp(lr):  # noqa: F811
    """configs[4]: 1,555,200 samples, full TDI-2 and the hybrid mode (TDI-1 on equal-arm constant delays)."""
    w = inputs.config(5)
    assert w.n == 1555200
    wins = _wins(w, lr, 6, seed=55)
    check_workload(lr, w, wins=wins)
    eq = inputs.orbit_table("eq", w.t0, w.t0 + w.n * w.dt, const_ltt=inputs.ARM / inputs.C_LIGHT)
    check_workload(lr, w, tdi_tab=eq, tdi_gen=1, proj=False, wins=_wins(w, lr, 4, seed=56, gen=1))


def test_full_size_parameters_in(lr):  # noqa: F811
    """configs[1] from the parameters (lr_response_gb, lr_loglike_gb) in the shape bench.py times: the one-call
    result equals lr_response on the generated h bit for bit, sampled windows of it match the oracle chain
    (exact-phase waveform, long-double projection and TDI), and log L of the template that made the data is
    exactly 0 while a neighbour's is negative."""
    import torch
    from oracle import oracle as orc
    from oracle import waveform as owf
    from parity_util import CH_NAMES, ORC_CH, assert_parity
    w = inputs.config(2)
    s = w.sources[0]
    a = owf.amplitudes_config(s.A, s.iota)
    gb = np.array([[a[0], a[1], s.f0, s.fdot, 0.0, s.phi0], [a[0], a[1], s.f0 * (1 + 1e-7), s.fdot, 0.0, s.phi0]])
    be, la, ps = [s.beta] * 2, [s.lam] * 2, [s.psi] * 2
    tab = w.table()
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="AET")
    out = R.response_gb(gb, be, la, ps, w.n)
    hp, hc = R.gb_waveform(gb, w.n)
    ref = R.response(hp, hc, be, la, ps)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    for lo, hi in _wins(w, lr, 3, width=256, seed=55):
        pad = mf + 8                                   # the oracle window needs y (hence h) over the TDI reach
        a0, a1 = max(lo - pad - mp, 0), min(hi + mb + mp + 8, w.n)
        op, oc = owf.gb_waveform(gb[0], w.t0, w.dt, a1 - a0, first=a0)   # exact phase: T amplifies 1e-12 of h
        hp_full = np.zeros(w.n)
        hc_full = np.zeros(w.n)
        hp_full[a0:a1], hc_full[a0:a1] = op, oc
        y = O.project(hp_full, hc_full, s.beta, s.lam, s.psi, lo=max(a0 + mp, mp), hi=min(a1 - mp, w.n - mp))
        oo = O.tdi(y, 2, nested=True, channels=ORC_CH["AET"], lo=lo, hi=hi)
        assert_parity(out[0, :, lo:hi].cpu().numpy(), oo[:, lo:hi], f"response_gb year [{lo},{hi})", CH_NAMES["AET"])
    nf = w.n // 2 + 1
    inv = torch.ones((3, nf), dtype=torch.float64, device="cuda")
    inv[:, 0] = 0
    data_f = torch.fft.rfft(out[0], dim=-1).contiguous()
    ll = R.loglike_gb(gb, be, la, ps, w.n, data_f, inv, -2.0 * w.dt / w.n).cpu().numpy()
    assert abs(ll[0]) <= 1e-18 * abs(ll[1]) and ll[1] < 0      # cuFFT on both sides: the same bits up to its plan
