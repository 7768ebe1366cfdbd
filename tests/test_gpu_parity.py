"""GPU parity: liblr (CUDA, through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Run on the B200 box with `pytest -m gpu`.

Per-call parity: lr_project against the oracle's projection of the same h;
lr_tdi against the oracle's TDI of the *same fp64 y* (the GPU's own).  Bar: parity_util.REL_L2_TOL /
MAX_ABS_TOL = 1e-10 (north_star).  Reduced sizes still span several 256-sample tiles and end in a ragged
tail; the full BASELINE.json sizes are checked on sampled windows in the launch configuration bench.py
times (test_full_size_*).
"""
import numpy as np
import pytest

from oracle import oracle as orc
from harness import inputs
from parity_util import (CH_NAMES, LINK_NAMES, ORC_CH, assert_parity, to_dev, windows)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lr():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    import paper_2204_06633_b200 as pkg
    from paper_2204_06633_b200 import build
    build.ensure_built()   # fresh checkout: the .so is git-ignored; compiling it needs nvcc (no CPU fallback)
    pkg.binding.lib()      # fail loudly if liblr.so cannot be loaded
    return pkg


def _stack(w, idx):
    hp, hc = zip(*(w.waveform(b) for b in idx))
    return np.stack(hp), np.stack(hc)


def check_workload(lr, w, *, chain="nested", channels=None, gen=None, idx=(0,), wins=None, tab=None,
                   tdi_tab=None, tdi_gen=None, proj=True, tdi_path="auto"):
    """Run w's templates `idx` through lr_project and lr_tdi and compare with the oracle.
    wins: list of (lo, hi) sample windows to compare on (None = the whole valid region)."""
    import torch
    channels = channels or w.channels
    gen = gen or w.tdi_gen
    tab = tab or w.table()
    n = w.n
    R = lr.Response(tab, w.dt, w.order, gen, t0=w.t0, chain=chain, channels=channels)
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    assert (mp, mf, mb) == O.margins(gen)
    hp, hc = _stack(w, idx)
    src = [w.sources[b] for b in idx]
    beta, lam, psi = ([getattr(s, k) for s in src] for k in ("beta", "lam", "psi"))
    y = R.project(to_dev(hp), to_dev(hc), beta, lam, psi)
    torch.cuda.synchronize()
    yh = y.cpu().numpy()
    assert np.all(yh[:, :, :mp] == 0) and np.all(yh[:, :, n - mp:] == 0)
    errs = {}
    if proj:
        for k, b in enumerate(idx):
            for lo, hi in (wins or [(mp, n - mp)]):
                lo, hi = max(lo, mp), min(hi, n - mp)
                yo = O.project(hp[k], hc[k], beta[k], lam[k], psi[k], lo=lo, hi=hi)
                errs[("proj", b, lo)] = assert_parity(yh[k][:, lo:hi], yo[:, lo:hi], f"{w.name} project b={b} [{lo},{hi})",
                                                      LINK_NAMES)
    # stage 2 on the GPU's own fp64 y; optionally with another handle (hybrid)
    Rt, Ot, g2 = R, O, gen
    if tdi_tab is not None:
        g2 = tdi_gen or gen
        Rt = lr.Response(tdi_tab, w.dt, w.order, g2, t0=w.t0, chain=chain, channels=channels)
        Ot = orc.Oracle(tdi_tab, w.dt, w.t0, w.order)
    Rt.set_tdi_path(tdi_path)
    out = Rt.tdi(y)
    torch.cuda.synchronize()
    oh = out.cpu().numpy()
    _, mf, mb = Rt.margins()
    assert np.all(oh[:, :, :mf] == 0) and np.all(oh[:, :, n - mb:] == 0)
    for k, b in enumerate(idx):
        for lo, hi in (wins or [(mf, n - mb)]):
            lo, hi = max(lo, mf), min(hi, n - mb)
            oo = Ot.tdi(yh[k], g2, nested=(chain == "nested"), channels=ORC_CH[channels], lo=lo, hi=hi)
            errs[("tdi", b, lo)] = assert_parity(oh[k][:, lo:hi], oo[:, lo:hi],
                                                 f"{w.name} tdi gen{g2} {chain} b={b} [{lo},{hi})", CH_NAMES[channels])
    return errs, yh, oh


# ------------------------------------------------------------------------------------------- config 1
def test_config1_tiny_full(lr):
    """BASELINE.json configs[0] at its full size: EQ orbits, constant equal light times, TDI-1 XYZ."""
    check_workload(lr, inputs.config(1))


def test_config1_tiny_fixed_point_ltt(lr):
    """Same with the flat-space fixed-point light times (L_ij != L_ji), nested and eq. 20 sums, gen 1 and 2,
    every lr_tdi path.  (X, Y, Z here: with exactly equal arms T is a null channel, |T| = 3e-5 |A|, and its
    relative error only measures that suppression; SURVEY.md §8(c) worked example.  A, E, T are covered on the
    Keplerian configs.)"""
    w = inputs.config(1)
    tab = inputs.orbit_table("eq", w.t0, w.t0 + w.n * w.dt)
    for chain in ("nested", "sum"):
        for gen in (1, 2):
            for path in ("per_sample", "fir3", "fir4"):
                check_workload(lr, w, tab=tab, chain=chain, gen=gen, channels="XYZ", tdi_path=path,
                               proj=(path == "per_sample"))


@pytest.mark.parametrize("ltt", ["fixed_point", "constant"])
def test_tdi_null_channel_strict(lr, ltt):
    """The same equal-arm cases with A, E, T.  T is a null channel here (|T| = 2.5e-5 |A|), the hardest per-call
    case of the repository: the STRICT bar (1e-10 relative to T itself, rel-L2 and max-abs) holds on every lr_tdi
    path, both generations and both chain forms (measured round 2: worst 2.6e-11 rel-L2 / 8.4e-11 max-abs, TDI-2,
    eq. 20 sums, per-sample path), and is asserted for all of them."""
    w = inputs.config(1)
    tab = inputs.orbit_table("eq", w.t0, w.t0 + w.n * w.dt) if ltt == "fixed_point" else w.table()
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    s = w.sources[0]
    hp, hc = w.waveform(0)
    for gen in (1, 2):
        for chain in ("nested", "sum"):
            oo = None
            for path in ("auto", "per_sample", "fir3", "fir4"):
                R = lr.Response(tab, w.dt, w.order, gen, t0=w.t0, channels="AET", tdi_path=path, chain=chain)
                mp, mf, mb = R.margins()
                y = R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
                out = R.tdi(y).cpu().numpy()[0]
                if oo is None:   # (the projection does not depend on the TDI path: one oracle run per case)
                    oo = O.tdi(y.cpu().numpy()[0], gen, nested=(chain == "nested"), channels=orc.CH_AET)
                v = slice(mf, w.n - mb)
                assert np.abs(oo[2, v]).max() < 1e-4 * np.abs(oo[0, v]).max()      # T really is the null channel
                assert_parity(out[:, v], oo[:, v], f"equal-arm {ltt} gen{gen} {chain} ({path})", ["A", "E", "T"])


def test_tdi_delay_crossing_whole_sample(lr):
    """Degenerate case of the FIR path: light times that drift THROUGH a whole number of samples inside the
    series (L = 10 s +- at dt = 10 s), so the integer part of several delays changes mid-tile; those tiles must
    fall back to the exact per-sample weights.  Also L exactly constant = 1 sample (eps = 0 everywhere)."""
    import torch
    dt, n, t0, order = 10.0, 5000, 3.0e7, 25
    base = inputs.orbit_table("kepler", t0, t0 + n * dt)
    tk = base.t_start + base.knot_dt * np.arange(base.n_knots)
    t_mid = t0 + 0.5 * n * dt
    rng = np.random.default_rng(5)
    t = t0 + dt * np.arange(n)
    y = np.stack([np.sin(2 * np.pi * f * t + p) for f, p in zip(rng.uniform(1e-3, 2e-2, 6), rng.uniform(0, 6, 6))])
    for ltt in (np.tile(10.0 + 2e-8 * (tk - t_mid), (6, 1)) * (1 + 1e-4 * np.arange(6))[:, None],
                np.full((6, base.n_knots), 10.0)):
        tab = inputs.OrbitTable(base.t_start, base.knot_dt, base.x, np.ascontiguousarray(ltt))
        O = orc.Oracle(tab, dt, t0, order)
        for gen in (1, 2):
            oo = None
            for path in ("per_sample", "fir3", "fir4"):
                R = lr.Response(tab, dt, order, gen, t0=t0, tdi_path=path)
                _, mf, mb = R.margins()
                out = R.tdi(to_dev(y)[None]).cpu().numpy()[0]
                torch.cuda.synchronize()
                if oo is None:
                    oo = O.tdi(y, gen, nested=True)
                assert_parity(out[:, mf:n - mb], oo[:, mf:n - mb], f"crossing gen{gen} {path}", CH_NAMES["XYZ"])


def test_tdi_fixup_skipped_only_where_no_tile_is_flagged(lr):
    """Once the plan's list of flagged tiles has reached the host, a launch whose window holds none of them skips the
    fork / fix-up kernel / join.  Light times that cross a whole number of samples in the MIDDLE of a 40,000-sample
    series flag a few tiles there (the fix-up kernel runs tdi_sample, so those tiles equal the per-sample path bit
    for bit; all others differ from it in the last digits).  The first call (list unknown), later calls (list
    known) and chunked lr_response calls (most chunks without a flagged tile) must agree bit for bit, flagged
    tiles included."""
    import torch
    dt, n, t0, order = 10.0, 40000, 3.0e7, 9
    base = inputs.orbit_table("kepler", t0, t0 + n * dt)
    tk = base.t_start + base.knot_dt * np.arange(base.n_knots)
    ltt = np.tile(10.0 + 2e-9 * (tk - (t0 + 0.5 * n * dt)), (6, 1)) * (1 + 1e-7 * np.arange(6))[:, None]
    tab = inputs.OrbitTable(base.t_start, base.knot_dt, base.x, np.ascontiguousarray(ltt))
    w = inputs.config(2, n=n, t0=t0)
    hp, hc = w.waveform(0)
    s = w.sources[0]
    hp_d, hc_d = to_dev(hp)[None], to_dev(hc)[None]
    R = lr.Response(tab, dt, order, 2, t0=t0, tdi_path="fir3")
    Rp = lr.Response(tab, dt, order, 2, t0=t0, tdi_path="per_sample")
    _, mf, mb = R.margins()
    y = R.project(hp_d, hc_d, [s.beta], [s.lam], [s.psi])
    first = R.tdi(y).cpu().numpy()[0]            # builds the plan; the list is still on its way to the host
    torch.cuda.synchronize()
    ps = Rp.tdi(y).cpu().numpy()[0]
    tile = 224
    same = [t for t in range(mf // tile + 1, (n - mb) // tile)
            if np.array_equal(first[:, t * tile:(t + 1) * tile], ps[:, t * tile:(t + 1) * tile])]
    assert 1 <= len(same) <= 40, len(same)       # the flagged tiles, and only a few of them
    assert all(abs(t * tile - n // 2) < 6000 for t in same), same
    for _ in range(3):                           # list known: whole-series window holds flagged tiles -> fix-up runs
        assert np.array_equal(R.tdi(y).cpu().numpy()[0], first)
    one = R.response(hp_d, hc_d, [s.beta], [s.lam], [s.psi]).cpu().numpy()[0]
    assert np.array_equal(one, first)
    lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, 1792)    # 23 chunks, flagged tiles in two or three of them
    for _ in range(2):
        assert np.array_equal(R.response(hp_d, hc_d, [s.beta], [s.lam], [s.psi]).cpu().numpy()[0], first)
    lo = (min(same) * tile // 1792) * 1792
    span = R.response_span(hp_d, hc_d, 0, [s.beta], [s.lam], [s.psi], n, 1792 * 2, 1792 * 3)   # no flagged tile in it
    assert lo > 1792 * 5 and np.array_equal(span.cpu().numpy()[0], first[:, 1792 * 2:1792 * 5])
    span = R.response_span(hp_d, hc_d, 0, [s.beta], [s.lam], [s.psi], n, lo, 1792 * 2)           # flagged tiles in it
    assert np.array_equal(span.cpu().numpy()[0], first[:, lo:lo + 1792 * 2])
    O = orc.Oracle(tab, dt, t0, order)
    oo = O.tdi(y.cpu().numpy()[0], 2, nested=True)
    assert_parity(first[:, mf:n - mb], oo[:, mf:n - mb], "fir3 with flagged tiles", CH_NAMES["XYZ"])


@pytest.mark.parametrize("ldot", [1e-9, 3e-8, 1e-6, 1e-5])
def test_tdi_auto_path_follows_the_light_time_rate(lr, ldot):
    """LR_TDI_AUTO picks quadratic / cubic FIR / per-sample weights from the largest |dL/dt| of the table
    (1e-9: Keplerian-like; 3e-8..1e-6: strongly perturbed orbits; 1e-5: beyond any orbit, a delay sweeps through
    whole samples every few hundred samples).  Whatever it picks must match the oracle, and the automatic
    choice must agree bit for bit with the explicitly selected path it is documented to take."""
    dt, n, t0, order = 5.0, 12000, 4.0e7, 25
    base = inputs.orbit_table("kepler", t0, t0 + n * dt)
    tk = base.t_start + base.knot_dt * np.arange(base.n_knots)
    rate = ldot * (1 + 0.1 * np.arange(6))[:, None] * np.array([1, -1, 1, -1, 1, -1])[:, None]
    ltt = 8.3 + 0.01 * np.arange(6)[:, None] + rate * (tk - (t0 + 0.5 * n * dt))[None, :]
    tab = inputs.OrbitTable(base.t_start, base.knot_dt, base.x, np.ascontiguousarray(ltt))
    rng = np.random.default_rng(17)
    t = t0 + dt * np.arange(n)
    y = np.stack([np.sin(2 * np.pi * f * t + p) for f, p in zip(rng.uniform(2e-4, 2e-2, 6), rng.uniform(0, 6, 6))])
    O = orc.Oracle(tab, dt, t0, order)
    oo = O.tdi(y, 2, nested=True, channels=orc.CH_XYZ_AET)
    R = lr.Response(tab, dt, order, 2, t0=t0, channels="XYZ_AET")
    _, mf, mb = R.margins()
    out = R.tdi(to_dev(y)[None]).cpu().numpy()[0]
    assert_parity(out[:, mf:n - mb], oo[:, mf:n - mb], f"auto path, dL/dt = {ldot:g}", CH_NAMES["XYZ_AET"])
    de = 7 * 1.6 * ldot * 224      # links x largest rate x tile
    expect = "fir3" if de <= 6e-6 else "fir4" if de <= 1.5e-4 else "per_sample"
    Re = lr.Response(tab, dt, order, 2, t0=t0, channels="XYZ_AET", tdi_path=expect)
    assert np.array_equal(Re.tdi(to_dev(y)[None]).cpu().numpy()[0], out), expect


# ------------------------------------------------------------------------------------------- config 2
@pytest.mark.parametrize("f0", [None, 1e-4, 1e-3, 1e-2])
@pytest.mark.parametrize("chain", ["nested", "sum"])
@pytest.mark.parametrize("tdi_path", ["auto", "per_sample", "fir3", "fir4"])
def test_config2_year_reduced(lr, f0, chain, tdi_path):
    """configs[1] shortened to 20,011 samples (79-90 tiles, ragged tail): Keplerian, TDI-2, XYZ+AET; the seeded
    source and the three fixed-frequency strata of SURVEY.md §8(c); every lr_tdi path."""
    check_workload(lr, inputs.config(2, n=20011, f0=f0, t0=3.0e7), chain=chain, tdi_path=tdi_path,
                   proj=(tdi_path == "auto"))


def test_config2_paper_sources(lr):
    """The paper's own three (f, fdot) points with its angles as seed-free sources."""
    w = inputs.config(2, n=6007, t0=1.0e7)
    for f, fd in ((6e-4, 1.5e-18), (2e-3, 1.2e-17), (6e-3, 1.3e-16)):
        w.sources = [inputs.Source(A=1e-22, f0=f, fdot=fd, iota=1.11, phi0=4.58, psi=0.45, lam=5.23, beta=0.09)]
        check_workload(lr, w)


# ------------------------------------------------------------------------------------------- config 3
def test_config3_batch_reduced(lr):
    """configs[2] with 7 templates of 9,001 samples in ONE launch: batch indexing, AET output."""
    w = inputs.config(3, batch=7, n=9001)
    check_workload(lr, w, idx=tuple(range(7)))


def test_source_basis_staging_paths_bitwise(lr):
    """Step P1 runs on the device: up to 16 templates per call carry their angles in the parameter buffer of
    source_basis_small_kernel, larger batches go through a host -> device copy and source_basis_kernel.  Both run
    the same device function, so a 19-template launch must equal 19 one-template launches bit for bit
    (lr_project, and lr_gb_waveform whose six numbers are staged the same way); template 0 against the oracle."""
    import torch
    w = inputs.config(3, batch=19, n=3001)
    R = lr.Response(w.table(), w.dt, 9, 2, t0=w.t0)
    hp, hc = _stack(w, range(19))
    hp_d, hc_d = to_dev(hp), to_dev(hc)
    be = [s.beta for s in w.sources]
    la = [s.lam for s in w.sources]
    ps = [s.psi for s in w.sources]
    y = R.project(hp_d, hc_d, be, la, ps).cpu().numpy()
    for b in range(19):
        yb = R.project(hp_d[b:b + 1], hc_d[b:b + 1], be[b:b + 1], la[b:b + 1], ps[b:b + 1]).cpu().numpy()
        assert np.array_equal(yb[0], y[b]), b
    O = orc.Oracle(w.table(), w.dt, w.t0, 9)
    mp = O.margins(2)[0]
    yo = O.project(hp[0], hc[0], be[0], la[0], ps[0])
    assert_parity(y[0, :, mp:w.n - mp], yo[:, mp:w.n - mp], "lr_project", LINK_NAMES)
    gb = np.array([[s.A * (1.0 + np.cos(s.iota) ** 2), -2.0 * s.A * np.cos(s.iota), s.f0, s.fdot, 0.0, s.phi0]
                   for s in w.sources])
    gp, gc = R.gb_waveform(gb, w.n)
    for b in (0, 7, 18):
        p1, c1 = R.gb_waveform(gb[b:b + 1], w.n)
        assert torch.equal(p1[0], gp[b]) and torch.equal(c1[0], gc[b])
    out = R.response_gb(gb, be, la, ps, w.n)
    assert torch.equal(out, R.response(gp, gc, be, la, ps))


# ------------------------------------------------------------------------------------------- config 4
@pytest.mark.parametrize("tdi_path", ["auto", "per_sample", "fir4"])
def test_config4_numerical_orbits_reduced(lr, tdi_path):
    """configs[3] shortened: perturbed-orbit tables (L_ij != L_ji), dt = 5 s, order 41, TDI-2 XYZ."""
    check_workload(lr, inputs.config(4, n=12345, t0=5.0e7), tdi_path=tdi_path)
    check_workload(lr, inputs.config(4, n=5000, t0=1.0e8, f0=1e-4), chain="sum", tdi_path=tdi_path)


# ------------------------------------------------------------------------------------------- config 5
def test_config5_chirp_reduced(lr):
    """configs[4] shortened (the last 30,001 samples of the chirp, where f sweeps fastest): full TDI-2 and
    the hybrid mode (projection on Keplerian orbits, TDI-1 on equal-arm constant delays)."""
    full = inputs.config(5)
    n = 30001
    w = inputs.config(5, n=n, t0=full.t0 + (full.n - n) * full.dt)
    hp, hc = full.waveform(0)
    w.waveform = lambda b=0: (hp[-n:].copy(), hc[-n:].copy())
    check_workload(lr, w)
    eq = inputs.orbit_table("eq", w.t0, w.t0 + n * w.dt, const_ltt=inputs.ARM / inputs.C_LIGHT)
    check_workload(lr, w, tdi_tab=eq, tdi_gen=1, proj=False)


# --------------------------------------------------------------------------------------------- orders
@pytest.mark.parametrize("order", [1, 3, 5, 7, 9, 11, 13, 15, 17, 21, 31, 35, 65])
def test_orders(lr, order):
    """Compile-time-P kernels (1-15, 21, 31; 25 and 41 are the configs' orders) and the run-time-P path
    (17, 35, 65)."""
    w = inputs.config(2, n=3001, f0=2e-3, t0=2.0e7)
    w.order = order
    check_workload(lr, w, channels="XYZ")
    check_workload(lr, w, channels="XYZ", tdi_path="per_sample", proj=False)


@pytest.mark.parametrize("order", [1, 5, 9, 13, 21, 25, 31, 41, 17])
def test_project_pair_path_bitwise(lr, order):
    """LR_PROJ_PAIR (two consecutive samples per thread, shared first differences, geometry parked in shared memory,
    de-interleaved window) against LR_PROJ_SINGLE: the same bits, on ragged multi-template launches, on a time chunk
    that starts at an odd global sample, and on orbits whose reception delay wraps through whole samples many
    times (the out-of-line path of a pair whose integer shifts differ).  Order 17 has no compile-time kernel: the
    option is accepted and runs the single path."""
    import torch
    w = inputs.config(3, batch=3, n=20011, t0=4.0e6)
    w.order = order
    hp, hc = _stack(w, range(3))
    be, la, ps = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    hpd, hcd = to_dev(hp), to_dev(hc)
    outs = {}
    for path in ("single", "pair"):
        R = lr.Response(w.table(), w.dt, order, 2, t0=w.t0)
        R.set_y_precision("plain")      # the pair kernel implements the plain delay form
        R.set_proj_path(path)
        y = R.project(hpd, hcd, be, la, ps)
        lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, 1792 * 2)    # chunks whose y window starts at a - halo
        outs[path] = (y.cpu().numpy(), R.response(hpd, hcd, be, la, ps).cpu().numpy())
    assert np.array_equal(outs["single"][0], outs["pair"][0])
    assert np.array_equal(outs["single"][1], outs["pair"][1])
    Rx = lr.Response(w.table(), w.dt, order, 2, t0=w.t0)
    Rx.set_proj_path("pair")            # with the default LR_Y_EXTENDED the option is accepted and runs the single kernel
    assert lr.lr_get_option(Rx.handle, lr.LR_OPT_Y_PRECISION) == lr.LR_Y_EXTENDED
    yx = Rx.project(hpd, hcd, be, la, ps).cpu().numpy()
    assert np.abs(yx - outs["single"][0]).max() <= 1e-12 * np.abs(yx).max()
    mp = Rx.margins()[0]
    assert np.count_nonzero(outs["pair"][0][:, :, mp:w.n - mp]) > 0.99 * 18 * (w.n - 2 * mp)
    if order == 25:   # template 0 against the oracle, through the pair path
        O = orc.Oracle(w.table(), w.dt, w.t0, order)
        yo = O.project(hp[0], hc[0], be[0], la[0], ps[0], lo=mp, hi=mp + 3000)
        assert_parity(outs["pair"][0][0][:, mp:mp + 3000], yo[:, mp:mp + 3000], "pair path", LINK_NAMES)


# ------------------------------------------------------------------------- LR_Y_EXTENDED (NEXT-1)
@pytest.mark.parametrize("f0", [1e-4, 1e-3, 1e-2])
def test_extended_y_end_to_end(lr, f0):
    """LR_OPT_Y_PRECISION = LR_Y_EXTENDED (the accuracy half of the fused row; PAPER.md:181
    eq. 16 and 193-197 eqs. 17-18 for the cancellations involved).  The end-to-end error of the path (GPU h -> out
    against the ALL-long-double oracle pipeline) is set by y: TDI amplifies errors of y by up to 1e6 in T at 0.1 mHz.
    With the emission delays placed relative to the reception split and the arm vectors splined directly, y agrees
    with the oracle to a few 1e-16 (plain: 2.4e-14) and end-to-end T is <= 1e-9 at 0.1 mHz and <= 1e-10 from 1 mHz
    (plain: 2.2e-8 and 2.2e-10); measured round 2: 7.8e-10, 8.1e-12, 1.8e-13 beside an fp64-y floor of 6.3e-11,
    6.8e-13, 3.6e-15.  The plain path is untouched (same kernel instantiation as before)."""
    w = inputs.config(2, n=20011, f0=f0, t0=3.0e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    yo = O.project(hp, hc, s.beta, s.lam, s.psi)
    o_ld = O.tdi(yo, 2, nested=True, channels=orc.CH_XYZ_AET)          # long-double y into long-double TDI
    errs = {}
    for mode in ("plain", "extended"):
        R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
        R.set_y_precision(mode)
        mp, mf, mb = R.margins()
        y = R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
        yh = y.cpu().numpy()[0]
        assert not yh[:, :mp].any() and not yh[:, w.n - mp:].any()
        ey = assert_parity(yh[:, mp:w.n - mp], yo[:, mp:w.n - mp], f"project ({mode})", LINK_NAMES)
        out = R.tdi(y).cpu().numpy()[0]
        from parity_util import channel_errors
        e2e = [channel_errors(out[c, mf:w.n - mb], o_ld[c, mf:w.n - mb]) for c in range(6)]
        errs[mode] = (max(r for r, _ in ey), e2e)
        if mode == "extended":
            one = R.response(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi]).cpu().numpy()[0]
            assert np.array_equal(one, out)                               # the one-call path takes the option too
    y_plain, y_ext = errs["plain"][0], errs["extended"][0]
    assert y_ext <= 5e-15 and y_ext < 0.3 * y_plain, (y_plain, y_ext)
    t_rel = errs["extended"][1][5][0]
    assert t_rel <= (1e-9 if f0 < 5e-4 else 1e-10), t_rel
    assert t_rel < 0.2 * errs["plain"][1][5][0]
    for c in range(5):                                                    # X, Y, Z, A, E end to end
        assert errs["extended"][1][c][0] <= 1e-11


@pytest.mark.parametrize("cfg,kw", [(1, {}), (3, {"batch": 3, "n": 9001}), (4, {"n": 12345, "t0": 5.0e7}),
                                    (5, {"n": 20001})])
def test_extended_y_parity_other_configs(lr, cfg, kw):
    """LR_Y_EXTENDED per call on the other configs' orbits and orders (equal-arm, Keplerian batch, perturbed orbits at
    order 41, chirp): lr_project within 1e-14 of the oracle per link, and the chunked one-call path bit-identical."""
    import torch
    w = inputs.config(cfg, **kw)
    tab = w.table()
    idx = range(len(w.sources))
    hp, hc = _stack(w, idx)
    be, la, ps = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    R = lr.Response(tab, w.dt, w.order, w.tdi_gen, t0=w.t0, channels=w.channels)
    R.set_y_precision("extended")
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    y = R.project(to_dev(hp), to_dev(hc), be, la, ps)
    yh = y.cpu().numpy()
    for k in idx:
        yo = O.project(hp[k], hc[k], be[k], la[k], ps[k])
        assert_parity(yh[k][:, mp:w.n - mp], yo[:, mp:w.n - mp], f"config {cfg} extended b={k}", LINK_NAMES,
                      rel_tol=1e-14, abs_tol=1e-13)
    ref = R.tdi(y).cpu().numpy()
    lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, 1792)
    assert np.array_equal(R.response(to_dev(hp), to_dev(hc), be, la, ps).cpu().numpy(), ref)
    oo = O.tdi(yh[0], w.tdi_gen, nested=True, channels=ORC_CH[w.channels])
    assert_parity(ref[0][:, mf:w.n - mb], oo[:, mf:w.n - mb], f"config {cfg} tdi of extended y", CH_NAMES[w.channels])
    # the arm-vector splines are the differences of the position splines (the fit is linear in the table)
    t = to_dev(np.linspace(w.t0 + 10 * w.dt, w.t0 + (w.n - 10) * w.dt, 257))
    ev = lambda ch: lr.lr_eval_orbit(R.handle, ch, t, torch.empty_like(t)).cpu().numpy()
    for arm in range(3):
        for a in range(3):
            d = ev(15 + arm * 3 + a)
            assert np.abs(d - (ev(arm * 3 + a) - ev(((arm + 1) % 3) * 3 + a))).max() <= 1e-4     # metres (ulp of 1 au: 3e-5)
            assert np.abs(d).max() < 3.2e9


# ---------------------------------------------------------------------------------------------- pins
@pytest.mark.parametrize("knot_dt", [400.0, 1000.0, 1290.0])
def test_dense_orbit_knots(lr, knot_dt):
    """Orbit knots closer than a projection tile (128 samples = 1280 s): at 400 s a tile spans four spline
    intervals and the kernel reads the coefficients from the global table; at 1000 s and 1290 s it spans two and
    uses its tile-local copy, with the interval boundary inside nearly every tile (reading A9)."""
    w = inputs.config(2, n=4001, f0=3e-3, t0=2.0e7)
    tab = inputs.orbit_table("kepler", w.t0, w.t0 + w.n * w.dt, knot_dt=knot_dt, pad=20000.0)
    check_workload(lr, w, tab=tab)


def test_gpu_laser_noise_suppression(lr):
    """Pin P3 run on the GPU TDI: three independent band-limited laser-noise series, y_ij = p_j(t - L_ij(t))
    - p_i(t) evaluated analytically; second-generation NESTED TDI must cancel them to interpolation level,
    eq. 20 sums and first generation must not."""
    import torch
    dt, n, t0, order = 10.0, 6000, 3.0e7, 25
    tab = inputs.orbit_table("kepler", t0, t0 + n * dt)
    O = orc.Oracle(tab, dt, t0, order)
    par = inputs.band_limited_noise(7)
    t = (np.longdouble(t0) + np.longdouble(dt) * np.arange(n)).astype(np.longdouble)
    y = np.zeros((6, n))
    for s, (i, j) in enumerate(inputs.LINKS):
        L = O.spline(9 + s, t)
        y[s] = (inputs.eval_tones(par, j - 1, t - L) - inputs.eval_tones(par, i - 1, t)).astype(np.float64)
    rms_p = float(np.sqrt(np.mean(inputs.eval_tones(par, 0, t).astype(np.float64) ** 2)))
    res = {}
    for gen in (1, 2):
        for chain in ("nested", "sum"):
            R = lr.Response(tab, dt, order, gen, t0=t0, chain=chain)
            _, mf, mb = R.margins()
            out = R.tdi(to_dev(y)[None]).cpu().numpy()[0]
            torch.cuda.synchronize()
            res[(gen, chain)] = float(np.sqrt(np.mean(out[0, mf:n - mb] ** 2))) / rms_p
    # fp64 y limits the residual to ~1e-16/rms; the survey's long-double value is 7.4e-14
    assert res[(2, "nested")] < 1e-12, res
    for key in ((2, "sum"), (1, "nested"), (1, "sum")):
        assert res[key] > 1e-10, res


def test_gpu_worked_example_golden(lr, golden_dir):
    """The CUDA path against the printed worked example (tests/golden/worked_example_p2.json; SURVEY.md §8(c),
    survey-computed from PAPER.md eqs. 10-18 with 40-digit arithmetic) WITHOUT the oracle in between: static
    equal-arm triangle, monochromatic source, every series is Re[(re + i im) e^{i w t}].  The fixture prints
    10 digits, and the fp64 input h limits the agreement to ~1e-11 at 2 mHz."""
    import json
    import os
    g = json.load(open(os.path.join(golden_dir, "worked_example_p2.json")))
    beta, lam, psi, iota, A, f = 0.2, 1.0, 0.3, 0.5, 1e-22, 2e-3
    dt, n, t0, order = 10.0, 3000, 5.0, 25
    tab = inputs.orbit_table("static", t0, t0 + n * dt, const_ltt=inputs.ARM / inputs.C_LIGHT)
    t = t0 + dt * np.arange(n)
    w = 2 * np.pi * f
    hp = A * (1 + np.cos(iota) ** 2) * np.cos(w * t)
    hc = -2 * A * np.cos(iota) * np.sin(w * t)
    for path in ("per_sample", "fir3"):
        outs = {}
        for gen in (1, 2):
            R = lr.Response(tab, dt, order, gen, t0=t0, channels="XYZ_AET", tdi_path=path)
            mp, mf, mb = R.margins()
            y = R.project(to_dev(hp)[None], to_dev(hc)[None], [beta], [lam], [psi])
            outs[gen] = (R.tdi(y).cpu().numpy()[0], mf, mb)
        yh = y.cpu().numpy()[0]
        for s, (i, j) in enumerate(inputs.LINKS):
            v = g["links"][f"{i}{j}"]
            want = v["re"] * np.cos(w * t) - v["im"] * np.sin(w * t)
            assert np.abs(yh[s, mp:n - mp] - want[mp:n - mp]).max() < 3e-9 * np.hypot(v["re"], v["im"]), (path, s)
        for gen in (1, 2):
            o, mf, mb = outs[gen]
            for c, name in enumerate("XYZ"):
                re, im = g["tdi"][name][f"gen{gen}"]
                want = re * np.cos(w * t) - im * np.sin(w * t)
                assert np.abs(o[c, mf:n - mb] - want[mf:n - mb]).max() < 3e-9 * np.hypot(re, im), (path, gen, name)
            for c in range(2):   # |A|, |E| (T is 3e-5 of A here: a null channel)
                basis = np.stack([np.cos(w * t[mf:n - mb]), np.sin(w * t[mf:n - mb])], axis=1)
                amp = float(np.hypot(*np.linalg.lstsq(basis, o[3 + c, mf:n - mb] * 1e24, rcond=None)[0])) * 1e-24
                assert abs(amp - g["aet_abs"][f"gen{gen}"][c]) < 1e-8 * amp
        ns = 1234   # t = 12345 s
        assert abs(yh[0, ns] - g["spot"]["y12"]) < 1e-9 * abs(g["spot"]["y12"])
        assert abs(outs[1][0][0, ns] - g["spot"]["X1"]) < 1e-9 * abs(g["spot"]["X1"])
        assert abs(outs[2][0][0, ns] - g["spot"]["X2"]) < 1e-9 * abs(g["spot"]["X2"])


def test_gpu_relabelling(lr):
    """Pin P4 on the GPU: cyclic relabelling of the spacecraft permutes (X,Y,Z) -> (Z,X,Y) of the relabelled
    run back onto (X,Y,Z); the reflection 2<->3 flips the sign of X."""
    w = inputs.config(2, n=4001, f0=3e-3, t0=2.5e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)

    def run(table):
        R = lr.Response(table, w.dt, w.order, 2, t0=w.t0)
        y = R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
        return R.tdi(y).cpu().numpy()[0], R.margins()

    base, (mp, mf, mb) = run(tab)
    cyc, _ = run(tab.relabel({1: 2, 2: 3, 3: 1}))   # new spacecraft 1 is old 2: new X = old Y
    ref, _ = run(tab.relabel({1: 1, 2: 3, 3: 2}))
    v = slice(mf, w.n - mb)
    scale = np.abs(base[:, v]).max()
    assert np.abs(cyc[0, v] - base[1, v]).max() < 1e-13 * scale
    assert np.abs(cyc[1, v] - base[2, v]).max() < 1e-13 * scale
    assert np.abs(cyc[2, v] - base[0, v]).max() < 1e-13 * scale
    assert np.abs(ref[0, v] + base[0, v]).max() < 1e-13 * scale
    assert np.abs(ref[1, v] + base[2, v]).max() < 1e-13 * scale


def test_gpu_hybrid_same_handle_bitwise(lr):
    """Pin P11: lr_tdi through a second handle built from the same table equals the same-handle run bit for
    bit; lr_response_host equals lr_project + lr_tdi bit for bit."""
    import torch
    w = inputs.config(2, n=5003, t0=1.5e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    R1 = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    R2 = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    y = R1.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
    a, b = R1.tdi(y).cpu().numpy(), R2.tdi(y).cpu().numpy()
    assert np.array_equal(a, b)
    out = np.empty((1, 6, w.n))
    R1.response_host(hp[None].copy(), hc[None].copy(), [s.beta], [s.lam], [s.psi], out)
    torch.cuda.synchronize()
    assert np.array_equal(out, a)


@pytest.mark.parametrize("tdi_path", ["auto", "per_sample", "fir4"])
def test_gpu_response_chunked_bitwise(lr, tdi_path):
    """lr_response (device, chunked through the small y scratch) and lr_response_host (pipelined copies) equal
    lr_project + lr_tdi bit for bit: 11 templates (two template chunks), 30,011 samples in chunks of 7,168
    (ragged last chunk), and the automatic single-chunk case; hybrid second handle included."""
    import torch
    w = inputs.config(3, batch=11, n=30011)
    tab = w.table()
    hp, hc = _stack(w, range(11))
    beta, lam, psi = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    eq = inputs.orbit_table("eq", w.t0, w.t0 + w.n * w.dt, const_ltt=inputs.ARM / inputs.C_LIGHT)
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET", tdi_path=tdi_path)
    R1 = lr.Response(eq, w.dt, w.order, 1, t0=w.t0, channels="AET", tdi_path=tdi_path)
    hpd, hcd = to_dev(hp), to_dev(hc)
    y = R.project(hpd, hcd, beta, lam, psi)
    for Rt in (R, R1):
        ref = Rt.tdi(y).cpu().numpy()
        for chunk in (0, 7168, 1792):
            lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, chunk)
            got = R.response(hpd, hcd, beta, lam, psi, tdi=Rt)
            torch.cuda.synchronize()
            assert np.array_equal(got.cpu().numpy(), ref), (tdi_path, chunk)
            out = torch.empty(ref.shape, dtype=torch.float64).pin_memory()
            R.response_host(torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory(), beta, lam, psi, out,
                            tdi=Rt)
            assert np.array_equal(out.numpy(), ref), (tdi_path, chunk, "host")
    # pageable host buffers work too
    lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, 7168)
    out = np.empty((11, 6, w.n))
    R.response_host(hp.copy(), hc.copy(), beta, lam, psi, out)
    assert np.array_equal(out, R.tdi(y).cpu().numpy())


@pytest.mark.parametrize("world", [2, 3])
def test_gpu_time_sharded_spans_bitwise(lr, world):
    """Time-axis sharding: every "rank" gets only its slice of h (span + halo, its own device
    tensors) and computes its span with lr_response_span; the concatenation equals the whole-series result bit
    for bit.  The ranks are run one after the other on the one GPU (they never wait on each other)."""
    import torch
    w = inputs.config(2, n=50021, f0=2e-3, t0=3.0e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    ref = R.tdi(R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])).cpu().numpy()
    lo, hi, unit = R.span_halo()
    got = np.full_like(ref, np.nan)
    for rank in range(world):
        first, count, h_first, h_len = lr.shard_time(w.n, rank, world, unit, lo, hi)
        Rk = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")     # the rank's own handle
        hps = to_dev(hp[h_first:h_first + h_len].copy())[None]
        hcs = to_dev(hc[h_first:h_first + h_len].copy())[None]
        out = Rk.response_span(hps, hcs, h_first, [s.beta], [s.lam], [s.psi], w.n, first, count)
        torch.cuda.synchronize()
        got[:, :, first:first + count] = out.cpu().numpy()
    assert np.array_equal(got, ref)
    # a slice that is too short is refused, as is a span that does not start on a unit
    first, count, h_first, h_len = lr.shard_time(w.n, 1, 2, unit, lo, hi)
    with pytest.raises(lr.LrError):
        R.response_span(to_dev(hp[first:first + count].copy())[None], to_dev(hc[first:first + count].copy())[None],
                        first, [s.beta], [s.lam], [s.psi], w.n, first, count)
    with pytest.raises(lr.LrError):
        R.response_span(to_dev(hp)[None], to_dev(hc)[None], 0, [s.beta], [s.lam], [s.psi], w.n, 100, 1000)


def test_gpu_non_default_stream(lr):
    """Every call enqueues on the stream it is given: the same results on a side stream (torch.cuda.Stream) as on
    the default stream, for the two-call path, the one-call paths and the host-buffer pipeline; a plan built on
    one stream is reused safely from another."""
    import torch
    w = inputs.config(2, n=30011, f0=5e-3, t0=2.0e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    hpd, hcd = to_dev(hp)[None], to_dev(hc)[None]
    ref = R.tdi(R.project(hpd, hcd, [s.beta], [s.lam], [s.psi])).cpu().numpy()      # default stream, builds the plan
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        y = R.project(hpd, hcd, [s.beta], [s.lam], [s.psi], stream=side)
        a = R.tdi(y, stream=side)
        b = R.response(hpd, hcd, [s.beta], [s.lam], [s.psi], stream=side)
        out = torch.empty(ref.shape, dtype=torch.float64).pin_memory()
        R.response_host(torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory(), [s.beta], [s.lam],
                        [s.psi], out, stream=side)
    side.synchronize()
    assert np.array_equal(a.cpu().numpy(), ref) and np.array_equal(b.cpu().numpy(), ref)
    assert np.array_equal(out.numpy(), ref)


def test_gpu_orbit_spline_matches_oracle(lr):
    """Orbit ingestion (lr_create's device spline) against the oracle's spline and scipy's not-a-knot
    CubicSpline at random times: positions to 1e-15 relative, light times to 1e-15 s."""
    import torch
    from scipy.interpolate import CubicSpline
    w = inputs.config(4, n=1000)
    tab = w.table()
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0)
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    rng = np.random.default_rng(3)
    t_end = tab.t_start + (tab.n_knots - 1) * tab.knot_dt
    t = np.sort(rng.uniform(tab.t_start, t_end, size=5000))
    tk = tab.t_start + tab.knot_dt * np.arange(tab.n_knots)
    td = to_dev(t)
    for ch in range(15):
        out = torch.empty_like(td)
        lr.lr_eval_orbit(R.handle, ch, td, out)
        g = out.cpu().numpy()
        o = O.spline(ch, t.astype(np.longdouble))
        table = tab.x.reshape(9, -1)[ch] if ch < 9 else tab.ltt[ch - 9]
        sp = CubicSpline(tk, table, bc_type="not-a-knot")(t)
        scale = np.abs(table).max()
        assert np.abs(g - o.astype(np.float64)).max() < 4e-15 * scale, ch
        assert np.abs(g - sp).max() < 1e-13 * scale, ch


def test_tdi_plan_cache(lr):
    """The FIR plan is a function of the orbits and the time grid only: with the cache on, a second call with
    another y, a call after a change of t0 / n / chain mode, and a cache-off call all give bit-identical
    results to a fresh handle."""
    w = inputs.config(2, n=6007, f0=3e-3, t0=3.0e7)
    tab = w.table()
    rng = np.random.default_rng(11)

    def fresh(y, n, t0, chain):
        R = lr.Response(tab, w.dt, w.order, 2, t0=t0, chain=chain, tdi_path="fir3")
        R.set_plan_cache(False)
        return R.tdi(to_dev(y[:, :n])[None]).cpu().numpy()

    ya, yb = (np.cumsum(rng.normal(size=(6, w.n)), axis=1) * 1e-3 for _ in range(2))
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, tdi_path="fir3")
    assert np.array_equal(R.tdi(to_dev(ya)[None]).cpu().numpy(), fresh(ya, w.n, w.t0, "nested"))
    assert np.array_equal(R.tdi(to_dev(yb)[None]).cpu().numpy(), fresh(yb, w.n, w.t0, "nested"))   # plan reused
    R.set_chain("sum")
    assert np.array_equal(R.tdi(to_dev(yb)[None]).cpu().numpy(), fresh(yb, w.n, w.t0, "sum"))
    R.set_chain("nested")
    lr.lr_set_option(R.handle, lr.LR_OPT_T0, w.t0 + 12345.0)
    assert np.array_equal(R.tdi(to_dev(ya)[None]).cpu().numpy(), fresh(ya, w.n, w.t0 + 12345.0, "nested"))
    assert np.array_equal(R.tdi(to_dev(ya[:, :5000].copy())[None]).cpu().numpy(), fresh(ya, 5000, w.t0 + 12345.0, "nested"))
    # one plan, several templates in one launch
    both = R.tdi(to_dev(np.stack([ya[:, :5000], yb[:, :5000]]))).cpu().numpy()
    assert np.array_equal(both[1:], fresh(yb, 5000, w.t0 + 12345.0, "nested"))


def test_plan_rebuilt_once_per_call_with_flagged_tiles(lr):
    """LR_OPT_TDI_PLAN_CACHE = 0 with more than 8 templates (two template chunks, several time chunks) and tiles the
    plan flags: the plan is rebuilt once per call, behind every fix-up kernel that still reads the old list, and the
    result equals the cached-plan two-call path bit for bit (the rebuild used to race with the deferred
    fix-up kernel of the previous chunk)."""
    import torch
    dt, n, t0, order = 10.0, 40000, 3.0e7, 9
    base = inputs.orbit_table("kepler", t0, t0 + n * dt)
    tk = base.t_start + base.knot_dt * np.arange(base.n_knots)
    ltt = np.tile(10.0 + 2e-9 * (tk - (t0 + 0.5 * n * dt)), (6, 1)) * (1 + 1e-7 * np.arange(6))[:, None]
    tab = inputs.OrbitTable(base.t_start, base.knot_dt, base.x, np.ascontiguousarray(ltt))
    w = inputs.config(3, batch=11, n=n, t0=t0)
    hp, hc = _stack(w, range(11))
    hpd, hcd = to_dev(hp), to_dev(hc)
    beta, lam, psi = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    R = lr.Response(tab, dt, order, 2, t0=t0, tdi_path="fir3")
    ref = R.tdi(R.project(hpd, hcd, beta, lam, psi)).cpu().numpy()
    Rn = lr.Response(tab, dt, order, 2, t0=t0, tdi_path="fir3")
    Rn.set_plan_cache(False)
    lr.lr_set_option(Rn.handle, lr.LR_OPT_CHUNK_SAMPLES, 1792 * 3)
    for _ in range(4):
        l0 = lr.lr_launch_count()
        got = Rn.response(hpd, hcd, beta, lam, psi)
        torch.cuda.synchronize()
        assert np.array_equal(got.cpu().numpy(), ref)
        chunks = 2 * -(-n // (1792 * 3))
        # source basis x2, ONE plan kernel, per chunk: projection + apply (+ fix-up where a flagged tile lies)
        assert 2 + 1 + 2 * chunks <= lr.lr_launch_count() - l0 <= 2 + 1 + 3 * chunks
    assert np.array_equal(Rn.tdi(R.project(hpd, hcd, beta, lam, psi)).cpu().numpy(), ref)


def test_shared_plan_two_streams_bitwise(lr):
    """lr_plan_create / lr_plan_attach (orbit information pre-computed once for the whole run): two
    handles on two streams share ONE read-only plan; results equal a handle's own plan bit for bit; no plan kernel
    runs in the attached handles; the plan outlives the handle that built it; a call on another grid falls back to
    the handle's own plan; a plan of other orbits is refused."""
    import torch
    w = inputs.config(2, n=60011, f0=3e-3, t0=3.0e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    mk = lambda: lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    Ra = mk()
    y1 = Ra.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
    y2 = (y1 * 0.5).contiguous()
    ref1, ref2 = Ra.tdi(y1).cpu().numpy(), Ra.tdi(y2).cpu().numpy()
    plan = lr.lr_plan_create(Ra.handle, w.n)
    assert lr.lr_plan_bytes(plan) > 12 * 31 * 3 * 8 * (w.n // 224)
    Ra.close()                                     # the creator goes, the plan stays
    Rc, Rd = mk(), mk()
    lr.lr_plan_attach(Rc.handle, plan)
    lr.lr_plan_attach(Rd.handle, plan)
    lr.lr_plan_release(plan)                       # the attached handles hold the remaining references
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    s1.wait_stream(torch.cuda.current_stream())
    s2.wait_stream(torch.cuda.current_stream())
    l0 = lr.lr_launch_count()
    for _ in range(3):
        o1 = Rc.tdi(y1, stream=s1)
        o2 = Rd.tdi(y2, stream=s2)
    s1.synchronize()
    s2.synchronize()
    assert lr.lr_launch_count() - l0 <= 6 * 2      # apply (+ fix-up) per call: no plan kernel
    assert np.array_equal(o1.cpu().numpy(), ref1) and np.array_equal(o2.cpu().numpy(), ref2)
    # another grid: the attached plan does not fit, the handle builds its own
    m = 30011
    Re = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    short = y1[:, :, :m].contiguous()
    assert np.array_equal(Rc.tdi(short).cpu().numpy(), Re.tdi(short).cpu().numpy())
    assert np.array_equal(Rc.tdi(y1).cpu().numpy(), ref1)          # and the shared one still serves its grid
    # other orbits / other order: refused
    other = lr.Response(inputs.orbit_table("eq", w.t0, w.t0 + w.n * w.dt), w.dt, w.order, 2, t0=w.t0)
    p2 = lr.lr_plan_create(Rc.handle, w.n)
    with pytest.raises(lr.LrError) as e:
        lr.lr_plan_attach(other.handle, p2)
    assert e.value.code == lr.LR_EINVAL
    lr.lr_plan_attach(Rc.handle, None)
    lr.lr_plan_release(p2)
    Rp = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, tdi_path="per_sample")
    with pytest.raises(lr.LrError):
        lr.lr_plan_create(Rp.handle, w.n)


def test_project_and_tdi_replay_from_a_cuda_graph(lr):
    """lr_project (parameter-buffer staging, batch <= 16) and lr_tdi can be captured into a CUDA graph once the plan
    exists: the tiny config (launch-latency bound: three launches) replays bit-identically, new inputs written into
    the captured buffers give the results of direct calls, and the calls that cannot be captured say so (LR_EINVAL)
    without breaking the capture."""
    import torch
    w = inputs.config(1)
    s = w.sources[0]
    hp, hc = w.waveform(0)
    hpd, hcd = to_dev(hp)[None].clone(), to_dev(hc)[None].clone()
    R = lr.Response(w.table(), w.dt, w.order, 1, t0=w.t0)
    y = torch.empty((1, 6, w.n), dtype=torch.float64, device="cuda")
    out = torch.empty((1, 3, w.n), dtype=torch.float64, device="cuda")
    for _ in range(2):                                     # outside a capture first: builds the plan
        R.project(hpd, hcd, [s.beta], [s.lam], [s.psi], y_out=y)
        R.tdi(y, out=out)
    torch.cuda.synchronize()
    ref = out.clone()
    st = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    refused = None
    with torch.cuda.graph(g, stream=st):
        R.project(hpd, hcd, [s.beta], [s.lam], [s.psi], y_out=y, stream=st)
        R.tdi(y, out=out, stream=st)
        try:
            R.response(hpd, hcd, [s.beta], [s.lam], [s.psi], out=out, stream=st)
        except lr.LrError as e:
            refused = e.code
    assert refused == lr.LR_EINVAL
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    # direct calls afterwards (bigger batches: the ring of staging slots is reallocated) leave the graph's own
    # staging slot alone
    wb = inputs.config(3, batch=19, n=w.n, t0=w.t0)
    hb, cb = _stack(wb, range(19))
    for nb in (19, 3, 19, 1, 5):
        R.project(to_dev(hb[:nb]), to_dev(cb[:nb]), [x.beta for x in wb.sources[:nb]], [x.lam for x in wb.sources[:nb]],
                  [x.psi for x in wb.sources[:nb]])
    torch.cuda.synchronize()
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    hpd.mul_(0.5)                                          # new input in the captured buffers
    hcd.mul_(0.5)
    g.replay()
    torch.cuda.synchronize()
    got = out.clone()
    want = R.tdi(R.project(hpd, hcd, [s.beta], [s.lam], [s.psi]))
    torch.cuda.synchronize()
    assert torch.equal(got, want)
    assert np.array_equal(R.tdi(R.project(hpd * 2, hcd * 2, [s.beta], [s.lam], [s.psi])).cpu().numpy(), ref.cpu().numpy())
    # a series with flagged tiles: the capture then holds the fork to the handle's side stream, the fix-up kernel and
    # the join back (light times that cross a whole number of samples in the middle of the series)
    dt, n, t0, order = 10.0, 40000, 3.0e7, 9
    base = inputs.orbit_table("kepler", t0, t0 + n * dt)
    tk = base.t_start + base.knot_dt * np.arange(base.n_knots)
    ltt = np.tile(10.0 + 2e-9 * (tk - (t0 + 0.5 * n * dt)), (6, 1)) * (1 + 1e-7 * np.arange(6))[:, None]
    tab = inputs.OrbitTable(base.t_start, base.knot_dt, base.x, np.ascontiguousarray(ltt))
    w2 = inputs.config(2, n=n, t0=t0)
    hp2, hc2 = w2.waveform(0)
    s2 = w2.sources[0]
    hp2d, hc2d = to_dev(hp2)[None], to_dev(hc2)[None]
    R2 = lr.Response(tab, dt, order, 2, t0=t0, tdi_path="fir3")
    y2 = torch.empty((1, 6, n), dtype=torch.float64, device="cuda")
    o2 = torch.empty((1, 3, n), dtype=torch.float64, device="cuda")
    for _ in range(2):
        R2.project(hp2d, hc2d, [s2.beta], [s2.lam], [s2.psi], y_out=y2)
        R2.tdi(y2, out=o2)
    torch.cuda.synchronize()
    ref2 = o2.clone()
    g2 = torch.cuda.CUDAGraph()
    l0 = lr.lr_launch_count()
    with torch.cuda.graph(g2, stream=st):
        R2.project(hp2d, hc2d, [s2.beta], [s2.lam], [s2.psi], y_out=y2, stream=st)
        R2.tdi(y2, out=o2, stream=st)
    assert lr.lr_launch_count() - l0 == 4                  # source basis, projection, fix-up, apply
    for _ in range(3):
        o2.zero_()
        g2.replay()
        torch.cuda.synchronize()
        assert torch.equal(o2, ref2)


def test_shared_plan_from_two_host_threads(lr):
    """include/lr.h: handles that share a plan may be used from different host threads and streams at the same time
    (each handle from one thread).  Two threads, each with its own handle, stream, y and out, 50 lr_tdi calls each on
    one attached plan (ctypes releases the GIL during the calls): every result equals the single-threaded one."""
    import threading
    import torch
    w = inputs.config(2, n=60011, f0=3e-3, t0=3.0e7)
    tab = w.table()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    R0 = lr.Response(tab, w.dt, w.order, 2, t0=w.t0)
    y = R0.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
    ys = [y, (y * 0.25).contiguous()]
    refs = [R0.tdi(v).clone() for v in ys]
    plan = R0.create_plan(w.n)
    torch.cuda.synchronize()
    errors = []

    def worker(k):
        try:
            torch.cuda.set_device(0)
            R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0)
            R.attach_plan(plan)
            st = torch.cuda.Stream()
            out = torch.empty_like(refs[k])
            for _ in range(50):
                out.zero_()
                R.tdi(ys[k], out=out, stream=st)
                st.synchronize()
                if not torch.equal(out, refs[k]):
                    errors.append((k, "mismatch"))
                    return
            R.close()
        except Exception as e:   # pragma: no cover
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    lr.lr_plan_release(plan)
    assert not errors, errors


def test_binding_checks_out_against_the_channel_option(lr):
    """The C ABI takes no size for `out`: the binding checks it against the handle's LR_OPT_CHANNELS (lr_get_option),
    so a [B,3,N] buffer is never handed to a handle that writes six rows; angle arrays must match the batch."""
    import torch
    w = inputs.config(2, n=4001, t0=2.0e7)
    s = w.sources[0]
    hp, hc = w.waveform(0)
    R = lr.Response(w.table(), w.dt, w.order, 2, t0=w.t0, channels="XYZ_AET")
    assert lr.lr_get_option(R.handle, lr.LR_OPT_CHANNELS) == lr.LR_XYZ_AET
    assert lr.lr_get_option(R.handle, lr.LR_OPT_T0) == w.t0
    hpd, hcd = to_dev(hp)[None], to_dev(hc)[None]
    y = R.project(hpd, hcd, [s.beta], [s.lam], [s.psi])
    small = torch.empty((1, 3, w.n), dtype=torch.float64, device="cuda")
    with pytest.raises(ValueError):
        R.tdi(y, out=small)
    with pytest.raises(ValueError):
        R.response(hpd, hcd, [s.beta], [s.lam], [s.psi], out=small)
    with pytest.raises(ValueError):
        R.response_host(hp[None].copy(), hc[None].copy(), [s.beta], [s.lam], [s.psi], np.empty((1, 3, w.n)))
    with pytest.raises(ValueError):
        R.response(hpd, hcd, [s.beta], [s.lam, s.lam], [s.psi])
    R3 = lr.Response(w.table(), w.dt, w.order, 2, t0=w.t0, channels="AET")
    with pytest.raises(ValueError):
        R3.tdi(y, out=torch.empty((1, 6, w.n), dtype=torch.float64, device="cuda"))
    with pytest.raises(lr.LrError):
        lr.lr_get_option(R.handle, 99)


# ------------------------------------------------------------------------------- likelihood (NEXT-2)
def test_gpu_inner_product_parity(lr):
    """lr_inner_product against the likelihood oracle on the SAME frequency-domain arrays (numpy FFT of real
    A, E, T series of 9 templates), both modes, batch_b = batch and = 1, odd nf: relative error <= 1e-13; and
    end to end from the GPU's own TDI output through torch.fft.rfft (cuFFT) against oracle TDI + numpy FFT."""
    import torch
    from oracle import likelihood as lk
    w = inputs.config(3, batch=9, n=40001)
    tab = w.table()
    hp, hc = _stack(w, range(9))
    beta, lam, psi = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="AET")
    aet = R.response(to_dev(hp), to_dev(hc), beta, lam, psi)
    torch.cuda.synchronize()
    aet_h = aet.cpu().numpy()
    n, dt = w.n, w.dt
    f = np.fft.rfftfreq(n, dt)
    psd = inputs.psd_standin(f)
    inv = np.zeros_like(psd)
    inv[:, 1:] = 1.0 / psd[:, 1:]
    fh = lk.to_frequency(aet_h, dt)                       # [9, 3, nf]
    fd = fh[4:5]                                          # "data" = template 4 (noiseless injection)
    df = 1.0 / (n * dt)
    fh_d, fd_d, inv_d = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (fh, fd, inv))
    want = lk.inner_product(fh, fd, psd, dt, n)           # <h_b|d> for every template
    got = lr.lr_inner_product(fh_d, fd_d, inv_d, 4 * df).cpu().numpy()
    assert np.abs(got - want.astype(np.float64)).max() <= 1e-13 * np.abs(want).max()
    want = lk.inner_product(fh, fh, psd, dt, n)
    got = lr.lr_inner_product(fh_d, fh_d, inv_d, 4 * df).cpu().numpy()
    assert np.abs(got - want.astype(np.float64)).max() <= 1e-13 * np.abs(want).max()
    ll = np.array([lk.log_likelihood(fd[0], fh[b], psd, dt, n) for b in range(9)], dtype=np.float64)
    got = lr.lr_inner_product(fh_d, fd_d, inv_d, -2 * df, mode=lr.LR_IP_DIFF).cpu().numpy()
    assert got[4] == 0.0 and np.all(got[np.arange(9) != 4] < 0)
    assert np.abs(got - ll).max() <= 1e-12 * np.abs(ll).max()
    # deterministic: the same call twice gives the same bits
    assert np.array_equal(got, lr.lr_inner_product(fh_d, fd_d, inv_d, -2 * df, mode=lr.LR_IP_DIFF).cpu().numpy())
    # end to end with the library FFT on the device
    fh_gpu = (dt * torch.fft.rfft(aet, dim=-1)).contiguous()
    got = lr.lr_inner_product(fh_gpu, fh_gpu, inv_d, 4 * df).cpu().numpy()
    assert np.abs(got - want.astype(np.float64)).max() <= 1e-11 * np.abs(want).max()
    with pytest.raises(lr.LrError):
        lr.lr_inner_product(fh_d, fh_d, inv_d, 1.0, mode=7)


def test_handles_release_their_device_memory(lr):
    """lr_destroy gives back everything a handle took: spline coefficients, staging slots, the TDI plan (its own and
    a shared one once the last reference goes), the y / h / spectrum scratch of the one-call paths and the cuFFT
    plan.  Forty create / use / destroy cycles leave the free device memory where it was."""
    import gc
    import torch
    w = inputs.config(3, batch=3, n=20011)
    tab = w.table()
    hp, hc = _stack(w, range(3))
    hpd, hcd = to_dev(hp), to_dev(hc)
    be, la, ps = ([getattr(s, k) for s in w.sources] for k in ("beta", "lam", "psi"))
    gb = np.array([[s.A * (1.0 + np.cos(s.iota) ** 2), -2.0 * s.A * np.cos(s.iota), s.f0, s.fdot, 0.0, s.phi0]
                   for s in w.sources])
    nf = w.n // 2 + 1
    inv = torch.ones((3, nf), dtype=torch.float64, device="cuda")
    out = torch.empty((3, 3, w.n), dtype=torch.float64, device="cuda")
    y = torch.empty((3, 6, w.n), dtype=torch.float64, device="cuda")
    host_out = np.empty((3, 3, w.n))

    def cycle():
        R = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="AET")
        R.project(hpd, hcd, be, la, ps, y_out=y)
        R.tdi(y, out=out)
        R.response(hpd, hcd, be, la, ps, out=out)
        R.response_host(hp, hc, be, la, ps, host_out)
        data_f = torch.fft.rfft(out[0], dim=-1).contiguous()
        R.loglike_gb(gb, be, la, ps, w.n, data_f, inv, -2.0 * w.dt / w.n)
        plan = R.create_plan(w.n)
        R2 = lr.Response(tab, w.dt, w.order, 2, t0=w.t0, channels="AET")
        R2.attach_plan(plan)
        lr.lr_plan_release(plan)
        R2.tdi(y, out=out)
        torch.cuda.synchronize()
        del data_f
        R.close()
        R2.close()

    for _ in range(3):          # the library's and torch's one-time allocations (cuFFT module, caching allocator)
        cycle()
    gc.collect()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(40):
        cycle()
    gc.collect()
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free0 - free1 <= 4 << 20, f"{(free0 - free1) / 2**20:.1f} MiB of device memory not returned after 40 cycles"


# ---------------------------------------------------------------------------------------- edge cases
def test_edge_cases_and_errors(lr):
    import torch
    B = lr.binding
    w = inputs.config(1)
    tab = w.table()
    for bad_order in (0, 2, 26, 67):
        with pytest.raises(lr.LrError) as e:
            lr.lr_create(tab, w.dt, bad_order, 1)
        assert e.value.code == lr.LR_EINVAL
    with pytest.raises(lr.LrError):
        lr.lr_create(tab, w.dt, 25, 3)
    with pytest.raises(lr.LrError):
        lr.lr_create(tab, -1.0, 25, 1)
    R = lr.Response(tab, w.dt, w.order, 1, t0=w.t0)
    mp, mf, mb = R.margins()
    s = w.sources[0]
    # n <= 2 m_proj: nothing valid -> LR_EINVAL ("empty" input)
    n = 2 * mp
    h = torch.zeros((1, n), dtype=torch.float64, device="cuda")
    with pytest.raises(lr.LrError) as e:
        R.project(h, h, [s.beta], [s.lam], [s.psi])
    assert e.value.code == lr.LR_EINVAL
    # smallest legal sizes: one valid sample per stage
    n = 2 * mp + 1
    hp, hc = inputs.gb_waveform(n, w.dt, w.t0, s.A, s.f0, s.fdot, s.iota, s.phi0)
    y = R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi]).cpu().numpy()[0]
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    yo = O.project(hp, hc, s.beta, s.lam, s.psi)
    assert np.count_nonzero(y) == 6
    assert_parity(y[:, mp:mp + 1], yo[:, mp:mp + 1], "single valid sample")
    n = mf + mb + 1
    yy = np.random.default_rng(0).normal(size=(6, n)) * 1e-22
    out = R.tdi(to_dev(yy)[None]).cpu().numpy()[0]
    oo = O.tdi(yy, 1)
    assert np.count_nonzero(out) == 3
    assert_parity(out[:, mf:mf + 1], oo[:, mf:mf + 1], "single valid tdi sample")
    with pytest.raises(lr.LrError) as e:
        R.tdi(to_dev(yy[:, :-1])[None])
    assert e.value.code == lr.LR_EINVAL
    # sample span outside the knot table -> LR_ERANGE, no extrapolation
    R2 = lr.Response(tab, w.dt, w.order, 1, t0=w.t0 + 40 * 86400.0)
    hp, hc = w.waveform(0)
    with pytest.raises(lr.LrError) as e:
        R2.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
    assert e.value.code == lr.LR_ERANGE
    assert "orbit table" in B.lr_strerror(lr.LR_ERANGE)
    # NaN propagates, does not crash
    hp2 = hp.copy()
    hp2[5000] = np.nan
    R3 = lr.Response(tab, w.dt, w.order, 1, t0=w.t0)
    y = R3.project(to_dev(hp2)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi]).cpu().numpy()[0]
    assert np.isnan(y).any() and np.isfinite(y[:, mp:4000]).all()


# ------------------------------------------------------------------------------------- seeded random sweep
@pytest.mark.parametrize("seed", range(40))
def test_random_configurations(lr, seed):
    """Seeded draws over the whole option space at sizes that span several tiles and a ragged tail: order 1-41,
    dt 2-20 s, generation, chain form, channel set, orbit family (equal-arm constant, Keplerian, perturbed),
    batch 1-3, TDI path, start time; lr_project + lr_tdi against the oracle (check_workload), then lr_response in
    odd chunks against the two-call result bit for bit."""
    import torch
    rng = np.random.default_rng(1000 + seed)
    order = int(rng.choice([1, 3, 5, 7, 9, 11, 13, 15, 21, 25, 31, 41]))
    dt = float(rng.choice([2.0, 5.0, 10.0, 15.0, 20.0]))
    gen = int(rng.choice([1, 2]))
    chain = str(rng.choice(["nested", "sum"]))
    channels = str(rng.choice(["XYZ", "AET", "XYZ_AET"]))
    kind = str(rng.choice(["eq", "kepler", "perturbed"]))
    batch = int(rng.integers(1, 4))
    n = int(rng.integers(2500, 5200))
    t0 = float(rng.uniform(1e6, 9e7))
    tdi_path = str(rng.choice(["auto", "per_sample", "fir3", "fir4"]))
    if kind == "eq":
        channels = "XYZ"   # T of exactly equal arms is a null (3e-5 of A): test_tdi_null_channel_absolute covers it
    srcs = [inputs.draw_gb(np.random.default_rng(50 * seed + b)) for b in range(batch)]
    w = inputs.Workload(f"random{seed}", n, dt, t0, order, gen, kind, 7 + seed,
                        inputs.ARM / inputs.C_LIGHT if kind == "eq" else None, srcs, channels=channels)
    errs, yh, oh = check_workload(lr, w, chain=chain, idx=tuple(range(batch)), tdi_path=tdi_path)
    R = lr.Response(w.table(), dt, order, gen, t0=t0, chain=chain, channels=channels, tdi_path=tdi_path)
    lr.lr_set_option(R.handle, lr.LR_OPT_CHUNK_SAMPLES, 1792 * int(rng.integers(1, 3)))
    hp, hc = _stack(w, range(batch))
    beta, lam, psi = ([getattr(s, k) for s in srcs] for k in ("beta", "lam", "psi"))
    out = R.response(to_dev(hp), to_dev(hc), beta, lam, psi)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oh), (order, dt, gen, chain, channels, kind, batch, n, tdi_path)
