"""Parity report: the three error tables of SURVEY.md §8(c) per configuration, as markdown.

  (i)   lr_project vs the oracle's projection of the same h              (bar 1e-10)
  (ii)  lr_tdi vs the oracle's TDI of the GPU's own fp64 y               (bar 1e-10)
  (iii) end to end (GPU h -> out) vs the all-long-double oracle, beside the floor any fp64-y interface
        has: long-double TDI of fp64-rounded long-double y vs long-double TDI of long-double y (information).

Run on a GPU box:  python tests/parity_report.py > gpurun_out/parity_report.md
Test infrastructure: imports oracle/.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle import oracle as orc  # noqa: E402
from harness import inputs  # noqa: E402
from parity_util import CH_NAMES, ORC_CH, channel_errors, to_dev  # noqa: E402


def fmt(errs):
    return " ".join(f"{r:.1e}/{m:.1e}" for r, m in errs)


def report(name, w, lr, chain="nested", tab=None, y_precision="plain"):
    tab = tab or w.table()
    n, gen, ch = w.n, w.tdi_gen, "XYZ_AET"
    R = lr.Response(tab, w.dt, w.order, gen, t0=w.t0, chain=chain, channels=ch)
    R.set_y_precision(y_precision)
    if y_precision != "plain":
        name += f", LR_Y_{y_precision.upper()}"
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    mp, mf, mb = R.margins()
    s = w.sources[0]
    hp, hc = w.waveform(0)
    y = R.project(to_dev(hp)[None], to_dev(hc)[None], [s.beta], [s.lam], [s.psi])
    out = R.tdi(y).cpu().numpy()[0]
    yh = y.cpu().numpy()[0]
    yo = O.project(hp, hc, s.beta, s.lam, s.psi)                      # long double y
    e1 = [channel_errors(yh[c, mp:n - mp], yo[c, mp:n - mp]) for c in range(6)]
    nested = chain == "nested"
    o_same = O.tdi(yh, gen, nested=nested, channels=ORC_CH[ch])        # oracle TDI of the GPU's y
    e2 = [channel_errors(out[c, mf:n - mb], o_same[c, mf:n - mb]) for c in range(6)]
    o_ld = O.tdi(yo, gen, nested=nested, channels=ORC_CH[ch])          # all long double
    e3 = [channel_errors(out[c, mf:n - mb], o_ld[c, mf:n - mb]) for c in range(6)]
    o_floor = O.tdi(yo.astype(np.float64), gen, nested=nested, channels=ORC_CH[ch])
    e4 = [channel_errors(o_floor[c, mf:n - mb].astype(np.float64), o_ld[c, mf:n - mb]) for c in range(6)]
    print(f"### {name} (n={n}, dt={w.dt}, order={w.order}, gen={gen}, {chain}, f0={s.f0:.3g})\n")
    print("relative L2 / max-abs÷max|channel| per channel\n")
    print(f"- (i) lr_project, links {' '.join(['12','23','31','13','32','21'])}: {fmt(e1)}")
    print(f"- (ii) lr_tdi on the GPU's y, {' '.join(CH_NAMES[ch])}: {fmt(e2)}")
    print(f"- (iii) end to end vs long-double pipeline: {fmt(e3)}")
    print(f"- floor of an fp64 y interface: {fmt(e4)}\n")
    worst = max(max(r, m) for r, m in e1 + e2)
    print(f"worst per-call error: {worst:.2e} ({'PASS' if worst <= 1e-10 else 'FAIL'} at 1e-10)\n", flush=True)
    return worst


def main():
    import torch
    import paper_2204_06633_b200 as lr
    assert torch.cuda.is_available()
    print("# Parity report (GPU vs CPU oracle)\n")
    print(f"device: {torch.cuda.get_device_name(0)}\n")
    worst = 0.0
    w = inputs.config(1)
    worst = max(worst, report("config 1 tiny (constant equal L, gen 1)", w, lr))
    w2 = inputs.config(1)
    w2.tdi_gen = 2
    worst = max(worst, report("config 1 tiny, EQ orbits with fixed-point L, gen 2", w2, lr,
                              tab=inputs.orbit_table("eq", w2.t0, w2.t0 + w2.n * w2.dt)))
    for f0 in (None, 1e-4, 1e-3, 1e-2):
        for chain in ("nested", "sum"):
            worst = max(worst, report("config 2 year (shortened)", inputs.config(2, n=20011, f0=f0, t0=3.0e7), lr, chain))
        worst = max(worst, report("config 2 year (shortened)", inputs.config(2, n=20011, f0=f0, t0=3.0e7), lr,
                                  y_precision="extended"))
    worst = max(worst, report("config 3 batch, template 0 (shortened)", inputs.config(3, batch=1, n=20011), lr))
    for f0 in (None, 1e-4):
        for yp in ("plain", "extended"):
            worst = max(worst, report("config 4 numerical-style orbits (shortened)",
                                      inputs.config(4, n=12345, t0=5.0e7, f0=f0), lr, y_precision=yp))
    full = inputs.config(5)
    n = 30001
    w5 = inputs.config(5, n=n, t0=full.t0 + (full.n - n) * full.dt)
    hp, hc = full.waveform(0)
    w5.waveform = lambda b=0: (hp[-n:].copy(), hc[-n:].copy())
    w5.sources[0].f0 = float("nan")
    worst = max(worst, report("config 5 chirp (last 30,001 samples)", w5, lr))
    print(f"## overall worst per-call error: {worst:.2e}")


if __name__ == "__main__":
    main()
