"""Shared helpers of the GPU parity tests: run liblr through its C ABI (ctypes binding) and the CPU oracle
on the same seeded inputs and compare per channel.

Bar (BASELINE.json north_star): relative L2 error <= 1e-10 per channel and max abs error <= 1e-10 x
max|channel|, per call, on the valid region (outside the margins both sides are exactly 0).
"""
from __future__ import annotations

import numpy as np

REL_L2_TOL = 1e-10
MAX_ABS_TOL = 1e-10
LD = np.longdouble


def channel_errors(g, o):
    """(relative L2, max abs / max|o|) of one channel; g fp64 (GPU), o long double (oracle)."""
    o = np.asarray(o, dtype=LD)
    d = np.asarray(g, dtype=LD) - o
    den = np.sqrt((o * o).sum())
    mx = np.abs(o).max()
    if den == 0 or mx == 0:
        return (0.0, 0.0) if not np.any(d) else (np.inf, np.inf)
    return float(np.sqrt((d * d).sum()) / den), float(np.abs(d).max() / mx)


def assert_parity(g, o, what, names=None, rel_tol=REL_L2_TOL, abs_tol=MAX_ABS_TOL):
    """g, o: [channels, samples].  Returns the list of (rel, maxabs)."""
    out = []
    for c in range(o.shape[0]):
        r, m = channel_errors(g[c], o[c])
        out.append((r, m))
        nm = names[c] if names else str(c)
        assert r <= rel_tol, f"{what} channel {nm}: relative L2 {r:.3e} > {rel_tol:g}"
        assert m <= abs_tol, f"{what} channel {nm}: max abs {m:.3e} x max|channel| > {abs_tol:g}"
    return out


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def windows(lo, hi, width, count, seed):
    """`count` windows [a, a+width) inside [lo, hi): the first, the last and seeded random ones."""
    if hi - lo <= width:
        return [(lo, hi)]
    rng = np.random.default_rng(seed)
    starts = [lo, hi - width] + [int(s) for s in rng.integers(lo, hi - width, size=max(0, count - 2))]
    return [(s, s + width) for s in starts]


LINK_NAMES = ["y12", "y23", "y31", "y13", "y32", "y21"]
CH_NAMES = {"XYZ": ["X", "Y", "Z"], "AET": ["A", "E", "T"], "XYZ_AET": ["X", "Y", "Z", "A", "E", "T"]}
ORC_CH = {"XYZ": 0, "AET": 1, "XYZ_AET": 2}
