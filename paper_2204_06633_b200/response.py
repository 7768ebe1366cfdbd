"""Convenience wrapper around the lr_* calls (allocation of outputs, option handling, batch sharding).

No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np

from . import binding as B

_CHANNELS = {"XYZ": B.LR_XYZ, "AET": B.LR_AET, "XYZ_AET": B.LR_XYZ_AET}


def shard_templates(batch, rank, world):
    """Contiguous slice [lo, hi) of `batch` templates owned by `rank` of `world` (no collective is needed:
    templates are independent).  The first batch % world ranks get one template more."""
    if world < 1 or not 0 <= rank < world or batch < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_time(n, rank, world, unit, lo, hi):
    """Span [first, first+count) of a series of n samples owned by `rank` of `world`, with starts on multiples of
    `unit`, and the slice [h_first, h_first+h_len) of h that rank must hold (its span plus the halo (lo, hi) of
    lr_get_span_halo, clipped to the series).  The spans partition [0, n); no collective is needed (SURVEY.md
    §8(e): halos are recomputed, not exchanged).  Ranks beyond the number of units get count = 0."""
    if world < 1 or not 0 <= rank < world or n < 1 or unit < 1:
        raise ValueError("bad shard arguments")
    units = -(-n // unit)
    a, b = shard_templates(units, rank, world)
    first, end = min(a * unit, n), min(b * unit, n)
    h_first, h_end = max(0, first - lo), min(n, end + hi)
    return first, end - first, h_first, (h_end - h_first if end > first else 0)


def gather_scalars(local, batch, rank, world, group=None):
    """The one exchange step of the path: every rank has the log-likelihoods of ITS templates
    (`shard_templates(batch, rank, world)`); afterwards every rank has all `batch` of them, in template order.
    One all-gather of at most ceil(batch / world) doubles per rank (NCCL for CUDA tensors, gloo for CPU ones);
    shards of unequal length are padded for the collective and trimmed afterwards."""
    import torch
    import torch.distributed as dist
    lo, hi = shard_templates(batch, rank, world)
    if local.numel() != hi - lo:
        raise ValueError("local must hold this rank's shard of the batch")
    if world == 1:
        return local.clone()
    width = -(-batch // world)
    padded = torch.zeros(width, dtype=local.dtype, device=local.device)
    padded[:hi - lo] = local
    gathered = torch.empty(world * width, dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(gathered, padded, group=group)
    parts = []
    for r in range(world):
        a, b = shard_templates(batch, r, world)
        parts.append(gathered[r * width:r * width + (b - a)])
    return torch.cat(parts)


class Response:
    """One orbit table + (dt, order, TDI generation): owns an lr_handle."""

    def __init__(self, table, dt, order=25, tdi_gen=2, t0=None, chain="nested", channels="XYZ", tdi_path="auto"):
        self._h = None
        self._h = B.lr_create(table, dt, order, tdi_gen)
        self.dt, self.order, self.tdi_gen = dt, order, tdi_gen
        if t0 is not None:
            B.lr_set_option(self._h, B.LR_OPT_T0, t0)
        self.set_chain(chain)
        self.set_channels(channels)
        if tdi_path != "auto":
            self.set_tdi_path(tdi_path)

    @property
    def handle(self):
        return self._h

    def set_chain(self, chain):
        B.lr_set_option(self._h, B.LR_OPT_CHAIN, {"nested": B.LR_CHAIN_NESTED, "sum": B.LR_CHAIN_SUM}[chain])

    def set_channels(self, channels):
        B.lr_set_option(self._h, B.LR_OPT_CHANNELS, _CHANNELS[channels])
        self.n_out = 6 if channels == "XYZ_AET" else 3

    def set_tdi_path(self, path):
        """"auto" | "per_sample" | "fir3" | "fir4" (LR_OPT_TDI_PATH)."""
        B.lr_set_option(self._h, B.LR_OPT_TDI_PATH, {"auto": B.LR_TDI_AUTO, "per_sample": B.LR_TDI_PER_SAMPLE,
                                                     "fir3": B.LR_TDI_FIR3, "fir4": B.LR_TDI_FIR4}[path])

    def set_proj_path(self, path):
        """"auto" | "single" | "pair" (LR_OPT_PROJ_PATH)."""
        B.lr_set_option(self._h, B.LR_OPT_PROJ_PATH, {"auto": B.LR_PROJ_AUTO, "single": B.LR_PROJ_SINGLE,
                                                      "pair": B.LR_PROJ_PAIR}[path])

    def set_y_precision(self, mode):
        """"plain" | "extended" (LR_OPT_Y_PRECISION)."""
        B.lr_set_option(self._h, B.LR_OPT_Y_PRECISION, {"plain": B.LR_Y_PLAIN, "extended": B.LR_Y_EXTENDED}[mode])

    def create_plan(self, n, stream=None):
        """A shareable read-only TDI plan for this handle's options and a series of n samples (lr_plan_create)."""
        return B.lr_plan_create(self._h, n, stream)

    def attach_plan(self, plan):
        B.lr_plan_attach(self._h, plan)

    def set_plan_cache(self, on):
        B.lr_set_option(self._h, B.LR_OPT_TDI_PLAN_CACHE, 1 if on else 0)

    def set_tdi_gen(self, gen):
        B.lr_set_option(self._h, B.LR_OPT_TDI_GEN, gen)
        self.tdi_gen = gen

    def tdi_info(self):
        """(resolved lr_tdi path, FIR taps per series, accumulators per sample) of this handle (LR_INFO_*)."""
        g = lambda k: int(B.lr_get_option(self._h, k))
        path = {B.LR_TDI_PER_SAMPLE: "per_sample", B.LR_TDI_FIR3: "fir3", B.LR_TDI_FIR4: "fir4"}[g(B.LR_INFO_TDI_PATH)]
        return path, g(B.LR_INFO_FIR_TAPS), g(B.LR_INFO_FIR_POWERS)

    def margins(self):
        return B.lr_get_margins(self._h)

    def project(self, h_plus, h_cross, beta, lam, psi, y_out=None, stream=None):
        import torch
        h_plus = h_plus.reshape(-1, h_plus.shape[-1])
        b, n = h_plus.shape
        if y_out is None:
            y_out = torch.empty((b, 6, n), dtype=torch.float64, device=h_plus.device)
        return B.lr_project(self._h, h_plus, h_cross, beta, lam, psi, y_out, stream)

    def tdi(self, y, out=None, stream=None):
        import torch
        b, _, n = y.shape
        if out is None:
            out = torch.empty((b, self.n_out, n), dtype=torch.float64, device=y.device)
        return B.lr_tdi(self._h, y, out, b, stream)

    def response(self, h_plus, h_cross, beta, lam, psi, out=None, tdi=None, stream=None):
        """h -> out on the device without a [B,6,N] array (lr_response)."""
        import torch
        h_plus = h_plus.reshape(-1, h_plus.shape[-1])
        b, n = h_plus.shape
        t = tdi or self
        if out is None:
            out = torch.empty((b, t.n_out, n), dtype=torch.float64, device=h_plus.device)
        return B.lr_response(self._h, t._h, h_plus, h_cross, beta, lam, psi, out, stream)

    def span_halo(self, tdi=None):
        return B.lr_get_span_halo(self._h, (tdi or self)._h)

    def response_span(self, h_plus, h_cross, h_first, beta, lam, psi, n, first, count, out=None, tdi=None, stream=None):
        """out[B, n_out, count] for the global samples [first, first+count) from the h slice starting at h_first."""
        import torch
        t = tdi or self
        h_plus = h_plus.reshape(-1, h_plus.shape[-1])
        if out is None:
            out = torch.empty((h_plus.shape[0], t.n_out, count), dtype=torch.float64, device=h_plus.device)
        return B.lr_response_span(self._h, t._h, h_plus, h_cross, h_first, beta, lam, psi, n, first, count, out, stream)

    def response_host(self, h_plus, h_cross, beta, lam, psi, out, tdi=None, stream=None):
        return B.lr_response_host(self._h, (tdi or self)._h, h_plus, h_cross, beta, lam, psi, out, stream)

    def gb_waveform(self, gb, n, stream=None):
        """(h_plus, h_cross) CUDA [B, n] of the Galactic binaries gb [B, 6] (eqs. 5-9)."""
        import torch
        nb = np.asarray(gb, dtype=np.float64).reshape(-1, B.LR_GB_NPAR).shape[0]
        hp = torch.empty((nb, n), dtype=torch.float64, device="cuda")
        hc = torch.empty_like(hp)
        B.lr_gb_waveform(self._h, gb, n, hp, hc, stream)
        return hp, hc

    def response_gb(self, gb, beta, lam, psi, n, out=None, tdi=None, stream=None):
        """Parameters -> TDI channels (CUDA [B, 3|6, n]); h and y only exist chunk-wise in scratch."""
        import torch
        t = tdi or self
        nb = np.asarray(gb, dtype=np.float64).reshape(-1, B.LR_GB_NPAR).shape[0]
        if out is None:
            out = torch.empty((nb, t.n_out, n), dtype=torch.float64, device="cuda")
        return B.lr_response_gb(self._h, t._h, gb, beta, lam, psi, n, out, stream)

    def set_fft_length(self, m):
        """Transform length of loglike_gb (>= n, zero padded; 0 = n).  See lr_fft_good_length."""
        B.lr_set_option(self._h, B.LR_OPT_FFT_LENGTH, int(m))
        self._fft_length = int(m)

    def loglike_gb(self, gb, beta, lam, psi, n, data_f, inv_psd, scale, mode=B.LR_IP_DIFF, out=None, tdi=None,
                   stream=None):
        """Parameters -> one scalar per template (CUDA [B]): waveform, response, FFT, noise-weighted inner product."""
        return B.lr_loglike_gb(self._h, (tdi or self)._h, gb, beta, lam, psi, n, data_f, inv_psd, scale, mode, out,
                               stream, n_fft=getattr(self, "_fft_length", 0) or None)

    def close(self):
        if self._h is not None:
            B.lr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
