"""ctypes binding of liblr (include/lr.h).  Argument marshalling only.

Every function below has the name and the meaning of the C entry point it calls; all arithmetic of the
response runs in the CUDA kernels of csrc/.  There is no CPU fallback: if liblr.so is missing or cannot
be loaded the import of the library fails loudly (`LrUnavailable`), and every computing call needs a CUDA
device.  PyTorch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("LR_LIBRARY", os.path.join(_HERE, "liblr.so"))  # override: A/B builds

LR_OK, LR_EINVAL, LR_ERANGE, LR_ECUDA, LR_ENOMEM, LR_ELIMIT = 0, -1, -2, -3, -4, -5
LR_IP_STATIC_MAX_BATCH = 64
LR_OPT_T0, LR_OPT_CHAIN, LR_OPT_CHANNELS, LR_OPT_TDI_GEN, LR_OPT_TDI_PATH = 1, 2, 3, 4, 5
LR_OPT_TDI_PLAN_CACHE = 6
LR_OPT_CHUNK_SAMPLES = 7
LR_OPT_FFT_LENGTH = 8
LR_OPT_PROJ_PATH = 9
LR_OPT_Y_PRECISION = 10
LR_Y_PLAIN, LR_Y_EXTENDED = 0, 1
LR_INFO_TDI_PATH, LR_INFO_FIR_TAPS, LR_INFO_FIR_POWERS = 101, 102, 103
LR_PROJ_AUTO, LR_PROJ_SINGLE, LR_PROJ_PAIR = -1, 1, 2
LR_IP_CROSS, LR_IP_DIFF, LR_IP_BLOCKS = 0, 1, 1024
LR_GB_NPAR = 6
LR_GB_PAPER, LR_GB_CONFIG = 0, 1
LR_TDI_AUTO, LR_TDI_PER_SAMPLE, LR_TDI_FIR3, LR_TDI_FIR4 = -1, 0, 3, 4
LR_CHAIN_NESTED, LR_CHAIN_SUM = 0, 1
LR_XYZ, LR_AET, LR_XYZ_AET = 0, 1, 2
LR_MAX_ORDER = 65

# every symbol include/lr.h declares
SYMBOLS = ("lr_create", "lr_destroy", "lr_set_option", "lr_get_option", "lr_get_margins", "lr_project", "lr_tdi",
           "lr_inner_product", "lr_inner_product_static", "lr_gb_parameters", "lr_fft_good_length", "lr_gb_waveform", "lr_response_gb", "lr_loglike_gb", "lr_response", "lr_response_span", "lr_get_span_halo", "lr_response_host", "lr_eval_orbit", "lr_measure_fp64_peak", "lr_launch_count", "lr_plan_create", "lr_plan_attach", "lr_plan_release", "lr_plan_bytes",
           "lr_last_cuda_error", "lr_strerror")


class LrUnavailable(RuntimeError):
    """liblr.so is not built / not loadable.  The library has no CPU path."""


class LrError(RuntimeError):
    def __init__(self, code, where, cuda=0):
        self.code = code
        self.cuda = cuda
        msg = lib().lr_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code}" + (f", cudaError {cuda})" if cuda else ")"))


class lr_orbits(ctypes.Structure):
    _fields_ = [("n_knots", ctypes.c_int64), ("t_start", ctypes.c_double), ("knot_dt", ctypes.c_double),
                ("x", ctypes.c_void_p), ("ltt", ctypes.c_void_p)]


_lib = None


def lib():
    """The loaded liblr (ctypes.CDLL) with argument types set."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LrUnavailable(f"{LIB_PATH} not found: build it with `python -m paper_2204_06633_b200.build` "
                            "(nvcc, sm_100a).  There is no CPU fallback.")
    try:
        L = ctypes.CDLL(LIB_PATH)
    except OSError as e:  # pragma: no cover
        raise LrUnavailable(f"cannot load {LIB_PATH}: {e}") from e
    i64, dbl, vp, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_int
    pi64 = ctypes.POINTER(i64)
    L.lr_create.argtypes = [ctypes.POINTER(lr_orbits), dbl, ci, ci, ctypes.POINTER(vp)]
    L.lr_create.restype = ci
    L.lr_destroy.argtypes = [vp]
    L.lr_destroy.restype = None
    L.lr_set_option.argtypes = [vp, ci, dbl]
    L.lr_get_option.argtypes = [vp, ci, ctypes.POINTER(dbl)]
    L.lr_get_margins.argtypes = [vp, pi64, pi64, pi64]
    L.lr_project.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, vp, vp]
    L.lr_tdi.argtypes = [vp, vp, i64, i64, vp, vp]
    L.lr_response.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i64, vp, vp]
    L.lr_response_span.argtypes = [vp, vp, vp, vp, i64, i64, vp, vp, vp, i64, i64, i64, i64, vp, vp]
    L.lr_get_span_halo.argtypes = [vp, vp, pi64, pi64, pi64]
    L.lr_response_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i64, vp, vp]
    L.lr_inner_product.argtypes = [vp, vp, vp, dbl, ci, i64, i64, ci, i64, vp, vp, vp]
    L.lr_inner_product_static.argtypes = [vp, vp, vp, dbl, ci, i64, i64, ci, i64, vp, vp]
    L.lr_gb_waveform.argtypes = [vp, vp, i64, i64, vp, vp, vp]
    L.lr_gb_parameters.argtypes = [dbl, dbl, dbl, dbl, dbl, ci, vp]
    L.lr_fft_good_length.argtypes = [i64]
    L.lr_fft_good_length.restype = i64
    L.lr_response_gb.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, vp, vp]
    L.lr_loglike_gb.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, vp, vp, dbl, ci, vp, vp]
    L.lr_eval_orbit.argtypes = [vp, ci, vp, i64, vp, vp]
    L.lr_measure_fp64_peak.argtypes = [dbl, ctypes.POINTER(dbl)]
    L.lr_plan_create.argtypes = [vp, i64, vp, ctypes.POINTER(vp)]
    L.lr_plan_attach.argtypes = [vp, vp]
    L.lr_plan_release.argtypes = [vp]
    L.lr_plan_release.restype = None
    L.lr_plan_bytes.argtypes = [vp]
    L.lr_plan_bytes.restype = i64
    L.lr_launch_count.argtypes = []
    L.lr_launch_count.restype = i64
    L.lr_last_cuda_error.argtypes = [vp]
    L.lr_strerror.argtypes = [ci]
    L.lr_strerror.restype = ctypes.c_char_p
    _lib = L
    return L


def _host(a):
    return np.ascontiguousarray(np.atleast_1d(a), dtype=np.float64)


def _check(rc, where, handle=None):
    if rc != LR_OK:
        cuda = lib().lr_last_cuda_error(handle) if handle else 0
        raise LrError(rc, where, cuda)


def _dev_ptr(t, name, numel=None):
    """data_ptr of a contiguous fp64 CUDA tensor."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous float64 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


# ------------------------------------------------------------------------------------------------ C calls
def lr_create(table, dt, lagrange_order, tdi_gen):
    """lr_create: `table` has .n_knots .t_start .knot_dt .x[3,3,K] .ltt[6,K] (host numpy).  Returns a handle."""
    x, ltt = _host(table.x), _host(table.ltt)
    if x.size != 9 * table.n_knots or ltt.size != 6 * table.n_knots:
        raise ValueError("orbit table: x must be [3,3,n_knots] and ltt [6,n_knots]")
    orb = lr_orbits(int(table.n_knots), float(table.t_start), float(table.knot_dt),
                    x.ctypes.data_as(ctypes.c_void_p), ltt.ctypes.data_as(ctypes.c_void_p))
    h = ctypes.c_void_p()
    _check(lib().lr_create(ctypes.byref(orb), float(dt), int(lagrange_order), int(tdi_gen), ctypes.byref(h)),
           "lr_create")
    return h


def lr_destroy(h):
    _N_OUT.pop(h.value if hasattr(h, "value") else int(h), None)
    lib().lr_destroy(h)


def lr_set_option(h, key, value):
    _check(lib().lr_set_option(h, int(key), float(value)), "lr_set_option", h)
    if int(key) == LR_OPT_CHANNELS:
        _N_OUT.pop(h.value if hasattr(h, "value") else int(h), None)


def lr_get_option(h, key):
    v = ctypes.c_double()
    _check(lib().lr_get_option(h, int(key), ctypes.byref(v)), "lr_get_option", h)
    return v.value


_N_OUT = {}   # handle address -> rows per template, kept in step by lr_set_option / lr_destroy (saves a call per launch)


def _n_out(h):
    """Rows per template lr_tdi writes with this handle's LR_OPT_CHANNELS (the C ABI takes no size for `out`)."""
    key = h.value if hasattr(h, "value") else int(h)
    n = _N_OUT.get(key)
    if n is None:
        n = _N_OUT[key] = 6 if int(lr_get_option(h, LR_OPT_CHANNELS)) == LR_XYZ_AET else 3
    return n


def _angles(beta, lam, psi):
    beta, lam, psi = _host(beta), _host(lam), _host(psi)
    if lam.size != beta.size or psi.size != beta.size:
        raise ValueError("beta, lambda, psi must have one entry per template")
    return beta, lam, psi, beta.size


def lr_get_margins(h):
    a, b, c = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
    _check(lib().lr_get_margins(h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "lr_get_margins", h)
    return a.value, b.value, c.value


def lr_project(h, h_plus, h_cross, beta, lam, psi, y_out, stream=None):
    """lr_project: h_plus, h_cross CUDA [B,N]; beta, lam, psi host [B]; y_out CUDA [B,6,N] (written)."""
    beta, lam, psi, B = _angles(beta, lam, psi)
    if h_plus.numel() % B:
        raise ValueError("h_plus size is not a multiple of the batch")
    n = h_plus.numel() // B
    _check(lib().lr_project(h, _dev_ptr(h_plus, "h_plus"), _dev_ptr(h_cross, "h_cross", B * n),
                            beta.ctypes.data, lam.ctypes.data, psi.ctypes.data, B, n,
                            _dev_ptr(y_out, "y_out", B * 6 * n), _stream(stream)), "lr_project", h)
    return y_out


def lr_tdi(h, y, out, batch, stream=None):
    """lr_tdi: y CUDA [B,6,N]; out CUDA [B,3|6,N] (written)."""
    if y.numel() % (6 * batch):
        raise ValueError("y must be [batch,6,n]")
    n = y.numel() // (6 * batch)
    if out.numel() != _n_out(h) * batch * n:
        raise ValueError(f"out must be [batch,{_n_out(h)},n] for this handle's LR_OPT_CHANNELS")
    _check(lib().lr_tdi(h, _dev_ptr(y, "y"), batch, n, _dev_ptr(out, "out"), _stream(stream)), "lr_tdi", h)
    return out


def lr_response(h_proj, h_tdi, h_plus, h_cross, beta, lam, psi, out, stream=None):
    """lr_response: h_plus, h_cross CUDA [B,N] -> out CUDA [B,3|6,N], no y array (chunked through L2)."""
    beta, lam, psi, B = _angles(beta, lam, psi)
    if h_plus.numel() % B:
        raise ValueError("h_plus size is not a multiple of the batch")
    n = h_plus.numel() // B
    if out.numel() != _n_out(h_tdi) * B * n:
        raise ValueError(f"out must be [batch,{_n_out(h_tdi)},n] for h_tdi's LR_OPT_CHANNELS")
    _check(lib().lr_response(h_proj, h_tdi, _dev_ptr(h_plus, "h_plus"), _dev_ptr(h_cross, "h_cross", B * n),
                             beta.ctypes.data, lam.ctypes.data, psi.ctypes.data, B, n, _dev_ptr(out, "out"),
                             _stream(stream)), "lr_response", h_proj)
    return out


def lr_get_span_halo(h_proj, h_tdi):
    """(lo, hi, unit): h samples a span needs before / after itself, and the alignment of a span's start."""
    a, b, c = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
    _check(lib().lr_get_span_halo(h_proj, h_tdi, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)),
           "lr_get_span_halo", h_proj)
    return a.value, b.value, c.value


def lr_response_span(h_proj, h_tdi, h_plus, h_cross, h_first, beta, lam, psi, n, first, count, out, stream=None):
    """lr_response_span: h_plus, h_cross CUDA [B, h_len] = global samples [h_first, h_first+h_len) of a series
    of n samples; out CUDA [B, 3|6, count] receives the global samples [first, first+count)."""
    beta, lam, psi, B = _angles(beta, lam, psi)
    if h_plus.numel() % B:
        raise ValueError("h_plus size is not a multiple of the batch")
    h_len = h_plus.numel() // B
    if out.numel() != _n_out(h_tdi) * B * count:
        raise ValueError(f"out must be [batch,{_n_out(h_tdi)},count] for h_tdi's LR_OPT_CHANNELS")
    _check(lib().lr_response_span(h_proj, h_tdi, _dev_ptr(h_plus, "h_plus"), _dev_ptr(h_cross, "h_cross", B * h_len),
                                  int(h_first), h_len, beta.ctypes.data, lam.ctypes.data, psi.ctypes.data, B, int(n),
                                  int(first), int(count), _dev_ptr(out, "out"), _stream(stream)),
           "lr_response_span", h_proj)
    return out


def lr_response_host(h_proj, h_tdi, h_plus, h_cross, beta, lam, psi, out, stream=None):
    """lr_response_host: host numpy (or pinned CPU tensors viewed as numpy) in, host out; synchronous."""
    beta, lam, psi, B = _angles(beta, lam, psi)
    hp, hc = _as_host_f64(h_plus), _as_host_f64(h_cross)
    o = _as_host_f64(out)
    n = hp.size // B
    if hp.size != B * n or hc.size != B * n or o.size != _n_out(h_tdi) * B * n:
        raise ValueError("lr_response_host: inconsistent sizes (out must hold 3 or 6 rows per template, per "
                         "h_tdi's LR_OPT_CHANNELS)")
    _check(lib().lr_response_host(h_proj, h_tdi, hp.ctypes.data, hc.ctypes.data, beta.ctypes.data,
                                  lam.ctypes.data, psi.ctypes.data, B, n, o.ctypes.data,
                                  _stream(stream) if stream is not None else _stream(None)),
           "lr_response_host", h_proj)
    return out


def _gb(gb):
    g = np.ascontiguousarray(np.asarray(gb, dtype=np.float64))
    if g.ndim == 1:
        g = g[None]
    if g.ndim != 2 or g.shape[1] != LR_GB_NPAR:
        raise ValueError("gb must be [batch, 6] = a_plus, a_cross, f0, fdot, fddot, phi0")
    return g


def lr_fft_good_length(n):
    """Smallest 7-smooth length >= n (a fast transform length for LR_OPT_FFT_LENGTH)."""
    m = lib().lr_fft_good_length(int(n))
    if m < 0:
        raise ValueError("n out of range")
    return int(m)


def lr_gb_parameters(A, f0, fdot, phi0, iota, form=LR_GB_PAPER):
    """lr_gb_parameters: the six numbers of one template (numpy [6])."""
    g = np.empty(LR_GB_NPAR)
    _check(lib().lr_gb_parameters(float(A), float(f0), float(fdot), float(phi0), float(iota), int(form),
                                  g.ctypes.data), "lr_gb_parameters")
    return g


def lr_gb_waveform(h, gb, n, h_plus, h_cross, stream=None):
    """lr_gb_waveform: gb host [B, 6] -> h_plus, h_cross CUDA [B, n] (written)."""
    g = _gb(gb)
    B = g.shape[0]
    _check(lib().lr_gb_waveform(h, g.ctypes.data, B, int(n), _dev_ptr(h_plus, "h_plus", B * n),
                                _dev_ptr(h_cross, "h_cross", B * n), _stream(stream)), "lr_gb_waveform", h)
    return h_plus, h_cross


def lr_response_gb(h_proj, h_tdi, gb, beta, lam, psi, n, out, stream=None):
    """lr_response_gb: waveform parameters host [B, 6] + sky angles -> out CUDA [B, 3|6, n]."""
    g = _gb(gb)
    beta, lam, psi = _host(beta), _host(lam), _host(psi)
    B = g.shape[0]
    if beta.size != B or lam.size != B or psi.size != B:
        raise ValueError("beta, lambda, psi must have one entry per template")
    if out.numel() != _n_out(h_tdi) * B * n:
        raise ValueError(f"out must be [batch,{_n_out(h_tdi)},n] for h_tdi's LR_OPT_CHANNELS")
    _check(lib().lr_response_gb(h_proj, h_tdi, g.ctypes.data, beta.ctypes.data, lam.ctypes.data, psi.ctypes.data,
                                B, int(n), _dev_ptr(out, "out"), _stream(stream)), "lr_response_gb", h_proj)
    return out


def lr_loglike_gb(h_proj, h_tdi, gb, beta, lam, psi, n, data_f, inv_psd, scale, mode=LR_IP_DIFF, out=None,
                  stream=None, n_fft=None):
    """lr_loglike_gb: waveform parameters host [B, 6] + sky angles -> out CUDA float64 [B]; data_f CUDA
    complex128 [3, n//2+1] (unnormalised DFT), inv_psd CUDA float64 [3, n//2+1]."""
    import torch
    g = _gb(gb)
    beta, lam, psi = _host(beta), _host(lam), _host(psi)
    B = g.shape[0]
    nf = (n_fft or n) // 2 + 1   # n_fft: the LR_OPT_FFT_LENGTH the caller set on h_proj (sizes are checked against it)
    if beta.size != B or lam.size != B or psi.size != B:
        raise ValueError("beta, lambda, psi must have one entry per template")
    if not (isinstance(data_f, torch.Tensor) and data_f.is_cuda and data_f.dtype == torch.complex128
            and data_f.is_contiguous() and data_f.numel() == 3 * nf):
        raise TypeError("data_f must be a contiguous CUDA complex128 tensor [3, n//2+1]")
    if out is None:
        out = torch.empty(B, dtype=torch.float64, device=data_f.device)
    _check(lib().lr_loglike_gb(h_proj, h_tdi, g.ctypes.data, beta.ctypes.data, lam.ctypes.data, psi.ctypes.data, B,
                               int(n), data_f.data_ptr(), _dev_ptr(inv_psd, "inv_psd", 3 * nf), float(scale),
                               int(mode), _dev_ptr(out, "out", B), _stream(stream)), "lr_loglike_gb", h_proj)
    return out


def _as_host_f64(a):
    if hasattr(a, "numpy") and not isinstance(a, np.ndarray):
        a = a.numpy()  # CPU (possibly pinned) torch tensor: shares memory
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]):
        raise TypeError("host buffers must be C-contiguous float64")
    return a


def lr_inner_product(fa, fb, inv_psd, scale, mode=LR_IP_CROSS, out=None, stream=None):
    """lr_inner_product: fa CUDA complex128 [B, nch, nf], fb [B or 1, nch, nf], inv_psd CUDA float64 [nch, nf];
    returns out CUDA float64 [B]."""
    import torch
    for name, t in (("fa", fa), ("fb", fb)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()
                and t.dim() == 3):
            raise TypeError(f"{name} must be a contiguous complex128 CUDA tensor [batch, nch, nf]")
    B, nch, nf = fa.shape
    if fb.shape[1:] != fa.shape[1:] or fb.shape[0] not in (1, B):
        raise ValueError("fb must be [batch or 1, nch, nf]")
    if out is None:
        out = torch.empty(B, dtype=torch.float64, device=fa.device)
    work = torch.empty(B * LR_IP_BLOCKS, dtype=torch.float64, device=fa.device)
    _check(lib().lr_inner_product(fa.data_ptr(), fb.data_ptr(), _dev_ptr(inv_psd, "inv_psd", nch * nf), float(scale),
                                  int(mode), B, fb.shape[0], nch, nf, work.data_ptr(), _dev_ptr(out, "out", B),
                                  _stream(stream)), "lr_inner_product")
    return out


def lr_inner_product_static(fa, fb, inv_psd, scale, out, mode=LR_IP_CROSS, stream=None):
    """lr_inner_product_static: as lr_inner_product, with the scratch inside the library (no allocation anywhere:
    `out` CUDA float64 [B] is the caller's).  B <= LR_IP_STATIC_MAX_BATCH, else LrError(LR_ELIMIT)."""
    import torch
    for name, t in (("fa", fa), ("fb", fb)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()
                and t.dim() == 3):
            raise TypeError(f"{name} must be a contiguous complex128 CUDA tensor [batch, nch, nf]")
    B, nch, nf = fa.shape
    if fb.shape[1:] != fa.shape[1:] or fb.shape[0] not in (1, B):
        raise ValueError("fb must be [batch or 1, nch, nf]")
    _check(lib().lr_inner_product_static(fa.data_ptr(), fb.data_ptr(), _dev_ptr(inv_psd, "inv_psd", nch * nf),
                                         float(scale), int(mode), B, fb.shape[0], nch, nf, _dev_ptr(out, "out", B),
                                         _stream(stream)), "lr_inner_product_static")
    return out


def lr_eval_orbit(h, channel, t, out, stream=None):
    _check(lib().lr_eval_orbit(h, int(channel), _dev_ptr(t, "t"), t.numel(), _dev_ptr(out, "out", t.numel()),
                               _stream(stream)), "lr_eval_orbit", h)
    return out


def lr_measure_fp64_peak(seconds=0.5):
    v = ctypes.c_double()
    _check(lib().lr_measure_fp64_peak(float(seconds), ctypes.byref(v)), "lr_measure_fp64_peak")
    return v.value


def lr_plan_create(h, n, stream=None):
    """lr_plan_create: the shareable, read-only TDI plan of handle h for a series of n samples."""
    p = ctypes.c_void_p()
    _check(lib().lr_plan_create(h, int(n), _stream(stream), ctypes.byref(p)), "lr_plan_create", h)
    return p


def lr_plan_attach(h, plan):
    _check(lib().lr_plan_attach(h, plan), "lr_plan_attach", h)


def lr_plan_release(plan):
    lib().lr_plan_release(plan)


def lr_plan_bytes(plan):
    return int(lib().lr_plan_bytes(plan))


def lr_launch_count():
    return int(lib().lr_launch_count())


def lr_strerror(code):
    return lib().lr_strerror(int(code)).decode()
