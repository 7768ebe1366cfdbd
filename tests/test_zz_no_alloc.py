"""lr_inner_product_static: the no-allocation variant of lr_inner_product (scratch in a file-scope device array of the
library) against the existing path.  Collected last (the file name sorts after every other test file) so that a
failure here hides no other test under `pytest -x`; passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lr():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    import paper_2204_06633_b200 as pkg
    from paper_2204_06633_b200 import build
    build.ensure_built()
    pkg.binding.lib()
    return pkg


def _spectra(batch, nch, nf, seed):
    """Seeded synthetic spectra [batch, nch, nf] (complex128), a data set [1, nch, nf] and 1/S_n [nch, nf] with a
    steep colour (10 decades across the band, like an instrument PSD), on the device."""
    import torch
    rng = np.random.default_rng(seed)
    f = np.arange(nf) / nf
    col = 1.0 / (1e-3 + f) ** 2
    fa = (rng.normal(size=(batch, nch, nf)) + 1j * rng.normal(size=(batch, nch, nf))) * col
    fd = (rng.normal(size=(1, nch, nf)) + 1j * rng.normal(size=(1, nch, nf))) * col
    inv = 1.0 / (1e-6 + f ** 4)[None, :] * np.linspace(1.0, 2.0, nch)[:, None]
    inv[:, 0] = 0.0
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return dev(fa), dev(fd), dev(inv)


def test_inner_product_static_matches_the_allocating_path_on_two_calls_in_a_row(lr):
    import torch
    B = lr.binding
    # call 1 fills the whole scratch (64 templates); call 2 is smaller and of another shape, so the array still holds
    # call 1's partial sums when it starts; call 3 repeats call 1 (same bits again)
    cases = [(64, 3, 40001, lr.LR_IP_DIFF, 1), (5, 2, 1237, lr.LR_IP_CROSS, 2), (64, 3, 40001, lr.LR_IP_DIFF, 1)]
    outs = []
    torch.cuda.synchronize()
    free0 = None
    for i, (batch, nch, nf, mode, seed) in enumerate(cases):
        fa, fd, inv = _spectra(batch, nch, nf, seed)
        fb = fd if mode == lr.LR_IP_DIFF else fa                      # one data set against all / pairwise
        want = lr.lr_inner_product(fa, fb, inv, 0.37, mode=mode)      # the existing path (caller-allocated work)
        out = torch.full((batch,), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        l0 = lr.lr_launch_count()
        B.lr_inner_product_static(fa, fb, inv, 0.37, out, mode=mode)
        B.lr_inner_product_static(fa, fb, inv, 0.37, out, mode=mode)  # twice in a row on the same stream
        torch.cuda.synchronize()
        assert lr.lr_launch_count() - l0 == 4                         # two kernels per call, nothing else
        assert torch.cuda.mem_get_info()[0] == free0                  # no device memory was taken
        w, g = want.cpu().numpy(), out.cpu().numpy()
        assert np.all(np.isfinite(g)) and np.all(g != 0)
        assert np.abs(g - w).max() <= 1e-13 * np.abs(w).max()         # the bar of test_gpu_inner_product_parity
        assert np.array_equal(g, w)                                   # same kernels, same tree: the same bits
        outs.append(g)
    assert np.array_equal(outs[0], outs[2])


def test_inner_product_static_rejects_what_does_not_fit(lr):
    import torch
    B = lr.binding
    assert B.LR_IP_STATIC_MAX_BATCH == 64
    fa, fd, inv = _spectra(65, 1, 300, 3)
    out = torch.zeros(65, dtype=torch.float64, device="cuda")
    l0 = lr.lr_launch_count()
    with pytest.raises(lr.LrError) as e:
        B.lr_inner_product_static(fa, fd, inv, 1.0, out, mode=lr.LR_IP_DIFF)
    assert e.value.code == B.LR_ELIMIT and "capacity" in str(e.value)
    assert lr.lr_launch_count() == l0 and not out.any()               # nothing ran
    with pytest.raises(lr.LrError) as e:
        B.lr_inner_product_static(fa[:2], fd, inv, 1.0, out[:2].contiguous(), mode=7)
    assert e.value.code == lr.LR_EINVAL
    # the limit itself is fine
    got = B.lr_inner_product_static(fa[:64].contiguous(), fd, inv, 1.0, out[:64].contiguous(), mode=lr.LR_IP_DIFF)
    want = lr.lr_inner_product(fa[:64].contiguous(), fd, inv, 1.0, mode=lr.LR_IP_DIFF)
    assert torch.equal(got, want)
