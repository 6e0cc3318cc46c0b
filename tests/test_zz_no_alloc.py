"""dse_gauss_legendre_noalloc (include/dse.h): the entry point for callers that cannot allocate device memory.  Its scratch
is a static device array of the library; everything else is the existing path (dse_gauss_legendre), so the results must be
the same.  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_noalloc_gauss_legendre_matches_existing_path_twice():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_1779_b200.binding import gauss_legendre, gauss_legendre_noalloc, GL_NOALLOC_MAX_N, DseError
    # two calls in a row on one stream; the second one is SMALLER, so the shared scratch still holds the first call's
    # entries beyond what the second call rewrites -- they must not matter
    for n in (4099, 257):
        x_ref, w_ref = gauss_legendre(n)                       # existing path: caller-provided scratch
        x = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        w = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        free_before = torch.cuda.mem_get_info()[0]
        gauss_legendre_noalloc(n, x, w)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before      # the call took no device memory
        xr, wr = x_ref.cpu().numpy(), w_ref.cpu().numpy()
        xn, wn = x.cpu().numpy(), w.cpu().numpy()
        # the tolerance of the device Gauss-Legendre tests (tests/test_gpu_schwinger.py); the kernels are the same ones
        assert np.allclose(xn, xr, rtol=0, atol=2e-15) and np.allclose(wn, wr, rtol=2e-11, atol=0)
        assert abs(wn.sum() - 2.0) < 1e-13
    # beyond the static scratch: refused with a clear error, nothing launched
    big = GL_NOALLOC_MAX_N + 1
    x = torch.empty(big, dtype=torch.float64, device="cuda"); w = torch.empty(big, dtype=torch.float64, device="cuda")
    with pytest.raises(DseError) as ei:
        gauss_legendre_noalloc(big, x, w)
    assert ei.value.code == -1 and "static scratch" in str(ei.value)
    # the largest size that fits runs (the paper's 2^17-node rule, fn.13)
    x = torch.empty(GL_NOALLOC_MAX_N, dtype=torch.float64, device="cuda"); w = torch.empty_like(x)
    gauss_legendre_noalloc(GL_NOALLOC_MAX_N, x, w)
    torch.cuda.synchronize()
    assert abs(float(w.sum()) - 2.0) < 1e-12 and bool(torch.all(x[1:] > x[:-1]))
