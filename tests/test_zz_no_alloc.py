"""ptycho_fft2_noalloc (include/ptycho_b200.h): the entry point that allocates nothing, against the existing path
(ptycho_test_fft2, which cudaMallocs its twiddle scratch and fills it from the host).  Collected last on purpose."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_FFT = 2e-6          # the FFT tolerance of tests/test_gpu_parity.py::test_fft2_vs_oracle


def rel(a, b):
    a, b = np.asarray(a, np.complex128).ravel(), np.asarray(b, np.complex128).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2202_03144_b200 import binding
    binding.lib()
    return binding


def test_noalloc_fft2_matches_the_existing_path_on_two_calls_in_a_row(B):
    """Two calls in a row with DIFFERENT sizes, so that the second one finds the first one's tables in the shared scratch; then
    the first size again, and the inverse.  Every result is compared with the existing path's on the same input."""
    import torch
    rng = np.random.default_rng(2024)
    for n, count, inverse in [(256, 7, False), (64, 37, False), (256, 7, True), (512, 3, False), (128, 5, True), (64, 37, True)]:
        x = (rng.standard_normal((count, n, n)) + 1j * rng.standard_normal((count, n, n))).astype(np.complex64)
        d = torch.from_numpy(x).cuda()
        want = B.test_fft2(d.clone(), inverse=inverse).cpu().numpy()        # existing path (synchronises)
        got = B.fft2_noalloc(d.clone(), inverse=inverse)                    # asynchronous on the current stream
        again = B.fft2_noalloc(d.clone(), inverse=inverse)                  # the same call once more, back to back
        torch.cuda.synchronize()
        got, again = got.cpu().numpy(), again.cpu().numpy()
        assert np.isfinite(got).all()
        assert rel(got, want) < TOL_FFT, (n, inverse, rel(got, want))
        assert np.array_equal(got, again), (n, inverse)
        ref = np.fft.ifft2(x.astype(np.complex128)) if inverse else np.fft.fft2(x.astype(np.complex128))
        assert rel(got, ref) < TOL_FFT, (n, inverse)


def test_noalloc_fft2_back_to_back_without_a_sync_between_sizes(B):
    """Stream order is what protects the shared scratch: two calls of different sizes queued with no synchronisation in between."""
    import torch
    rng = np.random.default_rng(7)
    xa = (rng.standard_normal((9, 128, 128)) + 1j * rng.standard_normal((9, 128, 128))).astype(np.complex64)
    xb = (rng.standard_normal((4, 512, 512)) + 1j * rng.standard_normal((4, 512, 512))).astype(np.complex64)
    da, db = torch.from_numpy(xa).cuda(), torch.from_numpy(xb).cuda()
    wa, wb = B.test_fft2(da.clone()).cpu().numpy(), B.test_fft2(db.clone()).cpu().numpy()
    torch.cuda.synchronize()
    B.fft2_noalloc(da)
    B.fft2_noalloc(db)
    torch.cuda.synchronize()
    assert rel(da.cpu().numpy(), wa) < TOL_FFT and rel(db.cpu().numpy(), wb) < TOL_FFT


def test_noalloc_fft2_rejects_what_does_not_fit(B):
    import torch
    d = torch.zeros((1, 1024, 1024), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.PtychoError) as e:
        B.fft2_noalloc(d)
    assert "ENOMEM" in str(e.value) and "exceeds the static scratch" in str(e.value) and "512" in str(e.value)
    assert float(d.abs().max()) == 0.0                                       # nothing ran
    d = torch.zeros((2, 96, 96), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.PtychoError) as e:
        B.fft2_noalloc(d)
    assert "EINVAL" in str(e.value)
