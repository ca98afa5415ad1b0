"""-m gpu: the segment FFT device code (eq.(3)) against the oracle's transforms."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("L", [512, 1024, 2048, 4096, 8192])
@pytest.mark.parametrize("inverse", [False, True])
def test_segment_fft_vs_oracle(oracle, L, inverse):
    import torch
    from paper_1711_10855_b200 import binding
    rng = np.random.default_rng(L + int(inverse))
    n_seg = 5
    x = (rng.standard_normal((n_seg, L)) + 1j * rng.standard_normal((n_seg, L))).astype(np.complex64)
    x[1] = 0; x[1, 1] = 1.0          # a pure tone: X_m = w_L^m (pins index order and sign)
    d_in = torch.from_numpy(x).cuda()
    d_out = torch.empty_like(d_in)
    binding.debug_fft(L, n_seg, d_in, d_out, inverse=inverse)
    y = d_out.cpu().numpy()
    sign = +1 if inverse else -1
    for s in range(n_seg):
        ref = oracle.fft(x[s].astype(np.complex128), sign=sign)
        scale = np.sqrt(L) * np.abs(x[s]).max()
        assert np.max(np.abs(y[s] - ref)) <= 2e-6 * scale * np.log2(L), (L, inverse, s)
    # the tone row against the closed form of eq.(3)
    k = np.arange(L)
    tone = np.exp(sign * 2j * np.pi * k / L)
    assert np.max(np.abs(y[1] - tone)) < 1e-5
