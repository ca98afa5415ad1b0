"""-m gpu: fdas_spectrum_exec (real series -> whitened spectrum, reading 18) against oracle.spectrum,
and the whole chain series -> spectrum -> power plane against the oracle's chain."""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import check

pytestmark = pytest.mark.gpu


def _series(n_t, seed, tone=None, red=0.0):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal(n_t)
    if red:
        x += red * np.cumsum(rng.standard_normal(n_t)) / np.sqrt(n_t)
    if tone:
        r, amp = tone
        x += amp * np.cos(2 * np.pi * r * np.arange(n_t) / n_t + 0.3)
    return x.astype(np.float32)


def _gpu_spectrum(x, blk):
    import torch
    from paper_1711_10855_b200 import binding
    plan = binding.SpectrumPlan(x.size, blk)
    assert plan.bins == x.size // 2
    d_x = torch.from_numpy(x).cuda()
    d_a = torch.full((x.size // 2,), float("nan"), dtype=torch.complex64, device="cuda")
    plan.exec(d_x, d_a)
    plan.exec(d_x, d_a)          # twice: the scratch buffers are reused
    torch.cuda.synchronize()
    plan.destroy()
    return d_a.cpu().numpy()


@pytest.mark.parametrize("log2n,blk", [(19, 0), (19, 1000), (20, 4096), (21, 777), (23, 4096)])
def test_spectrum_vs_oracle(oracle, log2n, blk):
    """float32 four-step transform against eq.(3) in double.  The rounding error of a float32 transform does not scale
    with the bin it lands in but with the largest values that pass through the butterflies: about eps log2(n) rms|X|
    typically, and up to a few eps max|X| in bins that share a butterfly (or the real/complex separation, bin k with
    bin N-k) with the strongest bins.  The series here is red, as real observations are (max|X| ~ 1000 rms|X|), so
    both terms matter; whitening multiplies bin and error alike by the block's scale s_b (1 when not whitened):
        |dA_k| <= s_b (1e-5 rms|X| + 4 * 2^-24 max|X|) + 1e-6 |A_k|
    Measured: 0.08 - 0.18 of that bound.  2^23 samples is the series behind BASELINE.json config 3 (2^22 bins)."""
    n_t = 1 << log2n
    x = _series(n_t, 100 + log2n, tone=(n_t // 7 + 3, 0.05), red=3.0)
    a = _gpu_spectrum(x, blk)
    assert np.all(np.isfinite(a.view(np.float32)))
    X = oracle.spectrum(x.astype(np.float64), 0)
    ref = oracle.spectrum(x.astype(np.float64), blk) if blk else X
    rms = np.sqrt(np.mean(np.abs(X) ** 2))
    scale = np.ones(X.size)
    if blk:
        nz = np.abs(X) > 0
        scale[nz] = np.abs(ref[nz]) / np.abs(X[nz])
        scale[0] = scale[1]                                   # bin 0 is forced to 0; it shares block 0's scale
    err = np.abs(a.astype(np.complex128) - ref)
    bound = scale * (1e-5 * rms + 4 * 2.0 ** -24 * np.abs(X).max()) + 1e-6 * np.abs(ref)
    worst = float((err / bound).max())
    assert worst <= 1.0, (log2n, blk, worst)
    if blk:
        assert a[0] == 0
        p = np.abs(a.astype(np.complex128)) ** 2
        n_full = (p.size // blk) * blk
        assert np.abs(p[:n_full].reshape(-1, blk).mean(axis=1) - 2.0).max() < 1e-4   # every block: mean power 2
    print(f"n_t=2^{log2n} blk={blk}: worst error / bound {worst:.3f}")


def test_series_to_power_plane_chain(oracle):
    """series -> fdas_spectrum_exec -> fdas_convolve on the GPU against oracle.spectrum -> oracle.direct: a weak
    accelerated-free tone (z = 0) ends up as the global maximum of the z = 0 row at its bin."""
    import torch
    from paper_1711_10855_b200 import binding
    n_t = 1 << 19
    r = 70001
    x = _series(n_t, 7, tone=(r, 0.06))
    H = workload.templates(32, 2, 128).astype(np.complex64)
    sp = binding.SpectrumPlan(n_t, 2048)
    n_f = sp.bins
    plan = binding.Plan(n_f, 32, 2, 128, 512)
    plan.set_templates(H)
    d_a = torch.empty((1, n_f), dtype=torch.complex64, device="cuda")
    d_p = torch.full((1, H.shape[0], n_f), float("nan"), dtype=torch.float32, device="cuda")
    sp.exec(torch.from_numpy(x).cuda(), d_a)
    plan.convolve(d_a, d_p)
    torch.cuda.synchronize()
    p = d_p.cpu().numpy()[0]
    a_ref = oracle.spectrum(x.astype(np.float64), 2048).astype(np.complex64)     # the oracle's own input, rounded once
    p_ref = oracle.direct(a_ref, H.astype(np.complex128))
    check(p, p_ref, what="chain")
    iz, ic = np.unravel_index(np.argmax(p), p.shape)
    assert iz == H.shape[0] // 2 and ic == r
    sp.destroy(); plan.destroy()


def test_spectrum_arguments():
    from paper_1711_10855_b200 import binding
    with pytest.raises(binding.FdasError) as ei:
        binding.SpectrumPlan(1 << 18)
    assert ei.value.status == binding.FDAS_ERR_UNSUPPORTED
    with pytest.raises(binding.FdasError) as ei:
        binding.SpectrumPlan((1 << 20) + 2)
    assert ei.value.status == binding.FDAS_ERR_INVALID_ARG


def test_spectrum_is_deterministic():
    import torch
    from paper_1711_10855_b200 import binding
    n_t = 1 << 21
    x = torch.from_numpy(_series(n_t, 3, red=1.0)).cuda()
    plan = binding.SpectrumPlan(n_t, 1500)
    outs = [torch.empty(n_t // 2, dtype=torch.complex64, device="cuda") for _ in range(3)]
    for o in outs:
        plan.exec(x, o)
    torch.cuda.synchronize()
    assert torch.equal(outs[0].view(torch.float32), outs[1].view(torch.float32))
    assert torch.equal(outs[0].view(torch.float32), outs[2].view(torch.float32))
    plan.destroy()
