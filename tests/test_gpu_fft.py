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


@pytest.mark.parametrize("n,e", [(512, 8), (1024, 8), (1024, 16), (2048, 16), (4096, 16), (8192, 16)])
@pytest.mark.parametrize("inverse", [False, True])
def test_batched_fft_vs_oracle(oracle, n, e, inverse):
    """fdas_fft_exec (the stand-alone FFT of P:46 / Table 1; elements per thread is its design axis) on a batch
    that is not a multiple of anything, natural order in and out, both directions."""
    import torch
    from paper_1711_10855_b200 import binding
    rng = np.random.default_rng(n + e + int(inverse))
    n_fft = 301
    x = (rng.standard_normal((n_fft, n)) + 1j * rng.standard_normal((n_fft, n))).astype(np.complex64)
    x[1] = 0; x[1, 1] = 1.0
    x[2] = 0; x[2, n - 1] = 1.0j
    plan = binding.FftPlan(n, e)
    assert plan.elems_per_thread == e and plan.grid >= 148
    d_in = torch.from_numpy(x).cuda()
    d_out = torch.full_like(d_in, float("nan"))
    plan.exec(n_fft, d_in, d_out, inverse=inverse)
    torch.cuda.synchronize()
    y = d_out.cpu().numpy()
    assert np.all(np.isfinite(y.view(np.float32)))
    sign = +1 if inverse else -1
    for s in (0, 1, 2, 147, 148, 300):
        ref = oracle.fft(x[s].astype(np.complex128), sign=sign)
        scale = np.sqrt(n) * np.abs(x[s]).max()
        assert np.max(np.abs(y[s] - ref)) <= 2e-6 * scale * np.log2(n), (n, e, inverse, s)
    # Parseval on every sequence (eq.(3) is unnormalised: sum |X|^2 = n sum |x|^2)
    ex = (np.abs(x.astype(np.complex128)) ** 2).sum(axis=1)
    ey = (np.abs(y.astype(np.complex128)) ** 2).sum(axis=1)
    assert np.max(np.abs(ey / (n * ex) - 1.0)) < 1e-5
    # inverse(forward(x)) = n x
    d_back = torch.empty_like(d_in)
    plan.exec(n_fft, d_out, d_back, inverse=not inverse)
    torch.cuda.synchronize()
    assert np.max(np.abs(d_back.cpu().numpy() / n - x)) < 2e-5
    plan.destroy()


def test_batched_fft_arguments():
    import torch
    from paper_1711_10855_b200 import binding
    with pytest.raises(binding.FdasError) as ei:
        binding.FftPlan(1000, 0)
    assert ei.value.status == binding.FDAS_ERR_UNSUPPORTED
    with pytest.raises(binding.FdasError) as ei:
        binding.FftPlan(4096, 8)
    assert ei.value.status == binding.FDAS_ERR_UNSUPPORTED
    plan = binding.FftPlan(1024)
    assert plan.elems_per_thread == 16
    buf = torch.zeros((4, 1024), dtype=torch.complex64, device="cuda")
    with pytest.raises(binding.FdasError):
        plan.exec(4, buf, buf)              # in place is not supported
    plan.exec(0, buf, torch.empty_like(buf))  # empty batch: nothing to do
    plan.destroy()


@pytest.mark.parametrize("n_launches,per", [(7, 13), (40, 5)])
def test_exec_many_walks_the_buffers(n_launches, per):
    """fdas_fft_exec_many ("100 FFTs per kernel launch, while launching 1000 of these kernels"): launch i
    transforms sequences [i*n_fft, (i+1)*n_fft), so the protocol equals one launch over all of them, bit for bit --
    as a loop of launches (7 launches) and as the recorded CUDA graph (40 launches: first call builds it, the second
    re-uses it, other arguments rebuild it)."""
    import torch
    from paper_1711_10855_b200 import binding
    n = 1024
    g = torch.Generator(device="cuda").manual_seed(46)
    x = torch.randn((n_launches * per, n, 2), device="cuda", generator=g)
    plan = binding.FftPlan(n)
    y_one = torch.full_like(x, float("nan"))
    plan.exec(n_launches * per, x, y_one)
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    for rep in range(3):
        y_many = torch.full_like(x, float("nan"))
        if rep < 2:
            y_keep = y_many if rep == 0 else y_keep
            target = y_keep                      # same arguments twice: the second call launches the cached graph
            target.fill_(float("nan"))
        else:
            target = y_many                      # another output buffer: the graph is rebuilt
        torch.cuda.synchronize()
        plan.exec_many(n_launches, per, x, target, stream=stream)
        torch.cuda.synchronize()
        assert torch.isfinite(target).all()
        assert torch.equal(y_one, target), rep
    # the inverse through the same entry, and back
    y_inv = torch.empty_like(x)
    plan.exec_many(n_launches, per, y_one, y_inv, inverse=True, stream=stream)
    torch.cuda.synchronize()
    assert (y_inv / n - x).abs().max().item() < 2e-5
    plan.destroy()
