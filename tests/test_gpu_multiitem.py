"""-m gpu: parity at sizes where a CTA of the persistent kernel takes MORE THAN ONE work item, for every kernel variant.

The hot kernel prefetches the next work item's segment from inside the z loop, and only when the launch has more items
than CTAs (grids: 1184 / 1184 / 592 / 296 / 148 CTAs for L = 512 ... 8192).  The BASELINE.json configs exercise that on
the power output with m = L/8 only.  Here the other variants run at such sizes, each against oracle.direct (eq.(2),
P:23) on sampled column blocks, all rows, at the tolerance of tests/parity.py:

  fdas_convolve_complex       N_f = 2^21, L = 2048, m = 256 and 384 -- the shapes `bench.py --mode general` times
  fdas_plan_set_symmetry(1)   C3 and C2 with a bit-exactly symmetrised bank -- the shapes profiles/r2_symmetry.md times
  trim mode 1 (m a small multiple of the thread count, m != L/8)      N_f = 2^21, L = 2048, m = 128
  trim mode 2 (anything else)                                         m = 384 at L = 2048; m = 510 at L = 4096, which
                                                                      also makes every segment take the guarded (non-bulk) load
  the chain series(2^23) -> fdas_spectrum_exec -> fdas_convolve on the C3 plan, against oracle.spectrum -> oracle.direct
"""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import ABS_TOL, check, sample_blocks

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as _t
    if not _t.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    return _t


@pytest.fixture(scope="module")
def binding():
    from paper_1711_10855_b200 import binding as _b
    _b.lib()
    return _b


def _blocks(n_f, S, rng, n_random=6, width=1024):
    class _W:  # sample_blocks only needs n_f
        pass
    w = _W()
    w.n_f = n_f
    return sample_blocks(w, S, n_random, width, rng)


def _check_power_blocks(d_pow_item, spec, H, S, rng, oracle, what):
    """d_pow_item: DEVICE float32 [n_z][n_f] of one spectrum; only the sampled blocks cross PCIe."""
    blocks = _blocks(spec.size, S, rng)
    refs = [oracle.direct(spec, H.astype(np.complex128), cols=blk) for blk in blocks]
    pm = max(float(r.max()) for r in refs)
    worst = 0.0
    for blk, ref in zip(blocks, refs):
        got = d_pow_item[:, blk[0]:blk[1]].cpu().numpy()
        a, _ = check(got, ref, p_max=pm, what=f"{what} cols {blk}")
        worst = max(worst, a)
    return worst


@pytest.mark.parametrize("m", [256, 384])
def test_complex_output_multi_item(torch, binding, oracle, m):
    n_f, z_max, z_step, L = 1 << 21, 84, 2, 2048
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, 6100 + m, 1)
    plan = binding.Plan(n_f, z_max, z_step, m, L)
    plan.set_templates(H)
    assert plan.n_seg > plan.grid, "more work items than CTAs"
    d_amp = torch.full((1, H.shape[0], n_f), float("nan"), dtype=torch.complex64, device="cuda")
    plan.convolve_complex(torch.from_numpy(spec).cuda(), d_amp)
    torch.cuda.synchronize()
    assert torch.isfinite(torch.view_as_real(d_amp)).all()
    rng = np.random.default_rng(m)
    blocks = _blocks(n_f, plan.step, rng)
    refs = [oracle.direct(spec[0], H.astype(np.complex128), cols=blk, want="amp") for blk in blocks]
    amax = max(float(np.abs(r).max()) for r in refs)
    worst = 0.0
    for blk, ref in zip(blocks, refs):
        got = d_amp[0][:, blk[0]:blk[1]].cpu().numpy().astype(np.complex128)
        err = float(np.abs(got - ref).max()) / amax
        assert err <= 0.5 * ABS_TOL, (m, blk, err)   # the amplitude form of 1e-4 max(P), as in test_gpu_outputs.py
        worst = max(worst, err)
    print(f"complex output m={m}: {plan.n_seg} items on {plan.grid} CTAs, max|dA|/max|A| = {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("cfg", [3, 2])
def test_symmetric_path_full_size(torch, binding, oracle, cfg):
    wl = workload.make_config(cfg)
    H = wl.templates.astype(np.complex64).copy()
    n_z = H.shape[0]
    for i in range(n_z // 2):               # row of -z := conj(row of +z), z = 0 real: symmetric bit for bit
        H[n_z - 1 - i] = np.conj(H[i])
    H[n_z // 2] = H[n_z // 2].real
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_symmetry(True)
    plan.set_templates(H)
    assert plan.symmetry_active
    assert cfg == 2 or plan.n_seg > plan.grid
    d_pow = torch.full((1, n_z, wl.n_f), float("nan"), dtype=torch.float32, device="cuda")
    plan.convolve(torch.from_numpy(wl.spectrum).cuda(), d_pow)
    torch.cuda.synchronize()
    assert torch.isfinite(d_pow).all()
    worst = _check_power_blocks(d_pow[0], wl.spectrum[0], H, plan.step, np.random.default_rng(cfg), oracle, f"sym C{cfg}")
    print(f"symmetric path C{cfg}: {plan.n_seg} items, max|dP|/max(P) = {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("n_f,z_max,z_step,m,L,aligned", [
    (1 << 21, 20, 2, 128, 2048, True),      # trim mode 1: m = NT/2 ... a small multiple of the thread count, not L/8
    (1 << 21, 20, 2, 384, 2048, True),      # trim mode 2
    (1 << 21, 10, 2, 510, 4096, True),      # trim mode 2 and m/2 odd: segment bases are not 16-byte aligned -> guarded loads
    (1 << 21, 10, 2, 512, 4096, False),     # spectrum only 8-byte aligned: guarded loads on the m = L/8 fast trim
    ((1 << 20) + 5, 20, 2, 96, 512, True),  # 64-thread plan, m not a multiple of 64
])
def test_power_trim_modes_multi_item(torch, binding, oracle, n_f, z_max, z_step, m, L, aligned):
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, 6200 + m + L, 1)
    plan = binding.Plan(n_f, z_max, z_step, m, L)
    plan.set_templates(H)
    assert plan.n_seg > plan.grid, "more work items than CTAs"
    if aligned:
        d_spec = torch.from_numpy(spec).cuda()
    else:
        buf = torch.empty(n_f + 1, dtype=torch.complex64, device="cuda")
        d_spec = buf[1:]
        d_spec.copy_(torch.from_numpy(spec[0]))
        assert d_spec.data_ptr() % 16 == 8
    d_pow = torch.full((1, H.shape[0], n_f), float("nan"), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    assert torch.isfinite(d_pow).all()
    worst = _check_power_blocks(d_pow[0], spec[0], H, plan.step, np.random.default_rng(m + L), oracle, f"m={m} L={L}")
    print(f"power m={m} L={L} aligned={aligned}: {plan.n_seg} items on {plan.grid} CTAs, max|dP|/max(P) = {worst:.2e}")
    plan.destroy()


def test_series_to_c3_plane_chain(torch, binding, oracle):
    """The 2^23-sample series behind BASELINE.json config 3 ("the FFT output of the observation"): GPU spectrum step
    -> fdas_convolve with C3's plan, against the oracle's chain (oracle.spectrum rounded once to complex64, as the GPU
    hands its spectrum on in complex64, then eq.(2) by direct summation) at north_star's tolerance."""
    wl3 = workload.make_config(3, with_spectrum=False)
    n_t = 1 << 23
    rng = np.random.default_rng(2323)
    x = rng.standard_normal(n_t)
    r_tone = 1234567
    x += 0.01 * np.cos(2 * np.pi * r_tone * np.arange(n_t) / n_t + 0.7)
    x = x.astype(np.float32)
    z_max, z_step, m, L = wl3.z_max, wl3.z_step, wl3.m, wl3.seg_len
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    sp = binding.SpectrumPlan(n_t, 4096)
    n_f = sp.bins
    assert n_f == wl3.n_f
    plan = binding.Plan(n_f, z_max, z_step, m, L)
    plan.set_templates(H)
    d_a = torch.empty((1, n_f), dtype=torch.complex64, device="cuda")
    d_p = torch.full((1, H.shape[0], n_f), float("nan"), dtype=torch.float32, device="cuda")
    sp.exec(torch.from_numpy(x).cuda(), d_a)
    plan.convolve(d_a, d_p)
    torch.cuda.synchronize()
    a_ref = oracle.spectrum(x.astype(np.float64), 4096).astype(np.complex64)
    class _W:
        pass
    w = _W(); w.n_f = n_f
    blocks = sample_blocks(w, plan.step, 5, 1024, rng, extra_cols=[r_tone])
    refs = [oracle.direct(a_ref, H.astype(np.complex128), cols=blk) for blk in blocks]
    pm = max(float(r.max()) for r in refs)
    worst = 0.0
    for blk, ref in zip(blocks, refs):
        a, _ = check(d_p[0][:, blk[0]:blk[1]].cpu().numpy(), ref, p_max=pm, what=f"chain cols {blk}")
        worst = max(worst, a)
    # the tone (z = 0) is the plane's maximum, in the middle row at its bin
    flat = int(torch.argmax(d_p[0]).item())
    assert flat // n_f == H.shape[0] // 2 and flat % n_f == r_tone
    print(f"series(2^23) -> spectrum -> C3 plane: max|dP|/max(P) = {worst:.2e}")
    sp.destroy(); plan.destroy()
