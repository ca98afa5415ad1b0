"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element, on the seeded
BASELINE.json configs and on edge cases.  Tolerances: tests/parity.py (BASELINE.json north_star)."""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import check, gpu_power, sample_blocks

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
    _b.lib()  # raises if libfdas.so is missing: no fallback
    return _b


def _sampled_parity(wl, p_gpu, oracle, rng, n_random=6, width=1024, b=0, what=""):
    S = wl.seg_len - wl.m
    sig_cols = [s.r_c for s in wl.signals[b]] if wl.signals else []
    blocks = sample_blocks(wl, S, n_random, width, rng, extra_cols=sig_cols)
    H = wl.templates.astype(np.complex128)
    refs = [oracle.direct(wl.spectrum[b], H, cols=blk) for blk in blocks]
    pm = max(float(r.max()) for r in refs)
    worst = (0.0, 0.0)
    for blk, ref in zip(blocks, refs):
        a, r = check(p_gpu[b][:, blk[0]:blk[1]], ref, p_max=pm, what=f"{what} cols {blk}")
        worst = (max(worst[0], a), max(worst[1], r))
    return worst


def test_c1_full_plane(torch, binding, oracle):
    wl = workload.make_config(1)
    p = gpu_power(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    a, r = check(p[0], ref, what="C1")
    # the injected signal peaks in its own row (BASELINE.json north_star), on the GPU plane too
    iz, ic = np.unravel_index(np.argmax(p[0]), p[0].shape)
    assert wl.z_values[iz] == 20 and ic == 20000
    print(f"C1 abs {a:.2e} rel {r:.2e}")


def test_c2_full_plane(torch, binding, oracle):
    wl = workload.make_config(2)
    p = gpu_power(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    a, r = check(p[0], ref, what="C2")
    print(f"C2 abs {a:.2e} rel {r:.2e}")


def test_c3_sampled(torch, binding, oracle):
    """Full size, the launch configuration bench.py times; oracle on sampled column blocks (all rows)."""
    wl = workload.make_config(3)
    p = gpu_power(wl, torch, binding)
    rng = np.random.default_rng(3)
    a, r = _sampled_parity(wl, p, oracle, rng, n_random=8, width=1024, what="C3")
    # properties that hold at any size: mean noise power 2 (unit templates), all finite, >= 0
    assert np.all(p >= 0)
    assert 1.9 < float(p[0][:, ::97].mean()) < 2.1
    print(f"C3 abs {a:.2e} rel {r:.2e}")


@pytest.mark.parametrize("pair", range(len(workload.C4_PAIRS)))
def test_c4_sweep_sampled(torch, binding, oracle, pair):
    wl = workload.make_config(4, pair=pair)
    p = gpu_power(wl, torch, binding)
    rng = np.random.default_rng(40 + pair)
    a, r = _sampled_parity(wl, p, oracle, rng, n_random=4, width=1024, what=wl.name)
    print(f"{wl.name} abs {a:.2e} rel {r:.2e}")


def test_c5_batched_sampled(torch, binding, oracle):
    wl = workload.make_config(5)
    p = gpu_power(wl, torch, binding)
    assert p.shape == (64, 85, 1 << 20)
    rng = np.random.default_rng(5)
    worst = (0.0, 0.0)
    for b in range(64):
        a, r = _sampled_parity(wl, p, oracle, rng, n_random=1, width=512, b=b, what=f"C5[{b}]")
        worst = (max(worst[0], a), max(worst[1], r))
    # one batched call == separate calls, bit for bit (no atomics, same kernel)
    for b in (0, 17, 63):
        single = gpu_power(wl, torch, binding, spectrum=wl.spectrum[b:b + 1])
        assert np.array_equal(single[0], p[b])
    print(f"C5 abs {worst[0]:.2e} rel {worst[1]:.2e}")


# ------------------------------------------------------------------------------------------------
# edge cases: ragged tails, tiny inputs, template widths that do not divide the thread count,
# a single template, every supported segment length
# ------------------------------------------------------------------------------------------------
def _custom(n_f, z_max, z_step, m, L, seed, n_batch=1):
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, seed, n_batch)
    return workload.Workload(f"custom[{n_f},{m},{L}]", n_f, z_max, z_step, m, L, n_batch, spec, H, [])


@pytest.mark.parametrize("n_f,z_max,z_step,m,L", [
    (1, 4, 2, 64, 512),            # a single bin
    (63, 4, 2, 64, 512),           # shorter than the template
    (447, 8, 4, 64, 512),          # one sample short of S
    (448, 8, 4, 64, 512),          # exactly one segment
    (449, 8, 4, 64, 512),          # one sample into the second segment
    (5000, 10, 2, 128, 512),
    (5001, 0, 1, 128, 1024),       # a single template (z = 0)
    (7777, 12, 3, 384, 1024),      # the paper's non-power-of-two filter length (Table 2)
    (7777, 12, 3, 384, 2048),
    (20011, 6, 2, 2, 2048),        # the shortest template
    (20011, 6, 2, 1000, 2048),     # m not a multiple of the thread count
    (30000, 6, 2, 2048, 4096),     # m = L/2, the largest allowed
    (30001, 6, 2, 510, 4096),
    (50000, 4, 2, 4096, 8192),
    (50001, 4, 2, 1022, 8192),
])
def test_edge_shapes_full_plane(torch, binding, oracle, n_f, z_max, z_step, m, L):
    wl = _custom(n_f, z_max, z_step, m, L, seed=n_f + m + L)
    p = gpu_power(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    check(p[0], ref, what=wl.name)


def test_random_templates_not_fdas_specific(torch, binding, oracle):
    """General convolution ("do not affect generality"): arbitrary complex taps, 3 batch items."""
    rng = np.random.default_rng(11)
    n_f, m, L, z_max = 9000, 100, 1024, 3
    H = (rng.standard_normal((7, m)) + 1j * rng.standard_normal((7, m))).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, 12, 3)
    wl = workload.Workload("random-taps", n_f, z_max, 1, m, L, 3, spec, H, [])
    p = gpu_power(wl, torch, binding)
    for b in range(3):
        ref = oracle.direct(spec[b], H.astype(np.complex128))
        check(p[b], ref, what=f"random taps b={b}")


def test_impulse_reproduces_template(torch, binding):
    """A = delta_{k0} => P[z][r0] = |h_z[r0 - k0 + m/2]|^2 (catches permutation / reversal bugs
    without the oracle: closed form from eq.(2))."""
    n_f, m, L, k0 = 6000, 128, 1024, 3000
    H = workload.templates(16, 2, m).astype(np.complex64)
    spec = np.zeros((1, n_f), np.complex64)
    spec[0, k0] = 1.0
    wl = workload.Workload("impulse", n_f, 16, 2, m, L, 1, spec, H, [])
    p = gpu_power(wl, torch, binding)[0]
    ref = np.zeros_like(p, dtype=np.float64)
    ref[:, k0 - m // 2: k0 + m // 2] = np.abs(H.astype(np.complex128)) ** 2
    assert np.max(np.abs(p - ref)) <= 1e-6 * ref.max()


def test_bitwise_deterministic_and_two_streams(torch, binding):
    wl = workload.make_config(1)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_templates(wl.templates)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    outs = [torch.empty((1, wl.n_z, wl.n_f), dtype=torch.float32, device="cuda") for _ in range(3)]
    plan.convolve(d_spec, outs[0])
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    plan.convolve(d_spec, outs[1], stream=s1)
    plan.convolve(d_spec, outs[2], stream=s2)
    torch.cuda.synchronize()
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])
    plan.destroy()


def test_set_templates_twice_and_errors(torch, binding):
    wl = workload.make_config(1)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    d_pow = torch.empty((1, wl.n_z, wl.n_f), dtype=torch.float32, device="cuda")
    with pytest.raises(binding.FdasError) as e:
        plan.convolve(d_spec, d_pow)
    assert e.value.status == binding.FDAS_ERR_NO_TEMPLATES
    plan.set_templates(np.zeros_like(wl.templates))
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    assert float(d_pow.abs().max()) == 0.0
    plan.set_templates(wl.templates)
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    assert float(d_pow.max()) > 10.0
    with pytest.raises(binding.FdasError) as e:
        plan.convolve(d_spec.data_ptr() + 4, d_pow)
    assert e.value.status == binding.FDAS_ERR_INVALID_ARG
    with pytest.raises(binding.FdasError):
        plan.convolve(None, d_pow)
    plan.destroy()


def test_convolve_host_equals_device(torch, binding):
    wl = workload.make_config(1)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_templates(wl.templates)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    d_pow = torch.empty((1, wl.n_z, wl.n_f), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    h_spec = torch.from_numpy(wl.spectrum).pin_memory()
    h_pow = torch.empty((1, wl.n_z, wl.n_f), dtype=torch.float32).pin_memory()
    plan.convolve_host(h_spec, h_pow)
    assert torch.equal(h_pow, d_pow.cpu())
    plan.destroy()


@pytest.mark.parametrize("L,m", [(512, 64), (1024, 128), (2048, 256), (4096, 512), (8192, 1024)])
def test_repeated_launches_are_bitwise_identical(torch, binding, L, m):
    """Race detector of last resort (compute-sanitizer is not available on the GPU pool): the hot loop
    re-uses its exchange buffers, template stage and tensor memory across z with one barrier per exchange;
    a missing ordering shows up as run-to-run differences.  Many CTAs per SM, several launches, two streams,
    every segment length; and the first launch is checked against an independent single-segment plan."""
    n_f = 40 * (L - m) + 17
    H = workload.templates(40, 2, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, 99 + L, 3)
    plan = binding.Plan(n_f, 40, 2, m, L, n_batch=3)
    plan.set_templates(H)
    d_spec = torch.from_numpy(spec).cuda()
    outs = [torch.full((3, 41, n_f), float("nan"), dtype=torch.float32, device="cuda") for _ in range(12)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for i, o in enumerate(outs):      # three streams: CTAs of different launches share SMs, large warp skews
        plan.convolve(d_spec, o, stream=streams[i % 3])
    torch.cuda.synchronize()
    for o in outs[1:]:
        assert torch.equal(outs[0], o)
    assert bool(torch.isfinite(outs[0]).all())
    # the same columns from a plan that sees only a window of the spectrum (different CTA <-> segment map)
    c0, c1 = 7 * (L - m), 9 * (L - m)
    lo, hi = c0 - m, c1 + m
    sub = binding.Plan(hi - lo, 40, 2, m, L, n_batch=1)
    sub.set_templates(H)
    d_sub = torch.from_numpy(np.ascontiguousarray(spec[1:2, lo:hi])).cuda()
    o_sub = torch.empty((1, 41, hi - lo), dtype=torch.float32, device="cuda")
    sub.convolve(d_sub, o_sub)
    torch.cuda.synchronize()
    a = outs[0][1, :, c0:c1].cpu().numpy().astype(np.float64)
    b = o_sub[0, :, c0 - lo:c1 - lo].cpu().numpy().astype(np.float64)
    assert np.max(np.abs(a - b)) <= 1e-5 * a.max()
    plan.destroy()
    sub.destroy()
