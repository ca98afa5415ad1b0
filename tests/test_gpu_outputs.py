"""-m gpu: the two other outputs of the hot kernel against the oracle.

fdas_convolve_complex  the paper's general convolution (Table 2: filter lengths 64 ... 512 incl. 384):
                       the filtered spectrum A' of eq.(2) itself, against oracle.direct(want="amp").
fdas_detect_blockmax   the hot path fused with the block-maximum step of detection (reading 17), against
                       oracle.blockmax of the oracle's power plane.  The argmax is an integer decided by floating
                       point: both sides decide on float32 powers; where the two best columns of a block are closer
                       than the parity tolerance either is valid, and the test checks exactly that.
"""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import ABS_TOL

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


def _custom(n_f, z_max, z_step, m, L, seed, n_batch=1, taps=None):
    H = workload.templates(z_max, z_step, m).astype(np.complex64) if taps is None else taps
    spec = workload.noise_spectrum(n_f, seed, n_batch)
    return workload.Workload(f"custom[{n_f},{m},{L}]", n_f, z_max, z_step, m, L, n_batch, spec, H, [])


# ---------------------------------------------------------------------------------------------------------
# complex output
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("m,L,n_f", [(64, 512, 3001), (128, 1024, 5000), (256, 2048, 9000), (384, 2048, 7777),
                                     (384, 4096, 12000), (512, 4096, 15000), (1024, 8192, 20000)])
def test_complex_output_matches_eq2(torch, binding, oracle, m, L, n_f):
    """|A'_gpu - A'_ref| <= 0.5e-4 max|A'_ref|: the amplitude form of north_star's 1e-4 max(P) (dP = 2 |A| d|A|)."""
    wl = _custom(n_f, 12, 3, m, L, seed=500 + m + L, n_batch=2)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len, n_batch=2)
    plan.set_templates(wl.templates)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    d_amp = torch.full((2, wl.n_z, n_f), float("nan"), dtype=torch.complex64, device="cuda")
    plan.convolve_complex(d_spec, d_amp)
    torch.cuda.synchronize()
    a = d_amp.cpu().numpy()
    assert np.all(np.isfinite(a.view(np.float32)))
    for b in range(2):
        ref = oracle.direct(wl.spectrum[b], wl.templates.astype(np.complex128), want="amp")
        err = np.abs(a[b].astype(np.complex128) - ref).max() / np.abs(ref).max()
        assert err <= 0.5 * ABS_TOL, (m, L, b, err)
    # and its power is what fdas_convolve writes, to rounding (the phase fix-up is a unit rotation)
    d_pow = torch.empty((2, wl.n_z, n_f), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    p = d_pow.cpu().numpy().astype(np.float64)
    assert np.abs(np.abs(a.astype(np.complex128)) ** 2 - p).max() <= 1e-5 * p.max()
    plan.destroy()


def test_complex_output_random_taps_not_symmetric(torch, binding, oracle):
    """Arbitrary complex taps (no FDAS symmetry): pins conj-not-reversed and the tap order on the complex output."""
    rng = np.random.default_rng(77)
    H = (rng.standard_normal((5, 128)) + 1j * rng.standard_normal((5, 128))).astype(np.complex64)
    wl = _custom(4000, 4, 2, 128, 1024, seed=78, taps=H)
    plan = binding.Plan(wl.n_f, 4, 2, 128, 1024)
    plan.set_templates(H)
    d_amp = torch.empty((1, 5, wl.n_f), dtype=torch.complex64, device="cuda")
    plan.convolve_complex(torch.from_numpy(wl.spectrum).cuda(), d_amp)
    torch.cuda.synchronize()
    ref = oracle.direct(wl.spectrum[0], H.astype(np.complex128), want="amp")
    assert np.abs(d_amp.cpu().numpy()[0] - ref).max() <= 0.5 * ABS_TOL * np.abs(ref).max()
    plan.destroy()


# ---------------------------------------------------------------------------------------------------------
# block maxima
# ---------------------------------------------------------------------------------------------------------
def _gpu_blockmax(wl, torch, binding, n_batch=None):
    nb = wl.spectrum.shape[0] if n_batch is None else n_batch
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len, n_batch=nb)
    plan.set_templates(wl.templates)
    n_blk, blk = plan.n_seg, plan.step
    d_max = torch.full((nb, wl.n_z, n_blk), float("nan"), dtype=torch.float32, device="cuda")
    d_arg = torch.full((nb, wl.n_z, n_blk), -7, dtype=torch.int32, device="cuda")
    plan.detect_blockmax(torch.from_numpy(np.ascontiguousarray(wl.spectrum[:nb])).cuda(), d_max, d_arg)
    torch.cuda.synchronize()
    plan.destroy()
    return d_max.cpu().numpy(), d_arg.cpu().numpy(), blk


def _check_blockmax(gmax, garg, p_ref, blk, oracle, what=""):
    """gmax/garg [rows][n_blk] from the GPU; p_ref float64 [rows][n_f] from the oracle."""
    rmax, rarg = oracle.blockmax(p_ref, blk)
    assert gmax.shape == rmax.shape and garg.shape == rarg.shape, (gmax.shape, rmax.shape)
    tol = ABS_TOL * float(p_ref.max())
    assert np.all(np.isfinite(gmax)), what
    assert np.abs(gmax.astype(np.float64) - rmax).max() <= tol, what
    n_f = p_ref.shape[1]
    n_blk = rmax.shape[1]
    width = np.minimum(blk, n_f - blk * np.arange(n_blk))
    assert np.all(garg >= 0) and np.all(garg < width[None, :]), what            # a column of its own block
    same = garg == rarg
    # where the index differs the GPU's column must be a near tie: its oracle power within 2 tol of the block maximum
    rr, bb = np.nonzero(~same)
    for r, b in zip(rr, bb):
        assert p_ref[r, b * blk + garg[r, b]] >= rmax[r, b] - 2 * tol, (what, r, b)
    # and it must be exact wherever the block's runner-up is further than that away
    return float(same.mean())


def test_blockmax_c1_full(torch, binding, oracle):
    wl = workload.make_config(1)
    gmax, garg, blk = _gpu_blockmax(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    frac = _check_blockmax(gmax[0], garg[0], ref, blk, oracle, "C1")
    r, b = np.unravel_index(np.argmax(gmax[0]), gmax[0].shape)
    assert wl.z_values[r] == 20 and b * blk + garg[0, r, b] == 20000        # the injected signal (BASELINE configs[0])
    assert frac > 0.999
    print(f"C1 blockmax: {frac:.5f} of argmax entries identical")


def test_blockmax_c2_full(torch, binding, oracle):
    wl = workload.make_config(2)
    gmax, garg, blk = _gpu_blockmax(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    frac = _check_blockmax(gmax[0], garg[0], ref, blk, oracle, "C2")
    assert frac > 0.999
    # every injected signal is the maximum of its block in its own row
    for sig in wl.signals[0]:
        r = int(np.argmin(np.abs(wl.z_values - sig.z)))
        b = int(round(sig.r_c)) // blk
        assert abs(b * blk + int(garg[0, r, b]) - sig.r_c) <= 1.0


@pytest.mark.parametrize("n_f,z_max,z_step,m,L", [
    (1, 4, 2, 64, 512), (63, 4, 2, 64, 512), (447, 8, 4, 64, 512), (448, 8, 4, 64, 512), (449, 8, 4, 64, 512),
    (5001, 0, 1, 128, 1024), (7777, 12, 3, 384, 2048), (20011, 6, 2, 1000, 2048), (30000, 6, 2, 2048, 4096),
    (40000, 4, 2, 1024, 8192), (9000, 6, 2, 512, 8192),
])
def test_blockmax_edge_shapes(torch, binding, oracle, n_f, z_max, z_step, m, L):
    wl = _custom(n_f, z_max, z_step, m, L, seed=n_f + m)
    gmax, garg, blk = _gpu_blockmax(wl, torch, binding)
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    _check_blockmax(gmax[0], garg[0], ref, blk, oracle, wl.name)


def test_blockmax_ties_resolve_to_lowest_column(torch, binding):
    """A zero spectrum: every power is exactly 0, every block must report (0, offset 0)."""
    wl = _custom(10000, 4, 2, 128, 1024, seed=1)
    wl.spectrum[:] = 0
    gmax, garg, blk = _gpu_blockmax(wl, torch, binding)
    assert np.all(gmax == 0) and np.all(garg == 0)


def test_blockmax_c3_rows_via_ols_and_batched_c5(torch, binding, oracle):
    """Full size, the launch configuration bench.py times.  C3: six rows of the plane from the oracle's double
    overlap-and-save (pinned to the direct sum in tests/test_oracle_direct.py), all 1171 blocks of each.  C5: the
    batched call equals per-spectrum calls, and one batch item's rows are checked the same way."""
    wl = workload.make_config(3)
    gmax, garg, blk = _gpu_blockmax(wl, torch, binding)
    H = wl.templates.astype(np.complex128)
    worst = 1.0
    for r in (0, 37, 100, 101, 163, 200):
        ref = oracle.ols(wl.spectrum[0], H, wl.seg_len, rows=(r, r + 1))
        worst = min(worst, _check_blockmax(gmax[0][r:r + 1], garg[0][r:r + 1], ref, blk, oracle, f"C3 row {r}"))
    for sig in wl.signals[0]:
        r = int(np.argmin(np.abs(wl.z_values - sig.z)))
        b = int(round(sig.r_c)) // blk
        assert abs(b * blk + int(garg[0, r, b]) - sig.r_c) <= 1.0 and gmax[0, r, b] > 20.0
    assert worst > 0.995
    wl5 = workload.make_config(5, n_batch=6)
    g5, a5, blk5 = _gpu_blockmax(wl5, torch, binding)
    one = workload.make_config(5, n_batch=6)
    one.spectrum = wl5.spectrum[4:5]
    g1, a1, _ = _gpu_blockmax(one, torch, binding, n_batch=1)
    assert np.array_equal(g5[4], g1[0]) and np.array_equal(a5[4], a1[0])
    H5 = wl5.templates.astype(np.complex128)
    for r in (0, 42, 84):
        ref = oracle.ols(wl5.spectrum[4], H5, wl5.seg_len, rows=(r, r + 1))
        _check_blockmax(g5[4][r:r + 1], a5[4][r:r + 1], ref, blk5, oracle, f"C5[4] row {r}")


def test_blockmax_host_entry_and_determinism(torch, binding):
    wl = workload.make_config(2)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_templates(wl.templates)
    shape = (1, wl.n_z, plan.n_seg)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    outs = []
    for _ in range(3):
        d_max = torch.empty(shape, dtype=torch.float32, device="cuda")
        d_arg = torch.empty(shape, dtype=torch.int32, device="cuda")
        plan.detect_blockmax(d_spec, d_max, d_arg)
        outs.append((d_max, d_arg))
    torch.cuda.synchronize()
    for m_, a_ in outs[1:]:
        assert torch.equal(m_, outs[0][0]) and torch.equal(a_, outs[0][1])
    h_spec = torch.from_numpy(wl.spectrum).pin_memory()
    h_max = torch.empty(shape, dtype=torch.float32).pin_memory()
    h_arg = torch.empty(shape, dtype=torch.int32).pin_memory()
    plan.detect_blockmax_host(h_spec, h_max, h_arg)
    assert torch.equal(h_max, outs[0][0].cpu()) and torch.equal(h_arg, outs[0][1].cpu())
    # the block maxima are the maxima of the plane fdas_convolve writes, bit for bit (same kernel arithmetic)
    d_pow = torch.empty((1, wl.n_z, wl.n_f), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    S = plan.step
    pad = plan.n_seg * S - wl.n_f
    pp = torch.nn.functional.pad(d_pow, (0, pad), value=-1.0).view(1, wl.n_z, plan.n_seg, S)
    assert torch.equal(pp.max(dim=3).values, outs[0][0])
    plan.destroy()
