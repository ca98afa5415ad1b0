"""-m gpu: the multi-wave branches of the HOST-pointer entry points (fdas_convolve_host, fdas_detect_blockmax_host).

When a call is several waves of the persistent grid those entries cut the work items into pieces: the plane goes
back by per-piece 2-D copies on the plan's copy stream, the spectrum comes up piece by piece in front of the
launches.  The shape here has 5 waves (1200 work items on 296 CTAs) over 3 batch items of 400 segments, so pieces of
240 items straddle both batch-item boundaries and the ragged last segment of every item is inside a piece.  The
result must equal, bit for bit, what the DEVICE-pointer entries produce in one launch.
"""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

pytestmark = pytest.mark.gpu

L, M, Z_MAX, Z_STEP, N_BATCH = 4096, 512, 2, 1, 3
N_F = 400 * (L - M) - 1000   # 400 segments per item, the last one ragged


@pytest.fixture(scope="module")
def torch():
    import torch as _t
    if not _t.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    return _t


@pytest.fixture(scope="module")
def setup(torch):
    from paper_1711_10855_b200 import binding
    binding.lib()
    H = workload.templates(Z_MAX, Z_STEP, M).astype(np.complex64)
    spec = workload.noise_spectrum(N_F, 777, N_BATCH)
    plan = binding.Plan(N_F, Z_MAX, Z_STEP, M, L, n_batch=N_BATCH)
    plan.set_templates(H)
    assert plan.n_seg == 400
    assert plan.n_seg * N_BATCH >= 3 * plan.grid, "the shape must be at least three waves"
    yield plan, spec, H.shape[0]
    plan.destroy()


def test_convolve_host_chunked_equals_device(torch, setup):
    plan, spec, n_z = setup
    d_spec = torch.from_numpy(spec).cuda()
    d_pow = torch.full((N_BATCH, n_z, N_F), float("nan"), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    assert plan.last_launch_count == 1
    h_spec = torch.from_numpy(spec).pin_memory()
    h_pow = torch.full((N_BATCH, n_z, N_F), float("nan"), dtype=torch.float32).pin_memory()
    plan.convolve_host(h_spec, h_pow)
    assert plan.last_launch_count > 1, "the chunked branch did not run"
    assert not torch.isnan(h_pow).any()
    assert torch.equal(h_pow, d_pow.cpu())
    # pageable host memory takes the same branch (synchronous copies)
    h_pow2 = np.full((N_BATCH, n_z, N_F), np.nan, dtype=np.float32)
    plan.convolve_host(np.ascontiguousarray(spec), h_pow2)
    assert np.array_equal(h_pow2, d_pow.cpu().numpy())


def test_blockmax_host_chunked_equals_device(torch, setup):
    plan, spec, n_z = setup
    shape = (N_BATCH, n_z, plan.n_seg)
    d_spec = torch.from_numpy(spec).cuda()
    d_max = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
    d_arg = torch.full(shape, -7, dtype=torch.int32, device="cuda")
    plan.detect_blockmax(d_spec, d_max, d_arg)
    torch.cuda.synchronize()
    assert plan.last_launch_count == 1
    h_spec = torch.from_numpy(spec).pin_memory()
    for _ in range(2):   # twice: the second call re-uses the plan's staging buffer, which still holds the first upload
        h_max = torch.full(shape, float("nan"), dtype=torch.float32).pin_memory()
        h_arg = torch.full(shape, -7, dtype=torch.int32).pin_memory()
        plan.detect_blockmax_host(h_spec, h_max, h_arg)
        assert plan.last_launch_count > 1, "the chunked branch did not run"
        assert torch.equal(h_max, d_max.cpu()) and torch.equal(h_arg, d_arg.cpu())
    # a different spectrum through the same staging buffer: a piece launched before its upload would see the old one
    spec2 = workload.noise_spectrum(N_F, 778, N_BATCH)
    plan.detect_blockmax(torch.from_numpy(spec2).cuda(), d_max, d_arg)
    torch.cuda.synchronize()
    h_max = torch.full(shape, float("nan"), dtype=torch.float32).pin_memory()
    h_arg = torch.full(shape, -7, dtype=torch.int32).pin_memory()
    plan.detect_blockmax_host(torch.from_numpy(spec2).pin_memory(), h_max, h_arg)
    assert torch.equal(h_max, d_max.cpu()) and torch.equal(h_arg, d_arg.cpu())
