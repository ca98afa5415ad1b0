"""fdas_convolve_noalloc: the entry point for hosts that are not allowed to allocate GPU memory.

Who that is: a long-running search back end that handed out the whole card at start-up (a cudaMalloc in mid-run
stalls all its streams and may find nothing left), a process whose free memory sits in a framework's pool where
the driver cannot see it, code working under a fixed memory budget.  For them the library keeps the memory a plan
would have allocated -- work counters, twiddle table, transformed template bank -- in a static device array inside
libfdas.so (limit: n_z * segment_len <= 2^20), and every call rebuilds all of it on the caller's stream.

What is checked here: the power plane of the new entry point against the plane the ordinary plan path
(fdas_plan_create + fdas_set_templates + fdas_convolve) produces from the same inputs, at the tolerance of
tests/parity.py, on calls made back to back WITHOUT a synchronisation in between and with a different segment
length, template width and bank each time -- so a call that trusted what its predecessor left in the shared
array (stale twiddles, stale bank, counters not at zero) fails.  Both shapes have more segments than the
persistent grid has CTAs, so the work counters in the static array are really used.

The file is named to be collected last: pytest -x stops at the first failure and this test must not hide the
parity suite.  It needs nothing from the other tests and passes alone in a fresh process too.
"""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import check


@pytest.fixture(scope="module")
def binding():
    from paper_1711_10855_b200 import binding as _b
    _b.lib()  # raises if libfdas.so is missing: no fallback
    return _b


def test_limit_and_arguments_checked_before_the_gpu_is_touched(binding):
    """Runs without a GPU: sizes and pointers are validated before the first CUDA call."""
    L = binding.lib()
    p = 4096  # any non-NULL, aligned address: these calls must return before it is used
    assert binding.NOALLOC_MAX_BANK == 1 << 20
    # 401 templates x 4096 = 1.6 M elements: beyond the static bank
    assert L.fdas_convolve_noalloc(1 << 20, 1, 200, 1, 512, 4096, p, p, p, None) == binding.FDAS_ERR_TOO_LARGE
    assert L.fdas_convolve_noalloc(1 << 20, 1, 64, 1, 512, 8192, p, p, p, None) == binding.FDAS_ERR_TOO_LARGE  # 129 x 8192
    assert binding.status_string(binding.FDAS_ERR_TOO_LARGE) == "FDAS_ERR_TOO_LARGE"
    # the rules of fdas_plan_create / fdas_convolve
    assert L.fdas_convolve_noalloc(0, 1, 4, 2, 64, 512, p, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 0, 4, 2, 64, 512, p, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 5, 2, 64, 512, p, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 63, 512, p, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 300, 512, p, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 256, p, p, p, None) == binding.FDAS_ERR_UNSUPPORTED
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 512, None, p, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 512, p, None, p, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 512, p, p, None, None) == binding.FDAS_ERR_INVALID_ARG
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 512, p + 4, p, p, None) == binding.FDAS_ERR_INVALID_ARG  # misaligned taps
    assert L.fdas_convolve_noalloc(1000, 1, 4, 2, 64, 512, p, p + 4, p, None) == binding.FDAS_ERR_INVALID_ARG


def _case(n_f, z_max, z_step, m, L, seed, n_batch):
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, seed, n_batch)
    return dict(n_f=n_f, z_max=z_max, z_step=z_step, m=m, L=L, n_batch=n_batch, H=H, spec=spec, n_z=H.shape[0])


@pytest.mark.gpu
def test_noalloc_equals_plan_path_on_consecutive_calls(binding):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")

    cases = [
        _case(1 << 20, 10, 2, 64, 512, seed=901, n_batch=1),      # 2341 segments on 1184 CTAs, m = L/8
        _case(600_001, 12, 3, 384, 2048, seed=902, n_batch=2),    # 2 x 361 segments on 592 CTAs, ragged tail, m = 384
    ]
    # the existing path first: one plan per case
    for c in cases:
        plan = binding.Plan(c["n_f"], c["z_max"], c["z_step"], c["m"], c["L"], n_batch=c["n_batch"])
        plan.set_templates(c["H"])
        assert plan.n_seg * c["n_batch"] > plan.grid, "the shape must need the work counters"
        c["d_spec"] = torch.from_numpy(np.ascontiguousarray(c["spec"])).cuda()
        d_ref = torch.full((c["n_batch"], c["n_z"], c["n_f"]), float("nan"), dtype=torch.float32, device="cuda")
        plan.convolve(c["d_spec"], d_ref)
        torch.cuda.synchronize()
        c["ref"] = d_ref.cpu().numpy()
        plan.destroy()
        del d_ref
        c["d_H"] = torch.from_numpy(np.ascontiguousarray(c["H"])).cuda()

    # the entry point under test: A, B, A again, back to back on one stream, no synchronisation in between
    order = [0, 1, 0]
    outs = []
    for i in order:
        c = cases[i]
        d_out = torch.full((c["n_batch"], c["n_z"], c["n_f"]), float("nan"), dtype=torch.float32, device="cuda")
        outs.append(d_out)
    for i, d_out in zip(order, outs):
        c = cases[i]
        binding.convolve_noalloc(c["n_f"], c["n_batch"], c["z_max"], c["z_step"], c["m"], c["L"], c["d_H"], c["d_spec"], d_out)
    torch.cuda.synchronize()

    for k, (i, d_out) in enumerate(zip(order, outs)):
        c = cases[i]
        got = d_out.cpu().numpy()
        for b in range(c["n_batch"]):
            a, r = check(got[b], c["ref"][b].astype(np.float64), what=f"call {k} (case {i}, item {b})")
            n_diff = int(np.count_nonzero(got[b] != c["ref"][b]))
            print(f"noalloc call {k} case {i} item {b}: abs {a:.2e} rel {r:.2e}, {n_diff} of {got[b].size} values differ in bits")
    # the same inputs give the same bits, whatever ran in between
    assert torch.equal(outs[0], outs[2])
