"""Shared helpers of the -m gpu parity tests: run the CUDA path through the C-ABI binding, run the
oracle on the same seeded input, compare with the BASELINE.json tolerances.

    |P_gpu - P_ref| <= 1e-4 * max(P_ref)            everywhere
    |P_gpu - P_ref| <= 1e-3 * P_ref                 wherever P_ref >= 1e-2 * max(P_ref)

max(P_ref) is taken per spectrum (reading 13).  When the oracle is evaluated on a sample of
column blocks only, the max over the sample is used: it is <= the true max, so the test is stricter.
"""
import numpy as np

ABS_TOL = 1e-4
REL_TOL = 1e-3
REL_FLOOR = 1e-2


def gpu_power(wl, torch, binding, spectrum=None, n_batch=None):
    """Run fdas_convolve on workload wl; returns a float32 numpy array [n_batch][n_z][n_f]."""
    spec = wl.spectrum if spectrum is None else spectrum
    nb = spec.shape[0] if n_batch is None else n_batch
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len, n_batch=nb)
    plan.set_templates(wl.templates)
    d_spec = torch.from_numpy(np.ascontiguousarray(spec)).cuda()
    d_pow = torch.full((nb, wl.n_z, wl.n_f), float("nan"), dtype=torch.float32, device="cuda")
    plan.convolve(d_spec, d_pow)
    torch.cuda.synchronize()
    out = d_pow.cpu().numpy()
    plan.destroy()
    return out


def check(p_gpu, p_ref, p_max=None, what=""):
    """p_gpu float32, p_ref float64, same shape.  Returns (max abs err / max, max rel err above floor)."""
    assert p_gpu.shape == p_ref.shape, (p_gpu.shape, p_ref.shape)
    assert np.all(np.isfinite(p_gpu)), f"{what}: non-finite or unwritten (NaN-filled) outputs"
    pm = float(p_ref.max()) if p_max is None else float(p_max)
    err = np.abs(p_gpu.astype(np.float64) - p_ref)
    a = float(err.max()) / pm
    big = p_ref >= REL_FLOOR * pm
    r = float((err[big] / p_ref[big]).max()) if big.any() else 0.0
    assert a <= ABS_TOL, f"{what}: max|dP|/max(P) = {a:.3e} > {ABS_TOL}"
    assert r <= REL_TOL, f"{what}: max rel err = {r:.3e} > {REL_TOL}"
    return a, r


def sample_blocks(wl, plan_step, n_random, width, rng, extra_cols=()):
    """Column blocks [c0, c1) for sampled parity: both edges, segment seams, signals, random."""
    n_f = wl.n_f
    S = plan_step
    blocks = [(0, min(width, n_f)), (max(0, n_f - width), n_f)]
    n_seg = (n_f + S - 1) // S
    for s in (1, 2, n_seg // 2, n_seg - 1):       # seams between segments
        c = s * S
        if 0 < c < n_f:
            blocks.append((max(0, c - width // 2), min(n_f, c + width // 2)))
    for c in extra_cols:
        c = int(c)
        blocks.append((max(0, c - width // 2), min(n_f, c + width // 2)))
    for _ in range(n_random):
        c = int(rng.integers(0, max(1, n_f - width)))
        blocks.append((c, min(n_f, c + width)))
    return blocks
