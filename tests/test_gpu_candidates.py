"""-m gpu: fdas_detect_candidates (threshold + ordered candidate list, reading 20) against oracle.candidates.

Floating point decides integers here twice: whether a block maximum passes the threshold, and which column attains the
maximum.  Both sides decide on float32 powers, but their powers differ by rounding (<= ABS_TOL * max P by the parity
tests), so:
  * the threshold of every test is placed in a gap of the ORACLE's block maxima that is wider than 4 x that tolerance:
    then membership is unambiguous and the (item, row, block) triples must be identical, in the same order;
  * the column must equal the oracle's unless the block's two best columns are closer than twice the tolerance (the
    near-tie rule of the block-maximum tests), in which case it must be one of those near-ties;
  * the power must agree within the tolerance.
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


def _threshold_in_a_gap(block_maxima, level, tol):
    """A threshold near `level` with no oracle block maximum within 2 * tol of it."""
    v = np.unique(block_maxima.astype(np.float32).ravel())
    i = int(np.searchsorted(v, level))
    for k in range(i, v.size - 1):
        if float(v[k + 1]) - float(v[k]) > 4 * tol:
            return 0.5 * (float(v[k]) + float(v[k + 1]))
    raise AssertionError("no gap wide enough above the level")


def _same(a, b):
    """Record arrays equal byte for byte (the untouched tail is -1 = NaN in the power field, so compare the bits)."""
    return np.array_equal(np.ascontiguousarray(a).view(np.int32), np.ascontiguousarray(b).view(np.int32))


def _gpu_candidates(plan, torch, binding, d_spec, thr, cap, host_spec=None):
    if host_spec is None:
        d_cand = torch.full((max(cap, 1), 4), -1, dtype=torch.int32, device="cuda")
        d_count = torch.full((2,), -1, dtype=torch.int32, device="cuda")
        plan.detect_candidates(d_spec, thr, cap, d_cand, d_count)
        torch.cuda.synchronize()
        cand, count = d_cand.cpu().numpy(), d_count.cpu().numpy()
    else:
        h_cand = torch.full((max(cap, 1), 4), -1, dtype=torch.int32).pin_memory()
        h_count = torch.full((2,), -1, dtype=torch.int32).pin_memory()
        plan.detect_candidates_host(host_spec, thr, cap, h_cand, h_count)
        cand, count = h_cand.numpy().copy(), h_count.numpy().copy()
    rec = cand.view(binding.CANDIDATE_DTYPE).reshape(-1)
    return int(count[0]), int(count[1]), rec


def _compare(rec, n_found, n_written, ref_planes, blk, thr, cap, tol, what):
    """ref_planes: list over batch items of the oracle's float64 plane [n_z][n_f]."""
    import oracle
    exp = []
    for b, p in enumerate(ref_planes):
        n, rr, cc, pp = oracle.candidates(p, blk, thr, 1 << 30)
        exp += [(b, int(r), int(c), float(v)) for r, c, v in zip(rr, cc, pp)]
    assert n_found == len(exp), (what, n_found, len(exp))
    assert n_written == min(len(exp), cap), what
    n_same = 0
    for k in range(n_written):
        b, r, c, v = exp[k]
        g = rec[k]
        assert (int(g["item"]), int(g["row"])) == (b, r), (what, k)
        assert int(g["column"]) // blk == c // blk, (what, k, "block")
        assert abs(float(g["power"]) - v) <= tol, (what, k)
        if int(g["column"]) == c:
            n_same += 1
        else:
            assert ref_planes[b][r, int(g["column"])] >= v - 2 * tol, (what, k, "not a near-tie")
    # untouched beyond the written part
    assert np.all(rec[n_written:]["item"] == -1)
    return n_same


@pytest.mark.parametrize("cfg,level", [(1, 14.0), (2, 20.0)])
def test_candidates_full_plane_configs(torch, binding, oracle, cfg, level):
    wl = workload.make_config(cfg)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_templates(wl.templates)
    blk = plan.step
    ref = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    tol = ABS_TOL * float(ref.max())
    thr = _threshold_in_a_gap(oracle.blockmax(ref, blk)[0], level, tol)
    d_spec = torch.from_numpy(wl.spectrum).cuda()
    n_found, n_written, rec = _gpu_candidates(plan, torch, binding, d_spec, thr, 1 << 16)
    assert 10 < n_found < (1 << 16)
    n_same = _compare(rec, n_found, n_written, [ref], blk, thr, 1 << 16, tol, f"C{cfg}")
    # a capacity smaller than the list: the same prefix, the full count
    cap = n_found // 3
    f2, w2, rec2 = _gpu_candidates(plan, torch, binding, d_spec, thr, cap)
    assert (f2, w2) == (n_found, cap) and _same(rec2[:cap], rec[:cap])
    # capacity 0 (NULL list allowed), a threshold nothing reaches, a threshold everything reaches
    d_count = torch.full((2,), -1, dtype=torch.int32, device="cuda")
    plan.detect_candidates(d_spec, thr, 0, None, d_count)
    torch.cuda.synchronize()
    assert d_count.tolist() == [n_found, 0]
    assert _gpu_candidates(plan, torch, binding, d_spec, float("inf"), 8)[:2] == (0, 0)
    f3, w3, _ = _gpu_candidates(plan, torch, binding, d_spec, 0.0, 8)
    assert (f3, w3) == (wl.n_z * plan.n_seg, 8)
    # the HOST entry returns the same bytes; so does a second run
    h_spec = torch.from_numpy(wl.spectrum).pin_memory()
    f4, w4, rec4 = _gpu_candidates(plan, torch, binding, None, thr, 1 << 16, host_spec=h_spec)
    assert (f4, w4) == (n_found, n_written) and _same(rec4[:w4], rec[:n_written])
    f5, w5, rec5 = _gpu_candidates(plan, torch, binding, d_spec, thr, 1 << 16)
    assert (f5, w5) == (n_found, n_written) and _same(rec5, rec)
    print(f"C{cfg}: threshold {thr:.3f}: {n_found} candidates, {n_same} columns identical, the others near-ties")
    plan.destroy()


def test_candidates_batched_ragged(torch, binding, oracle):
    """Three spectra, ragged last block, the 64-thread plan: the item field and the order across items."""
    n_f, z_max, z_step, m, L = 30011, 8, 2, 64, 512
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    spec = workload.noise_spectrum(n_f, 321, 3)
    plan = binding.Plan(n_f, z_max, z_step, m, L, n_batch=3)
    plan.set_templates(H)
    refs = [oracle.direct(spec[b], H.astype(np.complex128)) for b in range(3)]
    tol = ABS_TOL * max(float(r.max()) for r in refs)
    allmax = np.concatenate([oracle.blockmax(r, plan.step)[0].ravel() for r in refs])
    thr = _threshold_in_a_gap(allmax, 12.0, tol)
    n_found, n_written, rec = _gpu_candidates(plan, torch, binding, torch.from_numpy(spec).cuda(), thr, 4096)
    assert n_found > 30
    _compare(rec, n_found, n_written, refs, plan.step, thr, 4096, tol, "batched")
    assert set(rec[:n_written]["item"].tolist()) == {0, 1, 2}
    plan.destroy()


def test_candidates_c3_full_size(torch, binding, oracle):
    """BASELINE.json config 3 at full size, the launch configuration bench.py times (chunked upload in the HOST entry):
    every candidate against the oracle's overlap-and-save plane, streamed in row chunks."""
    wl = workload.make_config(3)
    plan = binding.Plan(wl.n_f, wl.z_max, wl.z_step, wl.m, wl.seg_len)
    plan.set_templates(wl.templates)
    blk = plan.step
    H = wl.templates.astype(np.complex128)
    # the oracle's block maxima of the whole plane, and its rows kept only where a block maximum is large (near-tie rule)
    chunks, pmax = [], 0.0
    for r0 in range(0, wl.n_z, 12):
        r1 = min(wl.n_z, r0 + 12)
        p = oracle.ols(wl.spectrum[0], H, wl.seg_len, rows=(r0, r1))
        pmax = max(pmax, float(p.max()))
        mx, ar = oracle.blockmax(p, blk)
        sel = np.argwhere(mx.astype(np.float32) >= np.float32(28.0))
        near = {(r0 + int(r), int(b)): p[r, b * blk:min((b + 1) * blk, wl.n_f)].copy() for r, b in sel}
        chunks.append((r0, mx, ar, near))
    tol = ABS_TOL * pmax
    thr = _threshold_in_a_gap(np.concatenate([c[1].ravel() for c in chunks]), 28.5, tol)
    exp = []
    for r0, mx, ar, near in chunks:
        for r in range(mx.shape[0]):
            for b in range(mx.shape[1]):
                if np.float32(mx[r, b]) >= np.float32(thr):
                    exp.append((r0 + r, b * blk + int(ar[r, b]), float(mx[r, b]), near[(r0 + r, b)]))
    cap = 1 << 16
    h_spec = torch.from_numpy(wl.spectrum).pin_memory()
    n_found, n_written, rec = _gpu_candidates(plan, torch, binding, None, thr, cap, host_spec=h_spec)
    assert plan.last_launch_count > 4, "chunked upload + three compaction launches"
    assert n_found == len(exp) and n_written == min(cap, len(exp)) and 20 < n_found < cap
    n_same = 0
    for k, (r, c, v, blockvals) in enumerate(exp):
        g = rec[k]
        assert (int(g["item"]), int(g["row"]), int(g["column"]) // blk) == (0, r, c // blk), k
        assert abs(float(g["power"]) - v) <= tol
        if int(g["column"]) == c:
            n_same += 1
        else:
            assert blockvals[int(g["column"]) % blk] >= v - 2 * tol
    f2, w2, rec2 = _gpu_candidates(plan, torch, binding, torch.from_numpy(wl.spectrum).cuda(), thr, cap)
    assert (f2, w2) == (n_found, n_written) and _same(rec2[:w2], rec[:n_written])
    print(f"C3: threshold {thr:.3f}: {n_found} candidates of {wl.n_z * plan.n_seg} block maxima, {n_same} columns identical")
    plan.destroy()
