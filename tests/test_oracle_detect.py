"""Pins of oracle.blockmax (the detection step over the power plane, reading 17): a plain Python
scan, numpy on shapes it can express, invariants, and the C1 injected signal of BASELINE.json configs[0]."""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload


def _python_scan(p, blk):
    """The definition, written out: per row and block, the maximum and the lowest in-block offset."""
    rows, cols = p.shape
    n_blk = (cols + blk - 1) // blk
    mx = [[None] * n_blk for _ in range(rows)]
    ar = [[None] * n_blk for _ in range(rows)]
    for r in range(rows):
        for b in range(n_blk):
            best, arg = None, None
            for c in range(b * blk, min((b + 1) * blk, cols)):
                if best is None or p[r][c] > best:
                    best, arg = p[r][c], c - b * blk
            mx[r][b], ar[r][b] = best, arg
    return np.array(mx, dtype=np.float64), np.array(ar, dtype=np.int64)


@pytest.mark.parametrize("rows,cols,blk", [(1, 1, 1), (1, 7, 3), (3, 10, 10), (3, 10, 11), (2, 33, 8), (4, 64, 16), (2, 5, 1)])
def test_blockmax_equals_python_scan(oracle, rows, cols, blk):
    rng = np.random.default_rng(rows * 1000 + cols * 10 + blk)
    p = rng.exponential(2.0, size=(rows, cols))
    mx, ar = oracle.blockmax(p, blk, float32_decision=False)
    mx_ref, ar_ref = _python_scan(p, blk)
    assert np.array_equal(mx, mx_ref) and np.array_equal(ar, ar_ref)


def test_blockmax_equals_numpy_on_divisible_shapes(oracle):
    rng = np.random.default_rng(7)
    p = rng.exponential(2.0, size=(5, 12 * 32))
    mx, ar = oracle.blockmax(p, 32, float32_decision=False)
    q = p.reshape(5, 12, 32)
    assert np.array_equal(mx, q.max(axis=2))
    assert np.array_equal(ar, q.argmax(axis=2))          # numpy's argmax is the first occurrence
    # one block spanning the row is the row maximum
    mx1, ar1 = oracle.blockmax(p, 10 ** 6, float32_decision=False)
    assert np.array_equal(mx1[:, 0], p.max(axis=1)) and np.array_equal(ar1[:, 0], p.argmax(axis=1))
    # the maximum over the blocks of a row is the row maximum, and the argmax points at it
    assert np.array_equal(mx.max(axis=1), p.max(axis=1))
    b = mx.argmax(axis=1)
    assert np.array_equal(b * 32 + ar[np.arange(5), b], p.argmax(axis=1))


def test_ties_take_the_lowest_column(oracle):
    p = np.array([[1.0, 4.0, 4.0, 2.0, 4.0, 4.0, 0.0]])
    mx, ar = oracle.blockmax(p, 4, float32_decision=False)
    assert mx.tolist() == [[4.0, 4.0]] and ar.tolist() == [[1, 0]]
    # constant plane: every block reports offset 0, the ragged tail too
    mx, ar = oracle.blockmax(np.full((2, 10), 3.5), 4)
    assert np.all(mx == 3.5) and np.all(ar == 0) and mx.shape == (2, 3)


def test_float32_decision_rounds_before_comparing(oracle):
    """Two powers that differ only below float32 resolution: in double the later one wins, in the kernel's
    precision they tie and the lower column wins; the reported maximum is the rounded value."""
    a = 1.0 + 2.0 ** -30
    b = 1.0 + 2.0 ** -29
    p = np.array([[0.5, a, b, 0.25]])
    mx64, ar64 = oracle.blockmax(p, 4, float32_decision=False)
    mx32, ar32 = oracle.blockmax(p, 4, float32_decision=True)
    assert ar64.tolist() == [[2]] and mx64[0, 0] == b
    assert ar32.tolist() == [[1]] and mx32[0, 0] == 1.0


def test_c1_signal_is_the_global_block_maximum(oracle):
    """BASELINE.json configs[0]: the 8 sigma signal at r = 20000.3, z = +20 peaks in its own template row at
    column 20000 (tests/golden/c1_peak.txt).  With blocks of S = L - m = 384 columns that is block 52, offset 32."""
    wl = workload.make_config(1)
    p = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    blk = wl.seg_len - wl.m
    mx, ar = oracle.blockmax(p, blk)
    assert mx.shape == (33, (wl.n_f + blk - 1) // blk)
    r, b = np.unravel_index(np.argmax(mx), mx.shape)
    assert wl.z_values[r] == 20 and b == 20000 // blk and ar[r, b] == 20000 - b * blk
    assert np.float32(p[r, 20000]) == mx[r, b]
    # noise blocks: the maximum of 384 exponential(mean 2) powers is about 2 ln 384 = 11.9
    others = np.delete(mx.ravel(), np.argmax(mx))
    assert 9.0 < np.median(others) < 15.0


def test_bad_arguments(oracle):
    with pytest.raises(ValueError):
        oracle.blockmax(np.zeros((2, 4)), 0)
    with pytest.raises(ValueError):
        oracle.blockmax(np.zeros(4), 2)


# ---------------------------------------------------------------------------------------------------------
# oracle.candidates (reading 20): pinned by a scan of the PLANE ITSELF that never forms block maxima
# first, by counting identities, and by the C1 injected signal
# ---------------------------------------------------------------------------------------------------------
def _candidates_from_plane(p, blk, thr, cap):
    """Independent route: walk the plane column by column; a column is a candidate iff it is >= thr (float32) and
    no column of its block is larger and no earlier column of its block is equal."""
    p32 = p.astype(np.float32)
    thr = np.float32(thr)
    out = []
    for r in range(p.shape[0]):
        for c in range(p.shape[1]):
            b0, b1 = (c // blk) * blk, min((c // blk + 1) * blk, p.shape[1])
            v = p32[r, c]
            if v >= thr and all(p32[r, k] < v for k in range(b0, c)) and all(p32[r, k] <= v for k in range(c + 1, b1)):
                out.append((r, c, float(v)))
    return len(out), out[:cap]


@pytest.mark.parametrize("rows,cols,blk,thr,cap", [(1, 7, 3, 1.0, 10), (3, 40, 8, 3.0, 100), (3, 40, 8, 3.0, 4),
                                                   (4, 33, 5, 0.0, 1000), (2, 20, 4, 1e9, 5), (2, 20, 20, 2.0, 0)])
def test_candidates_equal_plane_scan(oracle, rows, cols, blk, thr, cap):
    rng = np.random.default_rng(rows + 10 * cols + blk)
    p = rng.exponential(2.0, size=(rows, cols))
    n, rr, cc, pp = oracle.candidates(p, blk, thr, cap)
    n_ref, ref = _candidates_from_plane(p, blk, thr, cap)
    assert n == n_ref
    assert list(zip(rr.tolist(), cc.tolist(), pp.tolist())) == ref


def test_candidates_counting_identities_and_order(oracle):
    rng = np.random.default_rng(20)
    p = rng.exponential(2.0, size=(6, 100))
    n_blk = 13                                                    # ceil(100 / 8)
    n0, r0, c0, p0 = oracle.candidates(p, 8, 0.0, 10 ** 6)        # threshold 0: every block of every row
    assert n0 == 6 * n_blk == r0.size
    assert oracle.candidates(p, 8, np.inf, 10)[0] == 0            # nothing is >= +inf
    n1, r1, c1, p1 = oracle.candidates(p, 8, 5.0, 10 ** 6)
    assert n1 == int((oracle.blockmax(p, 8)[0].astype(np.float32) >= np.float32(5.0)).sum())
    assert np.all(p1.astype(np.float32) >= np.float32(5.0))
    assert np.array_equal(p1, p[r1, c1].astype(np.float32))       # the reported power is the plane's float32 value there
    key = r1 * 1000 + c1
    assert np.all(np.diff(key) > 0)                               # ordered by (row, column), no duplicates
    # the threshold is inclusive, in float32
    v = float(np.float32(p1.min()))
    assert oracle.candidates(p, 8, v, 10 ** 6)[0] == n1
    assert oracle.candidates(p, 8, float(np.nextafter(np.float32(v), np.float32(np.inf))), 10 ** 6)[0] == n1 - 1
    # truncation keeps a prefix and still counts everything
    n2, r2, c2, p2 = oracle.candidates(p, 8, 5.0, 3)
    assert n2 == n1 and np.array_equal(r2, r1[:3]) and np.array_equal(c2, c1[:3]) and np.array_equal(p2, p1[:3])


def test_c1_signal_is_the_strongest_candidate(oracle):
    """BASELINE.json configs[0]: the z = +20 signal at bin 20000 (peak power 39 against noise maxima of 20-27).  With
    the threshold at 0.74 of the plane maximum the list holds only the signal's footprint -- its own row and the
    neighbouring trials, all at the signal's bin -- and its strongest entry is (row of z = +20, column 20000)."""
    wl = workload.make_config(1)
    p = oracle.direct(wl.spectrum[0], wl.templates.astype(np.complex128))
    n, rr, cc, pp = oracle.candidates(p, 384, 0.74 * p.max(), 1000)
    assert 2 <= n <= 8 and n == rr.size
    k = int(np.argmax(pp))
    assert wl.z_values[rr[k]] == 20 and cc[k] == 20000
    assert np.all(np.abs(cc - 20000) <= 4)
    assert all(abs(wl.z_values[r] - 20) <= 6 for r in rr)
