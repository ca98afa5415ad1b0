"""Pins for the oracle's direct sum (eq.(2)) and its double overlap-and-save
(PAPER.md line 31).  CPU only.  Nothing here calls the CUDA path."""
import os

import numpy as np
import pytest

from paper_1711_10855_b200 import workload

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "c1_peak.txt")


def _rand(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(n) + 1j * rng.standard_normal(n)


def _bank(n_z, m, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n_z, m)) + 1j * rng.standard_normal((n_z, m))


def test_direct_is_eq2_written_out(oracle):
    # P[z][r0] = | sum_j A[r0 + m/2 - j] conj(h_z[j]) |^2 with Python loops, tiny case
    n_f, m, n_z = 23, 6, 3
    A, H = _rand(n_f, 1), _bank(n_z, m, 2)
    ref = np.zeros((n_z, n_f), complex)
    for z in range(n_z):
        for r0 in range(n_f):
            for j in range(m):
                k = r0 + m // 2 - j
                if 0 <= k < n_f:
                    ref[z, r0] += A[k] * np.conj(H[z, j])
    p, a = oracle.direct(A, H, want="both")
    assert np.max(np.abs(a - ref)) < 1e-13
    assert np.max(np.abs(p - np.abs(ref) ** 2)) < 1e-12


@pytest.mark.parametrize("n_f,m", [(1000, 64), (777, 128), (130, 128), (64, 128)])
def test_direct_equals_numpy_convolve(oracle, n_f, m):
    # textbook reduction: A' = (A conv conj(h))[m/2 : m/2 + n_f]
    A, H = _rand(n_f, 3), _bank(4, m, 4)
    a = oracle.direct(A, H, want="amp")
    for z in range(4):
        ref = np.convolve(A, np.conj(H[z]))[m // 2: m // 2 + n_f]
        assert np.max(np.abs(a[z] - ref)) < 1e-11


def test_conjugate_not_reversed(oracle):
    # eq.(2) multiplies by conj(H_{r0-k}); using H unconjugated, or reversed, must differ
    A, H = _rand(300, 5), _bank(1, 32, 6)
    a = oracle.direct(A, H, want="amp")[0]
    wrong1 = np.convolve(A, H[0])[16:316]
    wrong2 = np.convolve(A, np.conj(H[0][::-1]))[16:316]
    assert np.max(np.abs(a - wrong1)) > 0.5 and np.max(np.abs(a - wrong2)) > 0.5


def test_impulse_reproduces_template_unreversed(oracle):
    # A = delta_{k0}  =>  P[z][r0] = |h_z[r0 - k0 + m/2]|^2, zero outside [k0 - m/2, k0 + m/2)
    n_f, m, k0 = 500, 64, 200
    H = oracle.templates(8, 4, m)
    A = np.zeros(n_f, complex); A[k0] = 1.0
    p = oracle.direct(A, H)
    for z in range(H.shape[0]):
        ref = np.zeros(n_f)
        ref[k0 - m // 2: k0 + m // 2] = np.abs(H[z]) ** 2
        assert np.max(np.abs(p[z] - ref)) < 1e-15


def test_constant_input_interior(oracle):
    # A = 1  =>  interior P = |sum_j conj(h_z[j])|^2
    n_f, m = 400, 32
    H = _bank(3, m, 8)
    p = oracle.direct(np.ones(n_f, complex), H)
    for z in range(3):
        assert np.max(np.abs(p[z, m:n_f - m] - abs(np.sum(H[z])) ** 2)) < 1e-10


def test_noise_free_unit_signal_matched_power(oracle):
    # unit signal at integer r_c with the matching z: P[z][r_c] = (window energy of the raw response)
    m, z, r_c, n_f = 128, 32, 700, 2048
    bins = np.arange(n_f)
    A = np.array([oracle.response((r_c - 0.5 * z) - b, z) for b in bins])
    H = oracle.templates(32, 2, m)
    p = oracle.direct(A, H)
    row = 32  # z = +32
    assert np.argmax(p) == row * n_f + r_c
    assert abs(p[row, r_c] - 0.999929) < 2e-6     # SURVEY.md Appendix A.2 window energy, m=128, z=32
    # the mismatched-sign row is much weaker
    assert p[0, r_c] < 0.2


def test_c1_injected_signal_peaks_in_matching_row(oracle):
    g = {}
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            g[k] = float(v)
    w = workload.make_config(1)
    p = oracle.direct(w.spectrum[0], w.templates)
    zi, ri = np.unravel_index(np.argmax(p), p.shape)
    assert w.z_values[zi] == g["peak_row_z"] and ri == g["peak_col"]
    assert g["peak_power_min"] < p[zi, ri] < g["peak_power_max"]
    # neighbouring rows are lower but still well above the noise (the response is ~|z| bins wide)
    assert p[zi - 1, ri] < p[zi, ri] and p[zi + 1, ri] < p[zi, ri]
    assert p[zi - 1, ri] > 20 and p[zi + 1, ri] > 20
    far = np.ones(p.shape[1], bool); far[19000:21000] = False
    assert g["noise_mean_min"] < p[:, far].mean() < g["noise_mean_max"]


def test_linearity_and_scaling(oracle):
    A1, A2, H = _rand(600, 10), _rand(600, 11), _bank(3, 64, 12)
    al, be = 0.7 - 0.2j, -1.3 + 0.5j
    a1 = oracle.direct(A1, H, want="amp")
    a2 = oracle.direct(A2, H, want="amp")
    a12 = oracle.direct(al * A1 + be * A2, H, want="amp")
    assert np.max(np.abs(a12 - (al * a1 + be * a2))) < 1e-11
    assert np.max(np.abs(oracle.direct(al * A1, H) - abs(al) ** 2 * oracle.direct(A1, H))) < 1e-10


def test_sub_plane_equals_full_plane(oracle):
    A, H = _rand(3000, 13), _bank(5, 64, 14)
    full = oracle.direct(A, H)
    for rows, cols in [((1, 4), (0, 700)), ((0, 5), (2990, 3000)), ((2, 3), (513, 1537)), ((0, 1), (0, 1))]:
        sub = oracle.direct(A, H, rows=rows, cols=cols)
        assert np.array_equal(sub, full[rows[0]:rows[1], cols[0]:cols[1]])


@pytest.mark.parametrize("n_f,m,L,S", [
    (5000, 128, 512, 385), (5000, 128, 512, 384), (5000, 128, 1024, 897), (4097, 64, 512, 449),
    (385 * 3, 128, 512, 385), (100, 128, 512, 385), (9000, 384, 2048, 1665), (3000, 128, 512, 200)])
def test_overlap_save_equals_direct(oracle, n_f, m, L, S):
    # overlap-and-save produces the linear convolution, for any step S <= L-m+1 and any L
    A, H = _rand(n_f, 20), _bank(3, m, 21)
    H /= np.sqrt(np.sum(np.abs(H) ** 2, axis=1, keepdims=True))
    p_dir = oracle.direct(A, H)
    p_ols = oracle.ols(A, H, L, S)
    assert np.max(np.abs(p_ols - p_dir)) < 1e-11 * np.max(p_dir)


def test_overlap_save_on_c1(oracle):
    w = workload.make_config(1)
    p_dir = oracle.direct(w.spectrum[0], w.templates)
    for S in (385, 384):
        p_ols = oracle.ols(w.spectrum[0], w.templates, 512, S)
        assert np.max(np.abs(p_ols - p_dir)) < 1e-12 * np.max(p_dir)


def test_parseval_on_segments(oracle):
    # BASELINE.json north_star: Parseval on segments -- sum |DFT(x_s)|^2 = L sum |x_s|^2
    w = workload.make_config(1)
    L, S, m = 512, 385, 128
    A = w.spectrum[0].astype(np.complex128)
    for s in (0, 7, 170):
        base = s * S - m // 2 + 1
        x = np.array([A[k] if 0 <= k < A.size else 0.0 for k in range(base, base + L)])
        X = oracle.fft(x)
        assert abs(np.sum(np.abs(X) ** 2) - L * np.sum(np.abs(x) ** 2)) < 1e-8 * L * L


def test_edges_are_zero_padded(oracle):
    # reading 6: A[k] = 0 outside [0, n_f); all n_f columns are produced
    n_f, m = 64, 16
    A, H = _rand(n_f, 30), _bank(1, m, 31)
    Apad = np.concatenate([np.zeros(m, complex), A, np.zeros(m, complex)])
    p_pad = oracle.direct(Apad, H)[0, m:m + n_f]
    p = oracle.direct(A, H)[0]
    assert np.max(np.abs(p - p_pad)) < 1e-13


def test_workload_is_seeded_and_shaped():
    a = workload.make_config(1)
    b = workload.make_config(1)
    assert np.array_equal(a.spectrum, b.spectrum) and np.array_equal(a.templates, b.templates)
    assert a.spectrum.dtype == np.complex64 and a.spectrum.shape == (1, 1 << 16)
    assert a.templates.shape == (33, 128) and a.n_z == 33
    assert abs(np.var(a.spectrum.real) - 1) < 0.05 and abs(np.var(a.spectrum.imag) - 1) < 0.05
    c = workload.make_config(5, n_batch=2, n_f=1 << 12)
    assert c.spectrum.shape == (2, 1 << 12) and not np.array_equal(c.spectrum[0], c.spectrum[1])
