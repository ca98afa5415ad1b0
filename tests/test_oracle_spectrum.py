"""Pins of oracle.spectrum ("the FFT output of the observation"; reading 18): eq.(3) written out,
numpy's real FFT, closed forms, and the whitening's defining properties."""
import numpy as np
import pytest


def test_equals_eq3_written_out(oracle):
    rng = np.random.default_rng(1)
    x = rng.standard_normal(32)
    n = np.arange(32)
    ref = np.array([np.sum(x * np.exp(-2j * np.pi * n * k / 32)) for k in range(16)])     # eq.(3)
    assert np.abs(oracle.spectrum(x) - ref).max() < 1e-12


@pytest.mark.parametrize("n_t", [4, 8, 64, 1024, 1 << 15])
def test_equals_numpy_rfft(oracle, n_t):
    x = np.random.default_rng(n_t).standard_normal(n_t)
    ref = np.fft.rfft(x)[: n_t // 2]          # bins 0 .. n_t/2 - 1: the Nyquist bin is not part of the spectrum
    got = oracle.spectrum(x)
    assert got.shape == (n_t // 2,)
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()


def test_closed_forms(oracle):
    n_t = 256
    n = np.arange(n_t)
    # a real sinusoid at an integer bin r with phase phi: X_r = (n_t/2) e^{i phi}, every other bin 0 (sign of eq.(3))
    r, phi = 37, 0.7
    X = oracle.spectrum(np.cos(2 * np.pi * r * n / n_t + phi))
    assert abs(X[r] - 0.5 * n_t * np.exp(1j * phi)) < 1e-10
    assert np.abs(np.delete(X, r)).max() < 1e-10
    # a constant: only the DC bin
    X = oracle.spectrum(np.full(n_t, 3.0))
    assert abs(X[0] - 3.0 * n_t) < 1e-10 and np.abs(X[1:]).max() < 1e-10
    # a unit impulse at sample 1: X_k = exp(-2 pi i k / n_t)
    x = np.zeros(n_t); x[1] = 1.0
    assert np.abs(oracle.spectrum(x) - np.exp(-2j * np.pi * np.arange(n_t // 2) / n_t)).max() < 1e-12


def test_whitening_definition(oracle):
    rng = np.random.default_rng(5)
    n_t, blk = 1 << 14, 300          # a block width that does not divide n_t/2: ragged last block
    # coloured noise: a strong slope in the spectrum that whitening must remove
    x = np.cumsum(rng.standard_normal(n_t)) * 0.05 + rng.standard_normal(n_t)
    X = oracle.spectrum(x)
    A = oracle.spectrum(x, blk)
    n_f = n_t // 2
    assert A[0] == 0
    for b0 in range(0, n_f, blk):
        b1 = min(n_f, b0 + blk)
        p = np.abs(X[b0:b1]) ** 2
        if b0 == 0:
            p[0] = 0.0
        scale = np.sqrt(2.0 / p.mean())
        want = X[b0:b1] * scale
        if b0 == 0:
            want[0] = 0
        assert np.abs(A[b0:b1] - want).max() <= 1e-12 * np.abs(want).max()
        pa = np.abs(A[b0:b1]) ** 2
        assert abs(pa.mean() - 2.0) < 1e-9          # mean power 2 = unit variance in re and in im
    # whitening is invariant under a rescaling of the series
    assert np.abs(oracle.spectrum(7.5 * x, blk) - A).max() < 1e-9


def test_whitened_noise_is_standard_normal_and_keeps_a_tone(oracle):
    """What the correlation expects as input (BASELINE.json configs: "re/im iid N(0,1)"): white Gaussian noise in,
    unit-variance components out; a weak tone stays where it was, at amplitude / sigma in the whitened units."""
    rng = np.random.default_rng(11)
    n_t, blk = 1 << 17, 1024
    n = np.arange(n_t)
    sigma, r, amp = 3.0, 12345, 0.25
    x = sigma * rng.standard_normal(n_t) + amp * np.cos(2 * np.pi * r * n / n_t)
    A = oracle.spectrum(x, blk)
    others = np.delete(A, [0, r])
    assert abs(others.real.std() - 1.0) < 0.01 and abs(others.imag.std() - 1.0) < 0.01
    assert abs(others.real.mean()) < 0.01
    # tone: |X_r| = amp n_t / 2; noise per component sigma sqrt(n_t / 2)  ->  whitened amplitude (amp/sigma) sqrt(n_t/2)
    expect = amp / sigma * np.sqrt(n_t / 2.0)
    assert np.argmax(np.abs(A)) == r and abs(np.abs(A[r]) - expect) < 3.0


def test_zero_block_and_bad_arguments(oracle):
    A = oracle.spectrum(np.zeros(64), 8)
    assert np.all(A == 0)
    with pytest.raises(ValueError):
        oracle.spectrum(np.zeros(48), 8)        # not a power of two
    with pytest.raises(ValueError):
        oracle.spectrum(np.zeros(2), 0)
