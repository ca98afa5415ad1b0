"""Pins for the oracle's transforms (eq.(3)): brute force, a library FFT, Parseval,
closed forms.  CPU only."""
import numpy as np
import pytest


def _rand(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(n) + 1j * rng.standard_normal(n)


@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64])
def test_fft_equals_bruteforce_dft(oracle, n):
    x = _rand(n, n)
    for sign in (-1, +1):
        assert np.max(np.abs(oracle.fft(x, sign) - oracle.dft(x, sign))) < 1e-12 * n


def test_dft_is_eq3_written_out(oracle):
    # eq.(3) with its own loop in Python, tiny N: X_m = sum_n x_n exp(-i 2 pi n m / N)
    n = 8
    x = _rand(n, 99)
    X = np.array([sum(x[k] * np.exp(-2j * np.pi * k * m_ / n) for k in range(n)) for m_ in range(n)])
    assert np.max(np.abs(oracle.dft(x) - X)) < 1e-13


@pytest.mark.parametrize("n", [512, 4096])
def test_fft_matches_library_fft(oracle, n):
    x = _rand(n, 7)
    assert np.max(np.abs(oracle.fft(x, -1) - np.fft.fft(x))) < 1e-10
    assert np.max(np.abs(oracle.fft(x, +1) - np.fft.ifft(x) * n)) < 1e-10


def test_dft_512_at_a_few_bins(oracle):
    n = 512
    x = _rand(n, 5)
    X = oracle.fft(x)
    for m_ in (0, 1, 77, 255, 256, 511):
        ref = np.sum(x * np.exp(-2j * np.pi * np.arange(n) * m_ / n))
        assert abs(X[m_] - ref) < 1e-10


@pytest.mark.parametrize("n", [64, 512, 2048])
def test_parseval(oracle, n):
    x = _rand(n, 3)
    X = oracle.fft(x)
    assert abs(np.sum(np.abs(X) ** 2) - n * np.sum(np.abs(x) ** 2)) < 1e-9 * n * n


def test_closed_forms(oracle):
    n = 64
    # delta at n0 -> pure phase ramp; constant -> N delta_0; tone at bin 5 -> N delta_5
    d = np.zeros(n, complex); d[3] = 1.0
    assert np.max(np.abs(oracle.fft(d) - np.exp(-2j * np.pi * 3 * np.arange(n) / n))) < 1e-13
    c = np.ones(n, complex)
    e0 = np.zeros(n, complex); e0[0] = n
    assert np.max(np.abs(oracle.fft(c) - e0)) < 1e-12
    t = np.exp(2j * np.pi * 5 * np.arange(n) / n)
    e5 = np.zeros(n, complex); e5[5] = n
    assert np.max(np.abs(oracle.fft(t) - e5)) < 1e-11


def test_inverse_roundtrip_and_sign(oracle):
    n = 256
    x = _rand(n, 11)
    assert np.max(np.abs(oracle.fft(oracle.fft(x, -1), +1) / n - x)) < 1e-12
    # a wrong sign would map bin 5 to bin n-5
    t = np.exp(2j * np.pi * 5 * np.arange(n) / n)
    assert np.argmax(np.abs(oracle.fft(t, -1))) == 5
    assert np.argmax(np.abs(oracle.fft(t, +1))) == n - 5


def test_fft_rejects_non_power_of_two(oracle):
    with pytest.raises(ValueError):
        oracle.fft(np.ones(12, complex))
