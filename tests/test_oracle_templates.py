"""Pins for the oracle's template generator ("predicted, normalized, Fourier
response"; formula derived in SURVEY.md section 8(c)).  CPU only.

Independent references used: scipy.special.fresnel, mpmath quadrature of the defining integral, the DFT
of a sampled chirp (pins the sign of z and "centred on the mean frequency"), closed forms and
symmetries, and the scipy-based generator in paper_1711_10855_b200.workload (a second implementation).
"""
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "template_pins.txt")


def _golden():
    vals, energies = [], []
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        if f[0] == "energy":
            energies.append((int(f[1]), int(f[2]), float(f[3])))
        else:
            vals.append((int(f[0]), int(f[1]), complex(float(f[2]), float(f[3]))))
    return vals, energies


def test_fresnel_against_scipy(oracle):
    from scipy.special import fresnel
    xs = np.concatenate([np.linspace(-4, 4, 401), np.linspace(4, 60, 300),
                         [1.4999, 1.5, 1.5001, 99.7, 257.25, 513.5, 724.0, -724.0, 0.0]])
    for x in xs:
        C, S = oracle.fresnel(x)
        s_ref, c_ref = fresnel(x)
        assert abs(C - c_ref) < 5e-13 and abs(S - s_ref) < 5e-13, x


def test_fresnel_small_argument_series_and_limits(oracle):
    # C(x) ~ x, S(x) ~ pi x^3 / 6 as x -> 0; C, S -> 1/2 as x -> inf
    C, S = oracle.fresnel(1e-3)
    assert abs(C - 1e-3) < 1e-15 and abs(S - np.pi * 1e-9 / 6) < 1e-20
    C, S = oracle.fresnel(1e4)
    assert abs(C - 0.5) < 1e-4 and abs(S - 0.5) < 1e-4


def test_response_against_mpmath_quadrature(oracle):
    import mpmath as mp
    mp.mp.dps = 30
    for z, q in [(20, -10), (20, -9), (20, -15), (20, 27), (-20, 10), (4, -2), (4, 3), (200, -100),
                 (200, -63), (-84, 42), (-84, 5), (2, -1), (2, 30.5), (0, 0.3), (0, 0), (7, -3.5)]:
        f = lambda u: mp.exp(1j * mp.pi * (2 * q * u + z * u * u))
        ref = complex(mp.quad(f, mp.linspace(0, 1, 65)))
        assert abs(oracle.response(q, z) - ref) < 1e-12, (z, q)


def test_golden_values_from_survey(oracle):
    vals, _ = _golden()
    for z, d, ref in vals:
        got = oracle.response(d - 0.5 * z, z)
        assert abs(got - ref) < 2e-12, (z, d, got, ref)


def test_window_energies_from_survey(oracle):
    _, energies = _golden()
    for m, z, e_ref in energies:
        d = np.arange(m) - m // 2
        e = sum(abs(oracle.response(dd - 0.5 * z, z)) ** 2 for dd in d)
        assert abs(e - e_ref) < 1.5e-6, (m, z, e)


def test_sampled_chirp_pins_sign_of_z_and_centering(oracle):
    # x_j = exp(2 pi i (r_s j/N + z j^2 / (2 N^2))): frequency RISES by z bins over the record.
    # Its DFT/N at bin r is I(r_s - r, z) up to O(1/N).  The mean frequency is r_s + z/2, and the
    # template H_z(d) = I(d - z/2, z) measured from it must be even in d.
    N, r_s, z = 4096, 1000.3, 20.0
    j = np.arange(N)
    x = np.exp(2j * np.pi * (r_s * j / N + z * j * j / (2.0 * N * N)))
    X = np.fft.fft(x) / N
    bins = np.arange(900, 1150)
    ref = np.array([oracle.response(r_s - r, z) for r in bins])
    assert np.max(np.abs(X[bins] - ref)) < 5e-4
    # the wrong sign of z (or of q) fails by O(0.1)
    bad = np.array([oracle.response(r_s - r, -z) for r in bins])
    assert np.max(np.abs(X[bins] - bad)) > 0.05
    # power is concentrated between r_s and r_s + z (drift upward), centred on r_s + z/2
    p = np.abs(X) ** 2
    centroid = np.sum(np.arange(N) * p) / np.sum(p)
    assert abs(centroid - (r_s + z / 2)) < 0.5


def test_z0_template_is_the_pure_tone_response(oracle):
    # I(q,0) = e^{i pi q} sinc(q); at integer offsets it is delta_{d,0}
    for d in range(-8, 9):
        v = oracle.response(d, 0)
        assert abs(v - (1.0 if d == 0 else 0.0)) < 1e-15
    for q in (0.25, -0.5, 3.3):
        ref = np.exp(1j * np.pi * q) * np.sinc(q)
        assert abs(oracle.response(q, 0) - ref) < 1e-14
    T = oracle.templates(4, 2, 16)
    row0 = T[2]
    e = np.zeros(16, complex); e[8] = 1.0
    assert np.max(np.abs(row0 - e)) < 1e-14


def test_symmetries(oracle):
    for z in (2, 20, 84, 200):
        d = np.arange(-64, 64)
        Hp = np.array([oracle.response(dd - 0.5 * z, z) for dd in d])
        Hm = np.array([oracle.response(dd + 0.5 * z, -z) for dd in d])
        Hr = np.array([oracle.response(-dd - 0.5 * z, z) for dd in d])
        assert np.max(np.abs(Hp - Hr)) < 1e-12          # H_z(-d) = H_z(d)
        assert np.max(np.abs(Hm - np.conj(Hp))) < 1e-12  # H_{-z}(d) = conj H_z(d)


def test_total_energy_and_plateau(oracle):
    # Parseval: sum over all d of |H_z(d)|^2 = 1; inside |d| < |z|/2 the power is ~ 1/|z|
    z = 40
    d = np.arange(-4000, 4000)
    H = np.array([oracle.response(dd - 0.5 * z, z) for dd in d])
    assert abs(np.sum(np.abs(H) ** 2) - 1.0) < 2e-4
    inner = np.abs(H[(d > -10) & (d < 10)]) ** 2
    assert abs(np.mean(inner) * z - 1.0) < 0.15


def test_bank_layout_and_normalisation(oracle):
    z_max, z_step, m = 32, 2, 128
    T = oracle.templates(z_max, z_step, m)
    assert T.shape == (33, 128)
    assert np.max(np.abs(np.sum(np.abs(T) ** 2, axis=1) - 1.0)) < 1e-13
    # row i <-> z = -z_max + i*z_step; tap j <-> d = j - m/2
    i, j = 26, 70   # z = +20, d = +6
    raw = np.array([oracle.response(dd - 10.0, 20.0) for dd in np.arange(m) - m // 2])
    assert abs(T[i, j] - raw[j] / np.sqrt(np.sum(np.abs(raw) ** 2))) < 1e-14
    # -z row is the element-wise conjugate of the +z row on the (asymmetric) window
    assert np.max(np.abs(T[6] - np.conj(T[26]))) < 1e-12


@pytest.mark.parametrize("z_max,z_step,m", [(32, 2, 128), (84, 2, 256), (200, 2, 512), (84, 2, 64),
                                            (84, 2, 1024), (9, 3, 384)])
def test_oracle_bank_equals_workload_bank(oracle, z_max, z_step, m):
    # two implementations (C + own Fresnel vs numpy + scipy.special.fresnel) of the same formula
    from paper_1711_10855_b200 import workload
    a = oracle.templates(z_max, z_step, m)
    b = workload.templates(z_max, z_step, m)
    assert a.shape == b.shape
    assert np.max(np.abs(a - b)) < 1e-11


def test_templates_reject_bad_arguments(oracle):
    with pytest.raises(ValueError):
        oracle.templates(5, 2, 16)
    with pytest.raises(ValueError):
        oracle.templates(4, 2, 15)
