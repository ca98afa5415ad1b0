"""Seeded synthetic FDAS workloads (inputs only -- none of the method's arithmetic lives here).

The library's inputs are a complex64 spectrum and a bank of complex templates; both are *data* to
`fdas_convolve`.  This module makes them, seeded, in the shape of the five BASELINE.json configs, and
serves the CUDA path (tests, bench.py) and the oracle (tests) alike.  It imports neither of them.

Recipe (restated in DESIGN.md "Input recipe"):
  rng   = numpy Generator(PCG64(171110855 + 1000*c + 100*pair + b)), c = config 1..5, pair = index of
          the (m, L) pair in the C4 sweep (0 elsewhere), b = batch index (0 unless C5)
  noise = rng.standard_normal((N_f, 2)) -> A = w[:,0] + i w[:,1]             (sigma = 1 per component)
  then per injected signal, in this order of draws: r_c, z (if drawn), k, phi
  A    += k e^{i phi} I((r_c - z/2) - bin, z) at ALL bins, in double; one cast to complex64.
  templates: h_z[j] = H_z(j - m/2)/||H_z||, H_z(d) = I(d - z/2, z), row i <-> z = -z_max + i*z_step.

I(q,z) = int_0^1 exp(i pi (2 q u + z u^2)) du is the Fourier response of a unit signal drifting by z
bins ("predicted ... Fourier response", Ransom et al. 2002); it is evaluated here with
scipy.special.fresnel, independently of the oracle's own C implementation (tests compare the two).
"""
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 171110855


def response(q, z):
    """I(q,z) for array q and scalar z (closed form; see module docstring)."""
    from scipy.special import fresnel  # returns (S, C)

    q = np.asarray(q, dtype=np.float64)
    z = float(z)
    if z == 0.0:
        return np.exp(1j * np.pi * q) * np.sinc(q)
    if z < 0.0:
        return np.conj(response(-q, -z))
    rt = np.sqrt(2.0 / z)
    sy, cy = fresnel(q * rt)
    sz, cz = fresnel((q + z) * rt)
    return np.exp(-1j * np.pi * q * q / z) / np.sqrt(2.0 * z) * ((cz - cy) + 1j * (sz - sy))


def templates(z_max: int, z_step: int, m: int) -> np.ndarray:
    """Unit-normalised template bank, complex128 [n_z][m]."""
    if z_step < 1 or z_max < 0 or z_max % z_step or m < 2 or m % 2:
        raise ValueError("bad template grid")
    zs = np.arange(-z_max, z_max + 1, z_step)
    d = np.arange(m) - m // 2
    out = np.empty((zs.size, m), dtype=np.complex128)
    for i, z in enumerate(zs):
        h = response(d - 0.5 * z, z)
        out[i] = h / np.sqrt(np.sum(np.abs(h) ** 2))
    return out


@dataclass
class Signal:
    r_c: float
    z: float
    k: float
    phi: float


@dataclass
class Workload:
    """One (N_f, z grid, m, L) problem with its seeded inputs."""
    name: str
    n_f: int
    z_max: int
    z_step: int
    m: int
    seg_len: int
    n_batch: int
    spectrum: Optional[np.ndarray]        # complex64 [n_batch][n_f]
    templates: np.ndarray                 # complex64 [n_z][m]  (what fdas_set_templates receives)
    signals: List[List[Signal]] = field(default_factory=list)  # per batch item

    @property
    def n_z(self) -> int:
        return 2 * self.z_max // self.z_step + 1

    @property
    def z_values(self) -> np.ndarray:
        return np.arange(-self.z_max, self.z_max + 1, self.z_step)

    @property
    def points(self) -> int:
        return self.n_batch * self.n_z * self.n_f


def _inject(A: np.ndarray, sig: Signal) -> None:
    bins = np.arange(A.size, dtype=np.float64)
    A += sig.k * np.exp(1j * sig.phi) * response((sig.r_c - 0.5 * sig.z) - bins, sig.z)


def make_spectrum(n_f: int, seed: int, draw_signals) -> Tuple[np.ndarray, List[Signal]]:
    """noise + signals -> complex64 [n_f].  draw_signals(rng) -> list of Signal (drawn after the noise)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    w = rng.standard_normal((n_f, 2))
    A = w[:, 0] + 1j * w[:, 1]
    sigs = draw_signals(rng)
    for s in sigs:
        _inject(A, s)
    return A.astype(np.complex64), sigs


# (n_f, z_max, z_step, m, L) of BASELINE.json configs 1..3 and 5; C4 is a sweep over (m, L).
_SHAPES = {
    1: (1 << 16, 32, 2, 128, 512),
    2: (1 << 20, 84, 2, 256, 2048),
    3: (1 << 22, 200, 2, 512, 4096),
    5: (1 << 20, 84, 2, 256, 2048),
}
C4_PAIRS = [(64, 512), (128, 1024), (256, 2048), (512, 4096), (1024, 8192)]
C4_NF = 1 << 21


def _drawer(c: int, n_f: int, m: int, z_max: int, z_step: int):
    grid = np.arange(-z_max, z_max + 1, z_step)

    def u_rc(rng):
        return float(rng.uniform(4 * m, n_f - 4 * m))

    def draw(rng):
        if c == 1:
            return [Signal(20000.3, 20.0, 8.0, float(rng.uniform(0, 2 * np.pi)))]
        if c == 2:
            out = []
            for z in (-60.0, 0.0, 44.0):
                r = u_rc(rng); k = float(rng.uniform(6, 10)); ph = float(rng.uniform(0, 2 * np.pi))
                out.append(Signal(r, z, k, ph))
            return out
        if c in (3, 5):
            out = []
            for _ in range(5 if c == 3 else 1):
                r = u_rc(rng); z = float(rng.choice(grid)); k = float(rng.uniform(6, 10))
                ph = float(rng.uniform(0, 2 * np.pi))
                out.append(Signal(r, z, k, ph))
            return out
        return []  # C4: noise only

    return draw


def make_config(c: int, pair: int = 0, n_batch: Optional[int] = None, n_f: Optional[int] = None,
                with_spectrum: bool = True) -> Workload:
    """BASELINE.json config c (1..5).  `pair` selects the (m, L) pair of the C4 sweep.

    n_batch / n_f override the config's own (used for reduced-size variants in tests); the seeds do
    not change, so a reduced variant is a prefix-independent draw of the same recipe.
    """
    if c == 4:
        m, L = C4_PAIRS[pair]
        nf, z_max, z_step = C4_NF, 84, 2
        name = f"C4[m={m},L={L}]"
    elif c in _SHAPES:
        nf, z_max, z_step, m, L = _SHAPES[c]
        name = f"C{c}"
    else:
        raise ValueError("config must be 1..5")
    if n_f is not None:
        nf = int(n_f)
    nb = (64 if c == 5 else 1) if n_batch is None else int(n_batch)
    H = templates(z_max, z_step, m).astype(np.complex64)
    spec, sigs = None, []
    if with_spectrum:
        spec = np.empty((nb, nf), dtype=np.complex64)
        draw = _drawer(c, nf, m, z_max, z_step)
        for b in range(nb):
            spec[b], s = make_spectrum(nf, SEED_BASE + 1000 * c + 100 * pair + b, draw)
            sigs.append(s)
    return Workload(name, nf, z_max, z_step, m, L, nb, spec, H, sigs)


def config_shape(c: int, pair: int = 0) -> dict:
    """Sizes of BASELINE.json config c without generating any data."""
    wl = make_config(c, pair=pair, n_f=None, with_spectrum=False)
    return {"name": wl.name, "n_f": wl.n_f, "n_z": wl.n_z, "m": wl.m, "seg_len": wl.seg_len, "n_batch": wl.n_batch}


def noise_spectrum(n_f: int, seed: int, n_batch: int = 1) -> np.ndarray:
    """Plain N(0,1)+iN(0,1) complex64 [n_batch][n_f] (bench.py's bulk input; no signals)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = np.empty((n_batch, n_f), dtype=np.complex64)
    for b in range(n_batch):
        w = rng.standard_normal((n_f, 2), dtype=np.float32)
        out[b] = w[:, 0] + 1j * w[:, 1]
    return out
