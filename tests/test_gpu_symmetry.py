"""-m gpu: the FDAS +-z symmetry path behind fdas_plan_set_symmetry.

The exact form P[-z](A) = P[+z](conj A) must give the oracle's plane for a symmetric bank -- including a TRUNCATED
bank (|z| up to 84 with only 64 taps), where the tempting shortcut G_{-z} = conj(G_{+z}) is wrong by 0.15 max(P)
 -- and must switch itself off for a bank that is not symmetric."""
import numpy as np
import pytest

from paper_1711_10855_b200 import workload

from parity import check

pytestmark = pytest.mark.gpu


def _run(torch, binding, n_f, z_max, z_step, m, L, H, spec, sym):
    plan = binding.Plan(n_f, z_max, z_step, m, L, n_batch=spec.shape[0])
    plan.set_symmetry(sym)
    plan.set_templates(H)
    active = plan.symmetry_active
    d_pow = torch.full((spec.shape[0], H.shape[0], n_f), float("nan"), dtype=torch.float32, device="cuda")
    plan.convolve(torch.from_numpy(spec).cuda(), d_pow)
    torch.cuda.synchronize()
    plan.destroy()
    return d_pow.cpu().numpy(), active


@pytest.mark.parametrize("n_f,z_max,z_step,m,L", [
    (30011, 84, 2, 64, 2048),      # truncated responses (window energy 0.76 at |z| = 84): the naive shortcut fails here
    (30011, 84, 4, 256, 2048),
    (50021, 200, 8, 512, 4096),    # C3's template family
    (9000, 0, 1, 128, 4096),       # a single template: the middle row alone
    (40000, 6, 2, 2048, 4096),     # m = L/2
])
def test_symmetric_path_matches_oracle(torch_mod, binding_mod, oracle, n_f, z_max, z_step, m, L):
    H = workload.templates(z_max, z_step, m).astype(np.complex64)
    # workload.templates gives conj-symmetric rows to rounding; make them so bit for bit, as a caller who wants the
    # fast path would (row of -z := conj(row of +z), z = 0 real)
    n_z = H.shape[0]
    for i in range(n_z // 2):
        H[n_z - 1 - i] = np.conj(H[i])
    H[n_z // 2] = H[n_z // 2].real
    spec = workload.noise_spectrum(n_f, 4242 + m, 2)
    p_sym, active = _run(torch_mod, binding_mod, n_f, z_max, z_step, m, L, H, spec, True)
    assert active
    p_gen, active0 = _run(torch_mod, binding_mod, n_f, z_max, z_step, m, L, H, spec, False)
    assert not active0
    for b in range(2):
        ref = oracle.direct(spec[b], H.astype(np.complex128))
        check(p_sym[b], ref, what=f"sym {m}/{L} b{b}")
        check(p_gen[b], ref, what=f"gen {m}/{L} b{b}")
    # the two paths agree to rounding, not bit for bit (different operand order in the -z rows)
    assert np.abs(p_sym.astype(np.float64) - p_gen).max() <= 1e-5 * p_gen.max()


def test_non_symmetric_bank_falls_back(torch_mod, binding_mod, oracle):
    rng = np.random.default_rng(5)
    H = (rng.standard_normal((5, 128)) + 1j * rng.standard_normal((5, 128))).astype(np.complex64)
    spec = workload.noise_spectrum(20000, 7, 1)
    p, active = _run(torch_mod, binding_mod, 20000, 4, 2, 128, 2048, H, spec, True)
    assert not active
    check(p[0], oracle.direct(spec[0], H.astype(np.complex128)), what="fallback")
    # nearly symmetric is not symmetric: one bit off in one tap
    Hs = workload.templates(4, 2, 128).astype(np.complex64)
    for i in range(2):
        Hs[4 - i] = np.conj(Hs[i])
    Hs[2] = Hs[2].real
    Hs[4, 17] = np.complex64(Hs[4, 17].real + np.float32(1e-7) * 1j + 1j * Hs[4, 17].imag)
    _, active = _run(torch_mod, binding_mod, 20000, 4, 2, 128, 2048, Hs, spec, True)
    assert not active
    # segment lengths without the spare tensor-memory block take the general path whatever the bank
    Hs[4, 17] = np.conj(Hs[0, 17])
    _, active = _run(torch_mod, binding_mod, 20000, 4, 2, 128, 1024, Hs, spec, True)
    assert not active
    _, active = _run(torch_mod, binding_mod, 20000, 4, 2, 128, 2048, Hs, spec, True)
    assert active


@pytest.fixture(scope="module")
def torch_mod():
    import torch as _t
    if not _t.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    return _t


@pytest.fixture(scope="module")
def binding_mod():
    from paper_1711_10855_b200 import binding as _b
    _b.lib()
    return _b
