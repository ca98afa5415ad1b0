"""CPU tests of the host-evaluable layout logic of the hot loop's inverse FFT (fft_device.cuh).

`fdas_debug_layout` runs, on the host, the very index functions the kernels use: which spectrum element a
thread register holds, the register permutation of the warp-shuffle exchange, the shared-memory addresses
of the remaining exchange(s) and the indices of the twiddle / modulation / phase tables.  Here the whole
inverse transform is replayed in numpy with ONLY those maps (one array row per thread, numpy's own small
DFTs for the in-register butterflies) and compared with the plain inverse DFT (eq.(3) of PAPER.md line 35
with the sign reversed): any wrong index, sign or transposed digit fails.  No GPU is needed.
"""
import numpy as np
import pytest

from paper_1711_10855_b200 import binding as B

LS = [512, 1024, 2048, 4096, 8192]


def geom(L):
    names = ["P", "E", "NT", "Ra", "Rb", "Gs", "NA", "NB", "BUF", "R0", "R1"]
    return {n: B.debug_layout(L, B.LAYOUT_GEOMETRY, 0, a) for a, n in enumerate(names)}


def idft(x):
    n = x.shape[-1]
    k = np.arange(n)
    return x @ np.exp(2j * np.pi * np.outer(k, k) / n)


def wl(L, idx):
    """conj(w_L^idx) = exp(+2 pi i idx / L): every table entry of the inverse is applied conjugated."""
    return np.exp(2j * np.pi * np.asarray(idx) / L)


def replay_inverse(L, Y):
    """Inverse DFT of Y (natural frequency order) using only the library's index maps."""
    g = geom(L)
    P, E, NT, Ra, Rb, Gs, NA, NB, R0, R1 = (g[k] for k in ("P", "E", "NT", "Ra", "Rb", "Gs", "NA", "NB", "R0", "R1"))
    q = lambda what, t, a=0, b=0: B.debug_layout(L, what, t, a, b)
    # loop entry: register i*Ra + k of thread t holds Y[freq] times the modulation folded into G
    v = np.empty((NT, E), complex)
    for t in range(NT):
        for i in range(NB):
            for k in range(Ra):
                v[t, i * Ra + k] = Y[q(B.LAYOUT_FREQ, t, i, k)] * wl(L, q(B.LAYOUT_GMOD, t, k))
    v = idft(v.reshape(NT, NB, Ra)).reshape(NT, E)                      # pass P-1
    w = np.full_like(v, np.nan)
    for t in range(NT):                                                  # shuffle exchange, Gs rounds
        grp, lane = divmod(t, Gs)
        for r in range(Gs):
            src = grp * Gs + ((lane + Gs - r) % Gs)
            for b in range(NB * NA):
                w[t, q(B.LAYOUT_SHFL_DST, t, r, b)] = v[src, q(B.LAYOUT_SHFL_SRC, t, r, b)]
    assert not np.isnan(w).any(), "shuffle does not fill every register"
    for t in range(NT):                                                  # multipliers of pass P-2
        for j in range(NA):
            for tau in range(1, Rb):
                w[t, j * Rb + tau] *= wl(L, q(B.LAYOUT_TWA, t, j, tau))
    w = idft(w.reshape(NT, NA, Rb)).reshape(NT, E)                      # pass P-2
    buf = np.full(g["BUF"], np.nan, complex)
    for t in range(NT):
        for j in range(NA):
            for kap in range(Rb):
                a = q(B.LAYOUT_WRITE_A, t, j, kap)
                assert np.isnan(buf[a]), "two registers write the same shared-memory element"
                buf[a] = w[t, j * Rb + kap]
    u = np.empty((NT, E), complex)
    if P == 3:
        for t in range(NT):
            for k in range(R0):
                u[t, k] = buf[q(B.LAYOUT_READ_A, t, 0, k)]
    else:
        x = np.empty((NT, E), complex)
        for t in range(NT):
            for b in range(E // R1):
                for k in range(R1):
                    x[t, b * R1 + k] = buf[q(B.LAYOUT_READ_A, t, b, k)] * wl(L, q(B.LAYOUT_TW_MID, t, k))
        x = idft(x.reshape(NT, E // R1, R1)).reshape(NT, E)             # pass 1
        bufb = np.full(g["BUF"], np.nan, complex)
        for t in range(NT):
            for b in range(E // R1):
                for n in range(R1):
                    a = q(B.LAYOUT_WRITE_B, t, b, n)
                    assert np.isnan(bufb[a])
                    bufb[a] = x[t, b * R1 + n]
        for t in range(NT):
            for k in range(R0):
                u[t, k] = bufb[q(B.LAYOUT_READ_B, t, k)]
    assert not np.isnan(u).any(), "an exchange read hits an element nobody wrote"
    tt = np.arange(NT)[:, None]
    u = idft(u * wl(L, np.arange(R0)[None, :] * tt))                     # pass 0: multipliers w_L^{d t}
    fix = np.array([np.exp(-2j * np.pi * q(B.LAYOUT_FIX, t) / L) for t in range(NT)])   # w_L^idx
    return u, fix


@pytest.mark.parametrize("L", LS)
def test_inverse_replayed_with_library_maps_equals_idft(L):
    rng = np.random.default_rng(L)
    Y = rng.standard_normal(L) + 1j * rng.standard_normal(L)
    ref = np.fft.ifft(Y) * L
    u, fix = replay_inverse(L, Y)
    NT = u.shape[0]
    out = u.T.reshape(L)                      # register d of thread t is output d*NT + t
    # the hot loop needs only |y|^2: exact up to a unit phase per thread
    assert np.max(np.abs(np.abs(out) ** 2 - np.abs(ref) ** 2)) <= 1e-9 * np.max(np.abs(ref)) ** 2
    # and the phase left on thread t's outputs is the one fdas_debug_fft removes
    out_fixed = (u * fix[:, None]).T.reshape(L)
    assert np.max(np.abs(out_fixed - ref)) <= 1e-9 * np.max(np.abs(ref))
    assert NT * u.shape[1] == L


@pytest.mark.parametrize("L", LS)
def test_loop_entry_layout_is_a_bijection(L):
    g = geom(L)
    seen = np.zeros(L, int)
    for t in range(g["NT"]):
        for i in range(g["NB"]):
            for k in range(g["Ra"]):
                seen[B.debug_layout(L, B.LAYOUT_FREQ, t, i, k)] += 1
    assert np.all(seen == 1)


@pytest.mark.parametrize("L", LS)
def test_shuffle_register_maps_are_permutations(L):
    g = geom(L)
    src, dst = [], []
    for r in range(g["Gs"]):
        for b in range(g["NA"] * g["NB"]):
            src.append(B.debug_layout(L, B.LAYOUT_SHFL_SRC, 0, r, b))
            dst.append(B.debug_layout(L, B.LAYOUT_SHFL_DST, 0, r, b))
    assert sorted(src) == list(range(g["E"])) and sorted(dst) == list(range(g["E"]))


def _bank_pairs_distinct(addrs):
    """64-bit shared-memory accesses: a half-warp (16 lanes) is conflict free iff the 16 element
    addresses (8 bytes each) are distinct modulo 16 (32 banks of 4 bytes)."""
    return len({a % 16 for a in addrs}) == len(addrs)


@pytest.mark.parametrize("L", [512, 2048, 4096])
def test_exchange_is_bank_conflict_free(L):
    """The shared-memory exchange of the hot loop: every 64-bit store and load of every half-warp hits
    16 distinct bank pairs (L = 1024 and 8192, whose shuffle groups have 4 lanes, keep a 2-way conflict
    on the store side: DESIGN.md section 6)."""
    g = geom(L)
    for h in range(g["NT"] // 16):
        lanes = range(16 * h, 16 * h + 16)
        for j in range(g["NA"]):
            for kap in range(g["Rb"]):
                assert _bank_pairs_distinct([B.debug_layout(L, B.LAYOUT_WRITE_A, t, j, kap) for t in lanes]), (h, j, kap)
        for k in range(g["R0"]):
            assert _bank_pairs_distinct([B.debug_layout(L, B.LAYOUT_READ_A, t, 0, k) for t in lanes]), (h, k)


@pytest.mark.parametrize("L", [1024, 8192])
def test_exchange_conflicts_bounded_for_small_groups(L):
    g = geom(L)
    R = g["R0"] if g["P"] == 3 else g["R1"]
    worst = 1
    for h in range(g["NT"] // 16):
        lanes = range(16 * h, 16 * h + 16)
        for j in range(g["NA"]):
            for kap in range(g["Rb"]):
                banks = [B.debug_layout(L, B.LAYOUT_WRITE_A, t, j, kap) % 16 for t in lanes]
                worst = max(worst, max(banks.count(b) for b in set(banks)))
        for b in range(g["E"] // R):
            for k in range(R):
                assert _bank_pairs_distinct([B.debug_layout(L, B.LAYOUT_READ_A, t, b, k) for t in lanes])
    assert worst <= 2


def test_layout_query_rejects_bad_arguments():
    assert B.debug_layout(300, B.LAYOUT_GEOMETRY, 0, 0) == -1      # unsupported segment length
    assert B.debug_layout(4096, B.LAYOUT_FREQ, 256, 0, 0) == -1    # thread out of range
    assert B.debug_layout(4096, 99, 0, 0, 0) == -1                 # unknown selector
    assert B.debug_layout(4096, B.LAYOUT_WRITE_B, 0, 0, 0) == -1   # three-pass plan has no second exchange


@pytest.mark.parametrize("L", [512, 1024, 2048, 4096, 8192])
def test_inverse_exchanges_are_bank_conflict_free(L):
    """Every 64-bit shared-memory access of the hot loop's exchanges: the 16 threads of a half-warp fall on 16
    distinct bank pairs (or on the same address).  Round 2 found the first-exchange writes of the NA = 2 plans
    (L = 1024, 8192) two-way conflicted: 28 % of their shared-memory wavefronts (profiles/r2_all_configs.md)."""
    g = lambda a: B.debug_layout(L, B.LAYOUT_GEOMETRY, 0, a)
    P, E, NT, Ra, Rb, Gs, NA, NB, BUF, R0, R1 = [g(i) for i in range(11)]
    accesses = [(B.LAYOUT_WRITE_A, NA, Rb), (B.LAYOUT_READ_A, E // (R0 if P == 3 else R1), R0 if P == 3 else R1)]
    if P == 4:
        accesses += [(B.LAYOUT_WRITE_B, E // R1, R1), (B.LAYOUT_READ_B, R0, 1)]
    for what, n1, n2 in accesses:
        for a in range(n1):
            for b in range(n2):
                addr = [B.debug_layout(L, what, t, a, b) for t in range(NT)]
                assert min(addr) >= 0 and max(addr) < BUF
                for h in range(0, NT, 16):
                    distinct = set(addr[h:h + 16])
                    assert len({x % 16 for x in distinct}) == len(distinct), (L, what, a, b, h)
