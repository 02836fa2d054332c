"""Pins for the oracle's Ising consumer and the statistical
sanity of every generator (8(c)-F).  CPU only.

Pinned against things that are NOT the oracle: brute-force enumeration of the
2^16 states of the 4x4 torus, Kaufman's closed form (tests/exact_ising.py),
the exact values printed in the paper's Table 1, detailed
balance / stationarity evaluated in numpy, and a numpy re-statement of the
half-sweep applied to draws obtained from fill_u32.
"""
import math

import numpy as np
import pytest

import oracle
from conftest import read_golden
from exact_ising import brute_force, energies_all_states, kaufman

G4 = read_golden("ising_L4.txt")
PC = read_golden("paper_constants.txt")


# ---------------------------------------------------------------- exact side
def test_brute_force_matches_stored_values_and_kaufman():
    bf = brute_force(4, 0.3)
    assert abs(bf["Z"] - float(G4["Z"][0])) < 1e-6
    assert abs(bf["e"] - float(G4["e"][0])) < 1e-11
    assert abs(bf["cv"] - float(G4["cv"][0])) < 1e-11
    dos = {int(a): int(b) for a, b in (t.split(":") for t in G4["dos"])}
    assert bf["dos"] == dos and sum(dos.values()) == 1 << 16
    kf = kaufman(4, 0.3)
    assert abs(kf["e"] - bf["e"]) < 1e-10 and abs(kf["cv"] - bf["cv"]) < 1e-9


def test_kaufman_reproduces_the_papers_table1_exact_row():
    # e = 1.106079207 (printed as -E/N), C_V = 0.8616983594, 1024^2, beta = 0.4
    kf = kaufman(1024, 0.4)
    assert abs(-kf["e"] - float(PC["ising_1024_e"][0])) < 5e-9
    assert abs(kf["cv"] - float(PC["ising_1024_cv"][0])) < 5e-9


# ---------------------------------------------------------------- oracle pieces
def test_energy_matches_enumeration_formula():
    E = energies_all_states(4)
    rng = np.random.default_rng(5)
    for idx in rng.integers(0, 1 << 16, size=200):
        sp = (((int(idx) >> np.arange(16)) & 1) * 2 - 1).astype(np.int8)
        assert oracle.ising_energy(sp, 4) == E[idx]
    # all up: every one of the 2 N bonds contributes -1
    assert oracle.ising_energy(np.ones(64 * 64, np.int8), 64) == -2 * 64 * 64
    # perfect checkerboard (antiferro ground state): +2N
    yy, xx = np.mgrid[0:6, 0:6]
    assert oracle.ising_energy((((xx + yy) & 1) * 2 - 1).astype(np.int8).ravel(), 6) == 2 * 36


def test_accept_table_is_metropolis_for_dE_equal_2h():
    for beta in (0.3, 0.4, 0.44068679350977147):
        P = oracle.ising_accept_table(beta)
        for i in range(5):
            h = 2 * i - 4
            assert P[i] == np.float32(math.exp(-2.0 * beta * h))
        assert P[2] == 1.0 and P[0] > 1 and P[1] > 1 and P[4] < P[3] < 1


def test_init_random_bits_come_from_splitmix64():
    L, seed = 8, 2
    sp = oracle.ising_init_random(L, seed)
    assert set(np.unique(sp)) <= {-1, 1}
    for i in (0, 1, 63):
        z = oracle.splitmix64(seed, i >> 6)
        assert sp[i] == (1 if (z >> (i & 63)) & 1 else -1)
    big = oracle.ising_init_random(256, 7)
    assert abs(big.astype(np.int64).sum()) < 5 * 256  # 5 sigma of +-1 coin flips


def _np_half_sweep(sp2, c, draws_q, P):
    """numpy restatement: sites of colour c numbered q = y*(L/2)+xh, x = 2xh+((y+c)&1)."""
    L = sp2.shape[0]
    nn = np.roll(sp2, 1, 0) + np.roll(sp2, -1, 0) + np.roll(sp2, 1, 1) + np.roll(sp2, -1, 1)
    h = sp2.astype(np.int32) * nn
    y, xh = np.divmod(np.arange(L * L // 2), L // 2)
    x = 2 * xh + ((y + c) & 1)
    u = (draws_q >> 8).astype(np.float32) * np.float32(2.0 ** -24)
    flip = u < P[(h[y, x] + 4) // 2]
    out = sp2.copy()
    out[y[flip], x[flip]] *= -1
    return out


@pytest.mark.parametrize("kind", [oracle.PHILOX4X32_10, oracle.XORWOW, oracle.LCG64, oracle.XS1024W])
@pytest.mark.parametrize("L,S", [(4, 8), (8, 32), (16, 32), (12, 72)])
def test_sweep_equals_fill_then_apply(kind, L, S):
    if kind == oracle.XS1024W and S % 32:
        pytest.skip("whole warp instances only")
    beta, nsw = 0.37, 5
    a = oracle.Rng(kind, S, 11)
    b = oracle.Rng(kind, S, 11)
    sp = oracle.ising_init_random(L, 3)
    ref = sp.reshape(L, L).copy()
    tr = a.ising_sweep(sp, L, beta, nsw, trace=True)
    P = oracle.ising_accept_table(beta)
    K = (L * L // 2) // S
    for t in range(nsw):
        for c in (0, 1):
            ref = _np_half_sweep(ref, c, b.fill_u32(K), P)  # stream-major draws[s*K+k] == draws[q]
        assert oracle.ising_energy(ref.ravel().copy(), L) == tr[t]
    assert np.array_equal(ref.ravel(), sp)
    assert a.draws_done == b.draws_done == 2 * nsw * K


def test_sweep_rejects_bad_arguments():
    r = oracle.Rng(oracle.PHILOX4X32_10, 7, 1)
    with pytest.raises(ValueError):
        r.ising_sweep(np.ones(64, np.int8), 8, 0.3, 1)  # 7 does not divide 32
    with pytest.raises(ValueError):
        oracle.Rng(oracle.PHILOX4X32_10, 1, 1).ising_sweep(np.ones(25, np.int8), 5, 0.3, 1)  # odd L


def test_half_sweep_leaves_boltzmann_distribution_stationary():
    """R-E2: exact check on the 4x4 torus.  One colour-c half-sweep with the
    oracle's acceptance table is a product of single-site Metropolis kernels on
    non-interacting sites, so pi P = pi must hold -- up to the float32 rounding of
    the table entries (relative 6e-8, times pi <= 0.042: bound 1e-8; a wrong rule,
    e.g. exp(-beta h) or a wrong sign, misses by ~1e-2).
    Evaluated here in numpy over all 2^16 states x 2^8 flip patterns."""
    L, beta = 4, 0.3
    P = np.minimum(1.0, oracle.ising_accept_table(beta).astype(np.float64))
    E = energies_all_states(L).astype(np.float64)
    pi = np.exp(-beta * E)
    pi /= pi.sum()
    idx = np.arange(1 << 16, dtype=np.int64)
    s = (((idx[:, None] >> np.arange(16)[None, :]) & 1) * 2 - 1).reshape(-1, L, L)
    nn = np.roll(s, 1, 1) + np.roll(s, -1, 1) + np.roll(s, 1, 2) + np.roll(s, -1, 2)
    pacc = P[(s * nn + 4) // 2].reshape(-1, 16)  # flip probability of every site in every state
    for c in (0, 1):
        sites = [y * L + x for y in range(L) for x in range(L) if (x + y) & 1 == c]
        new = np.zeros_like(pi)
        for pat in range(1 << 8):
            w = pi.copy()
            mask = 0
            for b, site in enumerate(sites):
                if (pat >> b) & 1:
                    w *= pacc[:, site]
                    mask |= 1 << site
                else:
                    w *= 1.0 - pacc[:, site]
            np.add.at(new, idx ^ mask, w)
        assert np.max(np.abs(new - pi)) < 1e-8


@pytest.mark.parametrize("kind,S", [(oracle.PHILOX4X32_10, 8), (oracle.XORWOW, 8), (oracle.LCG64, 4)])
def test_monte_carlo_energy_within_3_sigma_of_enumeration(kind, S):
    """north_star: L = 4, beta = 0.3, MC energy agrees with exact enumeration within 3 sigma."""
    L, beta = 4, 0.3
    # (XS1024W needs n_streams % 32 == 0, which cannot divide the 8 sites per colour of L = 4.)
    r = oracle.Rng(kind, S, 1)
    sp = oracle.ising_init_random(L, 2)
    r.ising_sweep(sp, L, beta, 1000)
    n = 200_000
    tr = r.ising_sweep(sp, L, beta, n, trace=True).astype(np.float64) / (L * L)
    # binning error (autocorrelation time at beta=0.3, L=4 is ~1 sweep; bins of 200)
    bins = tr.reshape(-1, 200).mean(axis=1)
    sigma = bins.std(ddof=1) / math.sqrt(len(bins))
    exact = float(G4["e"][0])
    assert abs(tr.mean() - exact) < 3 * sigma, (tr.mean(), exact, sigma)
    assert 5e-4 < sigma < 5e-3
    # specific heat from the same run, loose (5%) -- catches a wrong acceptance table
    cv = beta * beta * tr.var() * (L * L)
    assert abs(cv - float(G4["cv"][0])) < 0.05 * float(G4["cv"][0])


# ---------------------------------------------------------------- 8(c)-F uniformity
@pytest.mark.parametrize("kind,S", [(oracle.LCG64, 1024), (oracle.LCG64_LEAPFROG, 64), (oracle.XORWOW, 1024),
                                    (oracle.PHILOX4X32_10, 1024), (oracle.XS1024W, 1024)])
def test_uniformity_mean_variance_chi_square(kind, S):
    n_total = 1 << 22 if kind != oracle.LCG64_LEAPFROG else 1 << 20
    r = oracle.Rng(kind, S, 1)
    f = r.fill_f32(n_total // S).astype(np.float64)
    n = f.size
    assert abs(f.mean() - 0.5) < 3 * math.sqrt(1 / (12 * n))
    assert abs(f.var() - 1 / 12) < 3 * math.sqrt(1 / (180 * n))
    r2 = oracle.Rng(kind, S, 1)
    u = r2.fill_u32(n_total // S)
    cnt = np.bincount(u >> 24, minlength=256).astype(np.float64)
    chi2 = ((cnt - n / 256) ** 2 / (n / 256)).sum()
    assert 255 - 3 * math.sqrt(510) < chi2 < 255 + 3 * math.sqrt(510), chi2
    # float stream is the integer stream through the fixed map
    assert np.array_equal((u >> 8).astype(np.float32) * np.float32(2.0 ** -24), f.astype(np.float32))
