"""Pins for the oracle's double-checkerboard multi-hit sweep (the paper's own consumer,
PAPER.md:56, :58; reading R-E9 in DESIGN.md).  CPU only.

Pinned against things that are not the oracle: a site-by-site Python brute force that goes
the OTHER way round (scans sites, derives tile / thread / stream / draw number from the
coordinates, decides with the full-lattice energy difference), exact flip counting at
beta = 0, the 2^16-state enumeration of the 4x4 torus (stationarity of every sub-step and
the Monte Carlo energy within 3 sigma), and Kaufman's exact e for a larger lattice."""
import math

import numpy as np
import pytest

import oracle
from conftest import read_golden
from exact_ising import energies_all_states, kaufman

G4 = read_golden("ising_L4.txt")


def _brute_force_sweeps(sp, L, beta, nsw, T, k, draws):
    """draws[s, j] = draw j of stream s (stream-major fill).  Every (sweep, C, hit, c) sub-step scans ALL sites,
    keeps those whose tile has coarse colour C and whose own colour is c, and flips with the Metropolis rule
    written with the energy difference of the whole lattice."""
    def energy(a):
        return -int((a * np.roll(a, -1, 0)).sum() + (a * np.roll(a, -1, 1)).sum())

    a = sp.reshape(L, L).astype(np.int64).copy()
    nth = L // T // 2
    for sw in range(nsw):
        for C in (0, 1):
            for hit in range(k):
                for c in (0, 1):
                    old = a.copy()                                   # sites of one sub-step do not interact
                    for y in range(L):
                        for x in range(L):
                            tx, ty = x // T, y // T
                            if (tx + ty) & 1 != C or (x + y) & 1 != c:
                                continue
                            p = ty * nth + tx // 2                   # number of the tile among those of colour C
                            t = (y % T) * (T // 2) + (x % T) // 2    # thread = horizontal domino of the tile
                            s = p * (T * T // 2) + t
                            j = ((2 * sw + C) * k + hit) * 2 + c
                            trial = old.copy()
                            trial[y, x] = -trial[y, x]
                            dE = energy(trial) - energy(old)
                            u = np.float32(int(draws[s, j]) >> 8) * np.float32(2.0 ** -24)
                            if u < np.float32(math.exp(-beta * dE)):   # min(1, e^{-beta dE}); u < 1 always
                                a[y, x] = -old[y, x]
    return a.astype(np.int8).ravel()


@pytest.mark.parametrize("kind", [oracle.PHILOX4X32_10, oracle.XORWOW])
@pytest.mark.parametrize("L,T,k", [(4, 2, 1), (8, 2, 3), (8, 4, 2), (12, 2, 1), (12, 6, 2)])
def test_multihit_equals_site_by_site_brute_force(kind, L, T, k):
    beta, nsw, S = 0.41, 2, L * L // 4
    sp = oracle.ising_init_random(L, 5)
    ref0 = sp.copy()
    r = oracle.Rng(kind, S, 3)
    tr = r.ising_sweep_multihit(sp, L, beta, nsw, T, k, trace=True)
    assert r.draws_done == 4 * k * nsw
    draws = oracle.Rng(kind, S, 3).fill_u32(4 * k * nsw).reshape(S, -1)
    ref = _brute_force_sweeps(ref0, L, beta, nsw, T, k, draws)
    assert np.array_equal(sp, ref)
    assert tr[-1] == oracle.ising_energy(ref, L)


@pytest.mark.parametrize("L,T,k", [(8, 2, 1), (8, 4, 3), (16, 4, 2), (24, 6, 5), (32, 8, 4), (64, 16, 1)])
def test_every_site_is_hit_exactly_k_times_per_sweep(L, T, k):
    # beta = 0: every proposal is accepted, so a sweep multiplies every spin by (-1)^k
    sp = oracle.ising_init_random(L, 9)
    ref = sp.copy()
    r = oracle.Rng(oracle.PHILOX4X32_10, L * L // 4, 1)
    r.ising_sweep_multihit(sp, L, 0.0, 3, T, k)
    assert np.array_equal(sp, ref * (-1) ** (3 * k))
    assert r.draws_done == 12 * k


def test_rejects_bad_geometry():
    sp = np.ones(64, np.int8)
    ok = oracle.Rng(oracle.PHILOX4X32_10, 16, 1)
    for T, k in ((3, 1), (8, 1), (2, 0), (1, 1)):      # odd tile; L/T odd; no hits; tile too small
        with pytest.raises(ValueError):
            ok.ising_sweep_multihit(sp, 8, 0.3, 1, T, k)
    with pytest.raises(ValueError):
        oracle.Rng(oracle.PHILOX4X32_10, 32, 1).ising_sweep_multihit(sp, 8, 0.3, 1, 2, 1)  # needs L*L/4 streams


def test_every_sub_step_leaves_the_boltzmann_distribution_stationary():
    """4x4 torus, T = 2: a sub-step (C, c) updates the 4 sites of fine colour c in the 2 tiles of coarse colour C.
    pi P = pi over all 2^16 states x 2^4 flip patterns, for each of the four sub-step types."""
    L, T, beta = 4, 2, 0.3
    P = np.minimum(1.0, oracle.ising_accept_table(beta).astype(np.float64))
    E = energies_all_states(L).astype(np.float64)
    pi = np.exp(-beta * E)
    pi /= pi.sum()
    idx = np.arange(1 << 16, dtype=np.int64)
    s = (((idx[:, None] >> np.arange(16)[None, :]) & 1) * 2 - 1).reshape(-1, L, L)
    nn = np.roll(s, 1, 1) + np.roll(s, -1, 1) + np.roll(s, 1, 2) + np.roll(s, -1, 2)
    pacc = P[(s * nn + 4) // 2].reshape(-1, 16)
    for C in (0, 1):
        for c in (0, 1):
            sites = [y * L + x for y in range(L) for x in range(L)
                     if ((x // T + y // T) & 1) == C and ((x + y) & 1) == c]
            assert len(sites) == 4
            new = np.zeros_like(pi)
            for pat in range(1 << 4):
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


@pytest.mark.parametrize("kind,k", [(oracle.PHILOX4X32_10, 1), (oracle.XORWOW, 3)])
def test_monte_carlo_energy_within_3_sigma_of_enumeration(kind, k):
    L, T, beta = 4, 2, 0.3
    r = oracle.Rng(kind, L * L // 4, 1)
    sp = oracle.ising_init_random(L, 2)
    r.ising_sweep_multihit(sp, L, beta, 1000, T, k)
    n = 100_000
    tr = r.ising_sweep_multihit(sp, L, beta, n, T, k, trace=True).astype(np.float64) / (L * L)
    bins = tr.reshape(-1, 200).mean(axis=1)
    sigma = bins.std(ddof=1) / math.sqrt(len(bins))
    exact = float(G4["e"][0])
    assert abs(tr.mean() - exact) < 3 * sigma, (tr.mean(), exact, sigma)
    assert 3e-4 < sigma < 8e-3


def test_monte_carlo_energy_L32_against_kaufman():
    # a lattice with several tiles per colour and k = 4 hits, against the exact finite-lattice energy
    L, T, k, beta = 32, 8, 4, 0.4
    exact = kaufman(L, beta)["e"]
    r = oracle.Rng(oracle.PHILOX4X32_10, L * L // 4, 7)
    sp = oracle.ising_init_random(L, 2)
    r.ising_sweep_multihit(sp, L, beta, 500, T, k)
    tr = r.ising_sweep_multihit(sp, L, beta, 6000, T, k, trace=True).astype(np.float64) / (L * L)
    bins = tr.reshape(-1, 100).mean(axis=1)
    sigma = bins.std(ddof=1) / math.sqrt(len(bins))
    assert abs(tr.mean() - exact) < 3 * sigma, (tr.mean(), exact, sigma)
