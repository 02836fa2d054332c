"""Pins for the oracle's splitmix64 and LCG64 (eq.(1)-(3), :58).

Nothing here calls the CUDA path.  Each pin is something other than the oracle
itself: printed constants, a closed form in Python big integers, brute force,
a structural property the paper states.
"""
import numpy as np
import pytest

import oracle
from conftest import read_golden

M64 = (1 << 64) - 1
G = read_golden("paper_constants.txt")
A = int(G["lcg64_a"][0])
Cc = int(G["lcg64_c"][0])


# ---------------------------------------------------------------- splitmix64
def test_splitmix64_published_sequence():
    g = read_golden("splitmix64.txt")
    want = [int(v) for v in g["seed_1234567"]]
    assert [oracle.splitmix64(1234567, k) for k in range(5)] == want
    assert [oracle.splitmix64(1, k) for k in range(4)] == [int(v, 16) for v in g["seed_1"]]
    assert oracle.splitmix64(0, 0) == int(g["seed_0"][0], 16)


def test_splitmix64_random_access_equals_sequential_state_walk():
    # state walk: s += gamma each call; k-th output only depends on seed + (k+1) gamma,
    # so output k of seed s equals output 0 of seed s + k*gamma
    gamma = 0x9E3779B97F4A7C15
    for seed in (0, 1, 2**63 + 5):
        for k in (1, 7, 1000):
            assert oracle.splitmix64(seed, k) == oracle.splitmix64((seed + k * gamma) & M64, 0)


# --------------------------------------------------------------------- LCG64
def test_constants_are_the_papers_and_full_period_conditions():
    # "an odd offset ... needs to be chosen to reach the maximal period";
    # Hull-Dobell for m = 2^64: c odd and a = 1 (mod 4).
    assert oracle.lcg64_step(0) == Cc              # x_1 = a*0 + c
    assert oracle.lcg64_step(1) == (A + Cc) & M64  # x_1 = a + c
    assert Cc % 2 == 1 and A % 4 == 1 and A % 8 == 5


def test_step_matches_eq1_on_random_inputs():
    rng = np.random.default_rng(7)
    for x in rng.integers(0, 2**64, size=200, dtype=np.uint64):
        x = int(x)
        assert oracle.lcg64_step(x) == (A * x + Cc) & M64


def test_printed_values_from_zero():
    g = read_golden("lcg64_values.txt")
    x, got = 0, []
    for _ in range(3):
        x = oracle.lcg64_step(x)
        got.append(x)
    assert got == [int(v, 16) for v in g["from_zero"]]
    assert oracle.lcg64_jump(1024) == tuple(int(v, 16) for v in g["jump_1024"])


def test_low_bits_have_short_period():
    # "the period of the kth least significant bit is only 2^k"
    x0 = oracle.splitmix64(3, 0)
    xs = [x0]
    for _ in range(1 << 11):
        xs.append(oracle.lcg64_step(xs[-1]))
    for k in range(1, 11):
        bits = [(x >> (k - 1)) & 1 for x in xs]
        p = 1 << k
        assert all(bits[i] == bits[i + p] for i in range(len(bits) - p))          # period divides 2^k
        assert any(bits[i] != bits[i + p // 2] for i in range(len(bits) - p))     # and not 2^(k-1)


def _closed_form(n):
    """eq.(2),(3) with exact integers: A_n = a^n, C_n = c (a^n - 1)/(a - 1)  (mod 2^64).
    a^n is reduced modulo (a-1) 2^64 so that the division stays exact."""
    mod = (A - 1) << 64
    an = pow(A, n, mod)
    return an & M64, (Cc * ((an - 1) // (A - 1))) & M64


@pytest.mark.parametrize("n", [0, 1, 2, 3, 5, 1000, 4096, 2**20 + 1, 2**40 + 12345, 2**63 + 1, 2**64 - 1])
def test_jump_equals_closed_form_in_big_integers(n):
    assert oracle.lcg64_jump(n) == _closed_form(n)


def test_jump_equals_brute_force_steps():
    # eq.(2): x_{n+t} = a_t x_n + c_t.  t = 1 must be eq.(1) itself (this is what
    # rejects the literal reading of the garbled eq.(3)).
    assert oracle.lcg64_jump(0) == (1, 0)
    assert oracle.lcg64_jump(1) == (A, Cc)
    x0 = 0x0123456789ABCDEF
    x = x0
    for t in range(1, 10001):
        x = oracle.lcg64_step(x)
        if t in (1, 2, 3, 10, 999, 1024, 4097, 10000):
            At, Ct = oracle.lcg64_jump(t)
            assert (At * x0 + Ct) & M64 == x


def test_jump_additivity():
    # (A_m, C_m) o (A_n, C_n) = (A_{m+n}, C_{m+n})
    for m, n in [(3, 5), (1000, 24), (2**33, 2**35 + 7)]:
        Am, Cm = oracle.lcg64_jump(m)
        An, Cn = oracle.lcg64_jump(n)
        assert ((Am * An) & M64, (Am * Cn + Cm) & M64) == oracle.lcg64_jump(m + n)


def test_eq2_holds_for_the_32bit_lcg_too():
    # the same closed form with the paper's LCG32 constants by brute force:
    # guards the *reading* of eq.(3) independently of the 64-bit code
    a, c, M = int(G["lcg32_a"][0]), int(G["lcg32_c"][0]), (1 << 32) - 1
    x = 12345
    xs = [x]
    for _ in range(100):
        xs.append((a * xs[-1] + c) & M)
    for t in (1, 2, 17, 100):
        at = pow(a, t, 1 << 32)
        ct = (c * sum(pow(a, i, 1 << 32) for i in range(t))) & M   # c * sum_{i=0}^{t-1} a^i
        assert (at * xs[0] + ct) & M == xs[t]


# ------------------------------------------------------------ stream objects
def test_lcg64_stream_layout_and_high_bits():
    S, n, seed = 5, 7, 1
    r = oracle.Rng(oracle.LCG64, S, seed)
    out = r.fill_u32(n).reshape(S, n)
    for s in range(S):
        x = oracle.splitmix64(seed, s)              # x_0^(s) = SM_seed[s]
        for j in range(n):
            assert out[s, j] == x >> 32             # 32 most significant bits
            x = (A * x + Cc) & M64


def test_lcg64_fill_continues():
    a = oracle.Rng(oracle.LCG64, 4, 9).fill_u32(11).reshape(4, 11)
    r = oracle.Rng(oracle.LCG64, 4, 9)
    b = np.concatenate([r.fill_u32(4).reshape(4, 4), r.fill_u32(7).reshape(4, 7)], axis=1)
    assert np.array_equal(a, b) and r.draws_done == 11


def test_leapfrog_is_one_global_sequence():
    # with t = number of threads "all threads can generate numbers out of
    # the same global sequence (1) concurrently".  Union of the streams, re-interleaved,
    # must be the single sequence started at SM_seed[0].
    S, n, seed = 6, 9, 1
    out = oracle.Rng(oracle.LCG64_LEAPFROG, S, seed).fill_u32(n).reshape(S, n)
    x = oracle.splitmix64(seed, 0)
    for m in range(S * n):
        assert out[m % S, m // S] == x >> 32
        x = (A * x + Cc) & M64
    # and stream s is the jump-by-S map applied to X_s (eq.(2) with t = S)
    AS, CS = _closed_form(S)
    x0 = oracle.splitmix64(seed, 0)
    for s in range(S):
        As, Cs = _closed_form(s)
        xs = (As * x0 + Cs) & M64
        for j in range(n):
            assert out[s, j] == xs >> 32
            xs = (AS * xs + CS) & M64


def test_leapfrog_shard_and_state():
    S, n, seed = 8, 5, 3
    whole = oracle.Rng(oracle.LCG64_LEAPFROG, S, seed)
    w = whole.fill_u32(n).reshape(S, n)
    part = oracle.Rng(oracle.LCG64_LEAPFROG, 3, seed, first=2, n_total=S)
    p = part.fill_u32(n).reshape(3, n)
    assert np.array_equal(w[2:5], p)
    st = part.get_state().view(np.uint64)
    nxt = part.fill_u32(1)
    assert np.array_equal(nxt, (st >> np.uint64(32)).astype(np.uint32))


def test_f32_map_is_exact_and_in_range():
    # BASELINE.json: f = (u >> 8) * 2^-24, exact, in [0, 1 - 2^-24]
    assert oracle.u32_to_f32(0) == 0.0
    assert oracle.u32_to_f32(0xFFFFFFFF) == 1.0 - 2.0**-24
    assert oracle.u32_to_f32(0x000000FF) == 0.0
    assert oracle.u32_to_f32(0x00000100) == 2.0**-24
    assert oracle.u32_to_f32(0x80000000) == 0.5
    r1, r2 = oracle.Rng(oracle.LCG64, 3, 5), oracle.Rng(oracle.LCG64, 3, 5)
    u, f = r1.fill_u32(100), r2.fill_f32(100)
    want = (u >> 8).astype(np.float64) / 2.0**24
    assert np.array_equal(f.astype(np.float64), want)       # float32 holds every 24-bit value exactly
    assert f.dtype == np.float32 and f.max() < 1.0 and f.min() >= 0.0


def test_draw_reduce_is_xor_and_sum_of_fill():
    for kind in (oracle.LCG64, oracle.XORWOW, oracle.PHILOX4X32_10, oracle.LCG64_LEAPFROG):
        S, n = 6, 37
        u = oracle.Rng(kind, S, 4).fill_u32(n).reshape(S, n)
        red = oracle.Rng(kind, S, 4).draw_reduce(n).reshape(S, 2)
        assert np.array_equal(red[:, 0], np.bitwise_xor.reduce(u, axis=1))
        assert np.array_equal(red[:, 1], u.sum(axis=1, dtype=np.uint64).astype(np.uint32))
