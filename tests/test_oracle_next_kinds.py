"""Pins of the two extra generator kinds of SURVEY.md 8(f)-1 (Table 2 of the paper, PAPER.md:259,
:269): the 32-bit LCG and Philox4x32-7.  Oracle only (-m "not gpu")."""
import numpy as np

import oracle

PHILOX7, LCG32, PHILOX10 = 5, 6, 3


def test_lcg32_textbook_sequence_and_full_period_conditions(golden):
    vals = [int(v, 16) for v in golden("lcg32_values.txt")["from_zero"]]
    x = 0
    for v in vals:
        x = oracle.lcg32_step(x)
        assert x == v
    a, c = 1664525, 1013904223
    assert oracle.lcg32_step(1) == (a + c) % 2**32 and oracle.lcg32_step(0) == c
    assert c % 2 == 1 and a % 4 == 1  # Hull-Dobell: period 2^32


def test_lcg32_streams_are_random_seeded_walks_of_eq1():
    S, n, seed = 5, 40, 1
    r = oracle.Rng(LCG32, S, seed)
    out = r.fill_u32(n).reshape(S, n)
    for s in range(S):
        x = oracle.splitmix64(seed, s) & 0xFFFFFFFF  # x_0 = low word of SM_seed[s]
        for j in range(n):
            assert out[s, j] == x  # draw j = x_j, all 32 bits (u = x/m)
            x = (1664525 * x + 1013904223) % 2**32
    assert list(r.get_state()) == [int(v) for v in oracle.Rng(LCG32, S, seed).fill_u32(n + 1).reshape(S, -1)[:, n]]
    # continuation and shards
    a = oracle.Rng(LCG32, 8, 3)
    whole = np.concatenate([a.fill_u32(3).reshape(8, 3), a.fill_u32(5).reshape(8, 5)], axis=1)
    assert np.array_equal(whole, oracle.Rng(LCG32, 8, 3).fill_u32(8).reshape(8, 8))
    assert np.array_equal(oracle.Rng(LCG32, 3, 3, first=4, n_total=8).fill_u32(8).reshape(3, 8), whole[4:7])


def test_philox7_is_seven_rounds_of_the_pinned_round_function(golden):
    kat = golden("philox_kat.txt")["zeros_r7"]
    assert [int(v, 16) for v in kat[7:]] == list(oracle.philox4x32([0, 0, 0, 0], [0, 0], 7))
    # three more rounds with the key schedule continued give the 10-round answer (pinned by its own KATs)
    rng = np.random.default_rng(0)
    W0, W1 = 0x9E3779B9, 0xBB67AE85
    for _ in range(50):
        ctr = rng.integers(0, 2**32, 4, dtype=np.uint64).astype(np.uint32)
        key = rng.integers(0, 2**32, 2, dtype=np.uint64).astype(np.uint32)
        o7 = oracle.philox4x32(ctr, key, 7)
        k7 = [(int(key[0]) + 7 * W0) % 2**32, (int(key[1]) + 7 * W1) % 2**32]
        assert np.array_equal(oracle.philox4x32(o7, k7, 3), oracle.philox4x32(ctr, key, 10))
        assert not np.array_equal(o7, oracle.philox4x32(ctr, key, 10))


def test_philox7_stream_mapping_is_that_of_philox10():
    S, n, seed = 6, 11, 9
    out = oracle.Rng(PHILOX7, S, seed, first=2, n_total=20).fill_u32(n).reshape(S, n)
    for s in range(S):
        K = (2 + s) ^ seed
        for j in range(n):
            o = oracle.philox4x32([j // 4, 0, 0, 0], [K & 0xFFFFFFFF, K >> 32], 7)
            assert out[s, j] == o[j % 4]
    r = oracle.Rng(PHILOX7, 4, 1)
    a = np.concatenate([r.fill_u32(3).reshape(4, 3), r.fill_u32(6).reshape(4, 6)], axis=1)
    assert np.array_equal(a, oracle.Rng(PHILOX7, 4, 1).fill_u32(9).reshape(4, 9))
    assert r.get_state().size == 0


def test_uniformity_of_the_extra_kinds():
    for kind in (PHILOX7, LCG32):
        f = oracle.Rng(kind, 1 << 12, 1).fill_f32(1 << 12).astype(np.float64)
        n = f.size
        assert abs(f.mean() - 0.5) < 3 * np.sqrt(1 / (12 * n))
        assert abs(f.var() - 1 / 12) < 3 * np.sqrt(1 / (180 * n))
        chi2 = ((np.bincount((f * 256).astype(int), minlength=256) - n / 256) ** 2 / (n / 256)).sum()
        assert 187 < chi2 < 323, (kind, chi2)


def test_lcg64_both_words_is_the_64_bit_sequence_cut_in_two():
    # the whole 64-bit state as two 32-bit numbers.  Against the big-integer recurrence
    # of eq.(1) with the constants of PAPER.md:46, high word first (R-F2); any split of
    # the calls, odd ones included, continues the same stream; the plain LCG64 kind is its even draws.
    a, c, m = 2862933555777941757, 1442695040888963407, 1 << 64
    S, seed, n = 3, 21, 11
    out = oracle.Rng(8, S, seed).fill_u32(n).reshape(S, n)
    for s in range(S):
        x = oracle.splitmix64(seed, s)
        want = []
        while len(want) < n:
            want += [x >> 32, x & 0xFFFFFFFF]
            x = (a * x + c) % m
        assert [int(v) for v in out[s]] == want[:n]
    r = oracle.Rng(8, S, seed)
    parts = [r.fill_u32(k).reshape(S, k) for k in (1, 3, 2, 5)]
    assert np.array_equal(np.concatenate(parts, axis=1), out)
    assert np.array_equal(oracle.Rng(oracle.LCG64, S, seed).fill_u32(5).reshape(S, 5), out[:, 0:10:2])
    # state after an odd number of draws is still x_i (it advances after the low word)
    r = oracle.Rng(8, S, seed)
    r.fill_u32(1)
    st = r.get_state().view(np.uint64)
    assert [int(v) for v in st] == [oracle.splitmix64(seed, s) for s in range(S)]
    r.fill_u32(1)
    assert [int(v) for v in r.get_state().view(np.uint64)] == [(a * oracle.splitmix64(seed, s) + c) % m for s in range(S)]


def test_lcg32_leapfrog_is_one_global_32_bit_sequence():
    # PAPER.md:39-46 (eq.(2),(3)) applied to the 32-bit LCG, the paper's Table 1 row "LCG32":
    # all streams draw from ONE sequence x_{m+1} = 1664525 x_m + 1013904223 mod 2^32, stream s draw j = x_{s + j S}.
    S, n, seed = 7, 9, 4
    out = oracle.Rng(oracle.LCG32_LEAPFROG, S, seed).fill_u32(n).reshape(S, n)
    x = oracle.splitmix64(seed, 0) & 0xFFFFFFFF
    seq = []
    for _ in range(S * n):
        seq.append(x)
        x = (1664525 * x + 1013904223) % (1 << 32)
    assert np.array_equal(out.T.reshape(-1), np.array(seq, dtype=np.uint32))
    # shards and continuation see the same sequence; the state is the stream's next element
    r = oracle.Rng(oracle.LCG32_LEAPFROG, 3, seed, first=2, n_total=S)
    a, b = r.fill_u32(4).reshape(3, 4), r.fill_u32(5).reshape(3, 5)
    assert np.array_equal(np.concatenate([a, b], axis=1), out[2:5])
    r2 = oracle.Rng(oracle.LCG32_LEAPFROG, S, seed)
    r2.fill_u32(2)
    assert [int(v) for v in r2.get_state()] == seq[2 * S:3 * S]
