"""Pins for the oracle's XORShift1024/Weyl, the paper's generator
(eq.(8), :177, :201-225 Listing 1, :232-240 eq.(9))."""
import numpy as np
import pytest

import oracle
from conftest import read_golden

G = read_golden("paper_constants.txt")
SA, SB, SC = (int(v) for v in G["xs1024_abc"])
MASK = (1 << 1024) - 1
M32 = 0xFFFFFFFF


def to_int(X):
    """lane 0 is the MOST significant word (DESIGN.md R-D1)."""
    v = 0
    for w in X:
        v = (v << 32) | int(w)
    return v


def to_words(v):
    return np.array([(v >> (32 * (31 - i))) & M32 for i in range(32)], dtype=np.uint32)


def update_bigint(v):
    """eq.(8) on a Python integer: x ^ (x << a) etc."""
    v ^= (v << SA) & MASK
    v ^= v >> SB
    v ^= (v << SC) & MASK
    return v


def update_listing1(state_words):
    """Transcription of Listing 1 for ONE warp, with the padded
    shared array of Fig.2: WORDSHIFT+1 zero words on either side, every
    thread first stores, then all threads read the *stored* values."""
    WARPSIZE, WORD = 32, 32
    WORDSHIFT = int(G["xs1024_wordshift"][0])
    RA, RB, RC = (int(v) for v in G["xs1024_rand_abc"])
    assert (WORDSHIFT, RA, RB, RC) == (SA // 32, SA % 32, SB % 32, SC % 32) and SB // 32 == SC // 32 == WORDSHIFT
    pad = WORDSHIFT + 1
    block = [0] * (pad + WARPSIZE + pad)          # zeros | warp state | zeros
    woff = pad
    st = [int(w) for w in state_words]

    def share():
        for lid in range(WARPSIZE):
            block[woff + lid] = st[lid]

    share()                                         # << A
    for lid in range(WARPSIZE):
        lp = lid + WORDSHIFT
        st[lid] ^= (block[woff + lp] << RA) & M32
        st[lid] ^= block[woff + lp + 1] >> (WORD - RA)
    share()                                         # >> B
    for lid in range(WARPSIZE):
        lm = lid - WORDSHIFT
        st[lid] ^= (block[woff + lm - 1] << (WORD - RB)) & M32
        st[lid] ^= block[woff + lm] >> RB
    share()                                         # << C
    for lid in range(WARPSIZE):
        lp = lid + WORDSHIFT
        st[lid] ^= (block[woff + lp] << RC) & M32
        st[lid] ^= block[woff + lp + 1] >> (WORD - RC)
    return np.array(st, dtype=np.uint32)


def _rand_state(rng):
    return rng.integers(0, 2**32, 32, dtype=np.uint64).astype(np.uint32)


def test_update_equals_eq8_on_big_integers_and_listing1():
    rng = np.random.default_rng(1)
    for _ in range(200):
        X = _rand_state(rng)
        Y = X.copy()
        oracle.xs1024_update(Y)
        assert to_int(Y) == update_bigint(to_int(X))
        assert np.array_equal(Y, update_listing1(X))


def test_lane0_is_most_significant_word():
    # with lane 0 = LEAST significant word Listing 1 and eq.(8) disagree: the reading is pinned
    rng = np.random.default_rng(2)
    X = _rand_state(rng)
    lsw_first = sum(int(w) << (32 * i) for i, w in enumerate(X))
    got = update_bigint(lsw_first)
    L1 = update_listing1(X)
    assert got != sum(int(w) << (32 * i) for i, w in enumerate(L1))


def test_one_hot_hand_trace():
    g = read_golden("xs1024_trace.txt")
    X = np.zeros(32, dtype=np.uint32)
    X[31] = 1
    oracle.xs1024_update(X)
    assert to_int(X) == sum(1 << int(b) for b in g["step1_bits"])
    want = {int(k): int(v, 16) for k, v in (e.split(":") for e in g["step1_lanes"])}
    assert {i: int(v) for i, v in enumerate(X) if v} == want
    oracle.xs1024_update(X)
    want = {int(k): int(v, 16) for k, v in (e.split(":") for e in g["step2_lanes"])}
    assert {i: int(v) for i, v in enumerate(X) if v} == want


def test_linear_zero_fixed_and_invertible():
    rng = np.random.default_rng(3)
    Z = np.zeros(32, dtype=np.uint32)
    oracle.xs1024_update(Z)
    assert not Z.any()
    for _ in range(50):
        A, B = _rand_state(rng), _rand_state(rng)
        AB = A ^ B
        for X in (A, B, AB):
            oracle.xs1024_update(X)
        assert np.array_equal(AB, A ^ B)

    # each factor (I + L^a) is unipotent: (I + L^a)^{-1} = I + L^a + L^2a + ... (finite sum)
    def inv_left(v, a):
        acc, t = 0, v
        while t:
            acc ^= t
            t = (t << a) & MASK
        return acc

    def inv_right(v, b):
        acc, t = 0, v
        while t:
            acc ^= t
            t >>= b
        return acc

    for _ in range(50):
        X = _rand_state(rng)
        Y = X.copy()
        oracle.xs1024_update(Y)
        v = inv_left(to_int(Y), SC)
        v = inv_right(v, SB)
        v = inv_left(v, SA)
        assert v == to_int(X)


def _berlekamp_massey(bits):
    """minimal LFSR (connection polynomial as an int bitmask, degree) of a bit sequence"""
    n = len(bits)
    s = 0
    for i, b in enumerate(bits):
        s |= (b & 1) << i
    C, B = 1, 1
    L, m = 0, 1
    for N in range(n):
        # discrepancy d = s_N + sum_{i=1..L} c_i s_{N-i}
        window = (s >> (N - L)) & ((1 << (L + 1)) - 1) if N >= L else 0
        # bit i of C pairs with s_{N-i}: reverse-align by iterating set bits of C
        d = 0
        c, i = C, 0
        acc = 0
        while c:
            if c & 1:
                acc ^= (s >> (N - i)) & 1
            c >>= 1
            i += 1
        d = acc
        if d:
            T = C
            C ^= B << m
            if 2 * L <= N:
                L, B, m = N + 1 - L, T, 1
            else:
                m += 1
        else:
            m += 1
    return C, L


def test_characteristic_polynomial_weight_475_degree_1024():
    # (a,b,c) = (329,347,344) "has a primitive characteristic polynomial of weight
    # 475" and maximal period 2^1024 - 1.  The minimal polynomial of any non-degenerate output
    # bit sequence is then that polynomial: Berlekamp-Massey on 2048 bits of one state bit must
    # give linear complexity 1024 and a connection polynomial with 475 non-zero terms.
    X = np.zeros(32, dtype=np.uint32)
    X[31] = 1
    bits = []
    for _ in range(2 * int(G["xs1024_charpoly_degree"][0])):
        oracle.xs1024_update(X)
        bits.append((int(X[15]) >> 5) & 1)               # bit 517 of X
    poly, L = _berlekamp_massey(bits)
    assert L == int(G["xs1024_charpoly_degree"][0])
    assert bin(poly).count("1") == int(G["xs1024_charpoly_weight"][0])


def test_wrong_triple_does_not_have_that_polynomial():
    # sanity of the pin itself: swapping b and c changes degree/weight
    def upd(v):
        v ^= (v << 329) & MASK
        v ^= v >> 344
        v ^= (v << 347) & MASK
        return v
    v, bits = 1, []
    for _ in range(2048):
        v = upd(v)
        bits.append((v >> 517) & 1)
    poly, L = _berlekamp_massey(bits)
    assert (L, bin(poly).count("1")) != (1024, 475)


def test_weyl_output_and_stream_layout():
    g = read_golden("xs1024_trace.txt")
    c = int(G["weyl_c"][0])
    gam = int(G["weyl_gamma"][0])
    terms = [((n * c) & M32) ^ (((n * c) & M32) >> gam) for n in (1, 2)]
    assert terms == [int(v, 16) for v in g["weyl_terms"]]

    S, n, seed = 64, 6, 1
    r = oracle.Rng(oracle.XS1024W, S, seed)
    st = r.get_state().copy()                            # word i of instance g at 32 g + i
    # seeding: lane 2k = lo32(SM[16 g + k]), lane 2k+1 = hi32  (PAPER.md:230 random seeding)
    for gi in range(S // 32):
        for k in range(16):
            z = oracle.splitmix64(seed, 16 * gi + k)
            assert int(st[32 * gi + 2 * k]) == z & M32 and int(st[32 * gi + 2 * k + 1]) == z >> 32
    out = r.fill_u32(n).reshape(S, n)
    for gi in range(S // 32):
        v = to_int(st[32 * gi:32 * gi + 32])
        for j in range(n):
            v = update_bigint(v)
            y = ((j + 1) * c) & M32
            t = y ^ (y >> gam)
            w = to_words(v)
            for i in range(32):
                assert out[32 * gi + i, j] == (t + int(w[i])) & M32
    # the Weyl index continues across calls (n = number of updates since creation)
    more = r.fill_u32(2).reshape(S, 2)
    r2 = oracle.Rng(oracle.XS1024W, S, seed)
    assert np.array_equal(r2.fill_u32(n + 2).reshape(S, n + 2)[:, n:], more)


def test_one_hot_draws_with_weyl():
    # SURVEY 8(c)-D6 values: X0 = 1 -> draw 1 lane 31 = 0x587c1, lane 0 = 0x587c0; draw 2 ...
    g = read_golden("xs1024_trace.txt")
    X = np.zeros(32, dtype=np.uint32)
    X[31] = 1
    for n, key in ((1, "draw1"), (2, "draw2")):
        oracle.xs1024_update(X)
        y = (n * 362437) & M32
        t = y ^ (y >> 16)
        for e in g[key]:
            lane, val = e.split(":")
            assert (t + int(X[int(lane)])) & M32 == int(val, 16)


def test_requires_whole_instances():
    with pytest.raises(ValueError):
        oracle.Rng(oracle.XS1024W, 48, 1)
    sh = oracle.Rng(oracle.XS1024W, 32, 1, first=32, n_total=96).fill_u32(3)
    whole = oracle.Rng(oracle.XS1024W, 96, 1).fill_u32(3).reshape(96, 3)
    assert np.array_equal(sh.reshape(32, 3), whole[32:64])
