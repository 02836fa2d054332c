"""Pins for the oracle's XORWOW and Philox4x32-10."""
import numpy as np
import pytest

import oracle
from conftest import read_golden

M32 = 0xFFFFFFFF


# -------------------------------------------------------------------- XORWOW
def _u32(vals):
    return np.array([int(v) for v in vals], dtype=np.uint32)


def test_xorwow_hand_trace_and_marsaglia_defaults():
    g = read_golden("xorwow_trace.txt")
    st = _u32(g["unit_state"])
    assert [oracle.xorwow_next(st) for _ in range(8)] == [int(v, 16) for v in g["unit_first8"]]
    st = _u32(g["marsaglia_state"])
    assert [oracle.xorwow_next(st) for _ in range(5)] == [int(v) for v in g["marsaglia_first5"]]


def test_xorwow_weyl_part_is_closed_form_and_xorshift_part_is_linear():
    # Weyl sequence d_n = d_0 + n c (mod 2^32), c = 362437
    c = int(read_golden("paper_constants.txt")["weyl_c"][0])
    rng = np.random.default_rng(11)
    s1 = rng.integers(0, 2**32, 6, dtype=np.uint64).astype(np.uint32)
    s2 = rng.integers(0, 2**32, 6, dtype=np.uint64).astype(np.uint32)
    d0 = int(s1[5])
    a, b, x = s1.copy(), s2.copy(), (s1 ^ s2)
    for n in range(1, 200):
        oracle.xorwow_next(a)
        oracle.xorwow_next(b)
        oracle.xorwow_next(x)
        assert int(a[5]) == (d0 + n * c) & M32
        # xorshift part (5 words) is GF(2)-linear: f(s1 ^ s2) = f(s1) ^ f(s2)
        assert np.array_equal(x[:5], a[:5] ^ b[:5])


def test_xorwow_output_is_weyl_plus_last_word_and_register_rotation():
    st = np.array([5, 6, 7, 8, 9, 100], dtype=np.uint32)
    old = st.copy()
    out = oracle.xorwow_next(st)
    assert list(st[:4]) == list(old[1:5])          # x<-y, y<-z, z<-w, w<-v
    assert out == (int(st[4]) + int(st[5])) & M32  # d + v after the advance
    t = int(old[0]) ^ (int(old[0]) >> 2)
    v = int(old[4])
    assert int(st[4]) == ((v ^ (v << 4)) ^ (t ^ (t << 1))) & M32


def test_xorwow_period_structure_on_tiny_input():
    # the xorshift part is an invertible linear map: zero is a fixed point and the
    # only state mapping to zero (a wrong shift direction would break invertibility
    # on random inputs with overwhelming probability: check injectivity on 2^12 states)
    z = np.zeros(6, dtype=np.uint32)
    oracle.xorwow_next(z)
    assert not z[:5].any()
    seen = set()
    for i in range(1 << 12):
        st = np.array([i & 0xF, (i >> 4) & 0xF, 0, 0, (i >> 8) & 0xF, 0], dtype=np.uint32)
        oracle.xorwow_next(st)
        seen.add(tuple(int(v) for v in st[:5]))
    assert len(seen) == 1 << 12


def test_xorwow_seeding_from_splitmix64_and_zero_guard():
    S, seed = 4, 1
    st = oracle.Rng(oracle.XORWOW, S, seed).get_state().reshape(S, 6)
    for s in range(S):
        z = [oracle.splitmix64(seed, 3 * s + p) for p in range(3)]
        want = [z[0] & M32, z[0] >> 32, z[1] & M32, z[1] >> 32, z[2] & M32, z[2] >> 32]
        assert [int(v) for v in st[s]] == want
    # shard: stream ids are global
    st2 = oracle.Rng(oracle.XORWOW, 2, seed, first=2, n_total=4).get_state().reshape(2, 6)
    assert np.array_equal(st2, st[2:4])


def test_xorwow_stream_fill_matches_elementary_function():
    S, n = 3, 20
    r = oracle.Rng(oracle.XORWOW, S, 2)
    st = r.get_state().reshape(S, 6).copy()
    out = r.fill_u32(n).reshape(S, n)
    for s in range(S):
        assert [oracle.xorwow_next(st[s]) for _ in range(n)] == [int(v) for v in out[s]]
    assert np.array_equal(r.get_state().reshape(S, 6), st)


# -------------------------------------------------------------------- Philox
M0, M1 = 0xD2511F53, 0xCD9E8D57
W0, W1 = 0x9E3779B9, 0xBB67AE85


def test_philox_known_answers():
    for name, v in read_golden("philox_kat.txt").items():
        R = int(v[0])
        ctr = [int(x, 16) for x in v[1:5]]
        key = [int(x, 16) for x in v[5:7]]
        want = [int(x, 16) for x in v[7:11]]
        assert [int(x) for x in oracle.philox4x32(ctr, key, R)] == want, name


def _sbox(L, R, M, k):
    """PAPER.md:290-292:  L' = mullo(R, M);  R' = mulhi(R, M) xor k xor L."""
    p = R * M
    return p & M32, ((p >> 32) ^ k ^ L) & M32


def _philox_paper_form(ctr, key, rounds):
    """The paper's description: per round N/2 = 2 S-boxes with different multipliers and
    constant key k per thread, then a permutation; Ref.[20] bumps the key
    words by the Weyl constants between rounds."""
    x = list(ctr)
    k = list(key)
    for _ in range(rounds):
        La, Ra = _sbox(x[1], x[2], M1, k[0])
        Lb, Rb = _sbox(x[3], x[0], M0, k[1])
        x = [Ra, La, Rb, Lb]
        k = [(k[0] + W0) & M32, (k[1] + W1) & M32]
    return x


def _philox_inverse(out, key, rounds):
    """"Since multiplication, permutation and XOR are bijective ... the
    transformation is bijective".  Undo each round: the mullo words give R back through the
    inverse of the (odd) multiplier mod 2^32; then L = R' xor mulhi(R, M) xor k."""
    i0, i1 = pow(M0, -1, 1 << 32), pow(M1, -1, 1 << 32)
    x = list(out)
    for r in reversed(range(rounds)):
        k0, k1 = (key[0] + r * W0) & M32, (key[1] + r * W1) & M32
        Ra, La, Rb, Lb = x
        c2 = (La * i1) & M32
        c0 = (Lb * i0) & M32
        c1 = Ra ^ ((c2 * M1) >> 32) ^ k0
        c3 = Rb ^ ((c0 * M0) >> 32) ^ k1
        x = [c0, c1, c2, c3]
    return x


def test_philox_matches_papers_sbox_description_and_is_bijective():
    rng = np.random.default_rng(5)
    for _ in range(300):
        ctr = [int(v) for v in rng.integers(0, 2**32, 4, dtype=np.uint64)]
        key = [int(v) for v in rng.integers(0, 2**32, 2, dtype=np.uint64)]
        for R in (7, 10):
            o = [int(v) for v in oracle.philox4x32(ctr, key, R)]
            assert o == _philox_paper_form(ctr, key, R)
            assert _philox_inverse(o, key, R) == ctr


def test_philox_toy_version_is_a_permutation():
    # 4 x 4-bit toy Philox with the same wiring: exhaustive over all 2^16 counters.
    def toy(ctr, key, rounds=4, w=4, m0=0xD, m1=0xB, w0=0x9, w1=0xB):
        mask = (1 << w) - 1
        x, k = list(ctr), list(key)
        for _ in range(rounds):
            pa, pb = x[2] * m1, x[0] * m0
            x = [((pa >> w) ^ k[0] ^ x[1]) & mask, pa & mask, ((pb >> w) ^ k[1] ^ x[3]) & mask, pb & mask]
            k = [(k[0] + w0) & mask, (k[1] + w1) & mask]
        return tuple(x)
    outs = {toy(((i >> 12) & 15, (i >> 8) & 15, (i >> 4) & 15, i & 15), (3, 7)) for i in range(1 << 16)}
    assert len(outs) == 1 << 16


def test_philox_stream_mapping_and_order_independence():
    # BASELINE.json config 2: key = stream id ^ seed, counter = draw index (per 4-word block)
    S, n, seed = 5, 23, 0x0123456789ABCDEF
    out = oracle.Rng(oracle.PHILOX4X32_10, S, seed).fill_u32(n).reshape(S, n)
    idx = [(s, j) for s in range(S) for j in range(n)]
    np.random.default_rng(0).shuffle(idx)
    for s, j in idx[:60]:                                       # any (s, j) alone, any order
        K = s ^ seed
        o = oracle.philox4x32([j // 4, 0, 0, 0], [K & M32, K >> 32])
        assert out[s, j] == o[j % 4]


def test_philox_fill_continues_across_unaligned_calls_and_shards():
    S, seed = 4, 77
    a = oracle.Rng(oracle.PHILOX4X32_10, S, seed).fill_u32(22).reshape(S, 22)
    r = oracle.Rng(oracle.PHILOX4X32_10, S, seed)
    parts = [r.fill_u32(k).reshape(S, k) for k in (3, 6, 1, 12)]
    assert np.array_equal(a, np.concatenate(parts, axis=1))
    sh = oracle.Rng(oracle.PHILOX4X32_10, 2, seed, first=1, n_total=S).fill_u32(22).reshape(2, 22)
    assert np.array_equal(sh, a[1:3])


def test_philox_high_counter_word_is_used():
    # block index >= 2^32 must reach the second counter word
    K = 9
    o = oracle.philox4x32([5, 1, 0, 0], [K, 0])
    assert not np.array_equal(o, oracle.philox4x32([5, 0, 0, 0], [K, 0]))


def test_philox_repositioned_stream_crosses_the_2_32_block_boundary():
    # the counter is the draw index (R-C2): a stream set to draw 4*(2^32 - 3) must produce the blocks
    # (2^32-3, 0), (2^32-2, 0), (2^32-1, 0), (0, 1), (1, 1) of the elementary function (Ref.[20] KAT-pinned)
    S, seed, start = 3, 0xABCDEF, 4 * ((1 << 32) - 3)
    for kind, R in ((oracle.PHILOX4X32_10, 10), (oracle.PHILOX4X32_7, 7)):
        r = oracle.Rng(kind, S, seed)
        r.draws_done = start + 2                      # unaligned on purpose
        out = r.fill_u32(18).reshape(S, 18)
        assert r.draws_done == start + 20
        for s in range(S):
            K = s ^ seed
            for j in range(18):
                b = (start + 2 + j) // 4
                o = oracle.philox4x32([b & M32, b >> 32, 0, 0], [K & M32, K >> 32], R)
                assert out[s, j] == o[(start + 2 + j) % 4]
    with pytest.raises(ValueError):
        oracle.Rng(oracle.XORWOW, 4, 1).draws_done = 8   # stateful streams cannot be repositioned
