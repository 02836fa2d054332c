"""Pins for the oracle's XORShift1024 skip-ahead seeding (instance g starts
g * 2^137 updates after a common state, by multiplying with the 2^137-th power of the
recursion matrix M).  The oracle walks the matrix route (rows of bits, repeated squaring,
vector-matrix products); here it is pinned against routes that share nothing with it:
brute-force stepping, eq.(8) on Python big integers, the period the paper states, and the
POLYNOMIAL route  X M^n = sum_i c_i X M^i  with  c(z) = z^n mod P(z),  P the characteristic
polynomial found by Berlekamp-Massey (weight 475)."""
import numpy as np
import pytest

import oracle
from test_oracle_xs1024 import MASK, _berlekamp_massey, to_int, to_words, update_bigint


def unit(r):
    X = np.zeros(32, dtype=np.uint32)
    X[r // 32] = np.uint32(1) << np.uint32(r % 32)
    return X


@pytest.fixture(scope="module")
def M():
    return oracle.xs1024_matpow2(0)


@pytest.fixture(scope="module")
def J():
    return oracle.xs1024_matpow2(137)


def test_matrix_rows_are_eq8_on_unit_vectors(M):
    # row r = image of e_r under eq.(8) evaluated on Python integers (not by the oracle's update)
    for r in list(range(0, 1024, 37)) + [0, 31, 32, 1023]:
        assert to_int(M[r]) == update_bigint(to_int(unit(r))), r
    # unit vector "word w, bit b" is bit 32*(31-w)+b of the 1024-bit X (lane 0 = MSW, R-D1)
    assert to_int(unit(5 * 32 + 3)) == 1 << (32 * 26 + 3)


def test_vecmat_is_one_update_and_is_linear(M):
    rng = np.random.default_rng(1)
    for _ in range(5):
        X = rng.integers(0, 2**32, 32, dtype=np.uint32)
        Y = rng.integers(0, 2**32, 32, dtype=np.uint32)
        assert to_int(oracle.xs1024_vecmat(X, M)) == update_bigint(to_int(X))
        assert np.array_equal(oracle.xs1024_vecmat(X ^ Y, M), oracle.xs1024_vecmat(X, M) ^ oracle.xs1024_vecmat(Y, M))
    assert not oracle.xs1024_vecmat(np.zeros(32, dtype=np.uint32), M).any()


def test_power_by_squaring_equals_brute_force_steps():
    # X M^(2^k) against 2^k single updates, k = 0..11 (4095 brute-force steps in total)
    rng = np.random.default_rng(2)
    X = rng.integers(0, 2**32, 32, dtype=np.uint32)
    v, steps = to_int(X), 0
    for k in range(12):
        while steps < (1 << k):
            v = update_bigint(v)
            steps += 1
        assert to_int(oracle.xs1024_vecmat(X, oracle.xs1024_matpow2(k))) == v, k


def test_matmul_is_composition_and_powers_add(M):
    A, B = oracle.xs1024_matpow2(3), oracle.xs1024_matpow2(5)
    AB = oracle.xs1024_matmul(A, B)
    assert np.array_equal(AB, oracle.xs1024_matmul(B, A))             # powers of one matrix commute
    X = np.random.default_rng(3).integers(0, 2**32, 32, dtype=np.uint32)
    v = to_int(X)
    for _ in range(8 + 32):
        v = update_bigint(v)
    assert to_int(oracle.xs1024_vecmat(X, AB)) == v                     # M^8 M^32 = M^40
    assert np.array_equal(oracle.xs1024_matmul(A, A), oracle.xs1024_matpow2(4))


def test_period_divides_2_1024_minus_1(M):
    # maximal period 2^1024 - 1, hence M^(2^1024) = M (and no smaller 2^k does it:
    # a smaller k with M^(2^k) = M would put the period inside 2^k - 1)
    P = M.copy()
    for k in range(1, 1025):
        P = oracle.xs1024_matmul(P, P)
        if k < 1024 and k % 64 == 0:
            assert not np.array_equal(P, M), k
    assert np.array_equal(P, M)


# ---- the independent polynomial route --------------------------------------------------
def _connection_polynomial():
    X = np.zeros(32, dtype=np.uint32)
    X[31] = 1
    bits = []
    for _ in range(2048):
        oracle.xs1024_update(X)
        bits.append((int(X[15]) >> 5) & 1)
    C, L = _berlekamp_massey(bits)          # connection polynomial 1 + c_1 z + ... + c_L z^L
    assert L == 1024
    return C


def _polymulmod(a, b, P):
    """a*b mod P over GF(2), polynomials as Python ints (bit i = coefficient of z^i), deg P = 1024"""
    r = 0
    while b:
        if b & 1:
            r ^= a
        b >>= 1
        a <<= 1
        if a >> 1024:
            a ^= P
    return r


def _apply_poly(c, v):
    """sum_i c_i (v M^i) on Python integers"""
    acc = 0
    for i in range(1024):
        if (c >> i) & 1:
            acc ^= v
        v = update_bigint(v)
    return acc


@pytest.fixture(scope="module")
def charpoly():
    # Berlekamp-Massey returns C(z) = 1 + c_1 z + ... + c_1024 z^1024 with s_N = sum c_i s_{N-i};
    # the characteristic polynomial of the recurrence is its reciprocal z^1024 C(1/z)
    C = _connection_polynomial()
    P = 0
    for i in range(1025):
        if (C >> i) & 1:
            P |= 1 << (1024 - i)
    assert P >> 1024 == 1 and P & 1 == 1 and bin(P).count("1") == 475
    return P


def test_cayley_hamilton_pins_the_polynomial(charpoly):
    # P(M) = 0: sum_i p_i X M^i = 0 for any X (1025 terms)
    v = to_int(np.random.default_rng(4).integers(0, 2**32, 32, dtype=np.uint32))
    acc, x = 0, v
    for i in range(1025):
        if (charpoly >> i) & 1:
            acc ^= x
        x = update_bigint(x)
    assert acc == 0


def test_skip_matrix_equals_polynomial_route(charpoly, J):
    # z^(2^137) mod P by 137 modular squarings, applied as a polynomial in M with 1024 big-int
    # updates, against the oracle's matrix M^(2^137)
    c = 2  # z
    for _ in range(137):
        c = _polymulmod(c, c, charpoly)
    rng = np.random.default_rng(5)
    for _ in range(3):
        X = rng.integers(0, 2**32, 32, dtype=np.uint32)
        assert to_int(oracle.xs1024_vecmat(X, J)) == _apply_poly(c, to_int(X))
    # and a small exponent through the same machinery against brute force (pins _polymulmod/_apply_poly)
    c5 = 2
    for _ in range(5):
        c5 = _polymulmod(c5, c5, charpoly)
    v = w = to_int(X)
    for _ in range(32):
        w = update_bigint(w)
    assert _apply_poly(c5, v) == w


def test_skip_seeded_instances_are_2_137_apart(J):
    S, seed = 32 * 5, 7
    r = oracle.Rng(oracle.XS1024W_SKIP, S, seed)
    st = r.get_state().reshape(5, 32)
    # instance 0 = the common start state = instance 0 of the random seeding (R-D7b)
    assert np.array_equal(st[0], oracle.Rng(oracle.XS1024W, 32, seed).get_state())
    for g in range(1, 5):
        assert np.array_equal(st[g], oracle.xs1024_vecmat(st[g - 1], J)), g
    # a shard sees the same instances; the generator itself is kind 4's (same update, same Weyl term)
    sh = oracle.Rng(oracle.XS1024W_SKIP, 64, seed, first=64, n_total=S)
    assert np.array_equal(sh.get_state().reshape(2, 32), st[2:4])
    a = oracle.Rng(oracle.XS1024W, 32, seed).fill_u32(9)
    b = oracle.Rng(oracle.XS1024W_SKIP, 32, seed).fill_u32(9)
    assert np.array_equal(a, b)                                        # instance 0 is common to both
    out = r.fill_u32(3).reshape(S, 3)
    X = st[1].copy()
    oracle.xs1024_update(X)
    y = 362437
    assert np.array_equal(out[32:64, 0], ((y ^ (y >> 16)) + X.astype(np.uint64)).astype(np.uint32))
    with pytest.raises(ValueError):
        oracle.Rng(oracle.XS1024W_SKIP, 48, 1)
