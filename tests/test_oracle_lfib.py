"""Pins for the oracle's lagged Fibonacci generators (eq.(5):
u_n = u_{n-r} + u_{n-s} mod 1 in single precision, (r,s) = (521,353) and (1279,861), ring buffer
shared by the 256 streams of an instance; readings R-G1..G3 in DESIGN.md).  CPU only.

Pinned against things that are not the oracle: the additive lagged Fibonacci recurrence on Python
integers mod 2^23 (the float recurrence must BE that, exactly), the shift-register structure of the
low bit (Berlekamp-Massey must find the trinomial z^r + z^s + 1 of PAPER.md:122), and uniformity."""
import math

import numpy as np
import pytest

import oracle
from test_oracle_xs1024 import _berlekamp_massey

T = 256
LAGS = {oracle.LFIB521: (521, 353), oracle.LFIB1279: (1279, 861)}
KINDS = list(LAGS)
IDS = ["r521", "r1279"]
M32 = 0xFFFFFFFF


def seed_ints(kind, seed, g):
    """R-G3 on Python integers: 23-bit fractions from the splitmix64 word sequence"""
    r, _ = LAGS[kind]
    k = []
    for i in range(r):
        w = g * r + i
        z = oracle.splitmix64(seed, w // 2)
        k.append((((z >> 32) if w & 1 else z) & M32) >> 9)
    if not any(v & 1 for v in k):
        k[0] += 1
    return k


def integer_sequence(kind, seed, g, count):
    """x_n = x_{n-r} + x_{n-s} mod 2^23 -- the textbook additive lagged Fibonacci generator"""
    r, s = LAGS[kind]
    x = seed_ints(kind, seed, g)
    for n in range(r, r + count):
        x.append((x[n - r] + x[n - s]) & ((1 << 23) - 1))
    return x[r:]


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_float_recurrence_is_the_integer_recurrence_mod_2_23(kind):
    S, seed, n = 2 * T, 5, 40
    out = oracle.Rng(kind, S, seed).fill_u32(n).reshape(S, n)
    f = oracle.Rng(kind, S, seed).fill_f32(n).reshape(S, n)
    for g in range(2):
        v = integer_sequence(kind, seed, g, n * T)
        want = np.array(v, dtype=np.uint64).reshape(n, T).T          # stream t, draw j = v[j*T + t] (R-G2)
        assert np.array_equal(out[g * T:(g + 1) * T] >> 9, want.astype(np.uint32))
        assert not (out[g * T:(g + 1) * T] & 0x1FF).any()
        assert np.array_equal(f[g * T:(g + 1) * T], (want.astype(np.float64) * 2.0 ** -23).astype(np.float32))
    # the fixed map (u >> 8) 2^-24 gives the float stream back
    assert np.array_equal((out >> 8).astype(np.float32) * np.float32(2.0 ** -24), f)


def test_one_float_addition_mod_1():
    add = oracle.lib().orc_lfib_add
    import ctypes as C
    add.restype, add.argtypes = C.c_float, [C.c_float, C.c_float]
    h = 2.0 ** -23
    assert add(0.25, 0.5) == 0.75
    assert add(0.75, 0.5) == 0.25
    assert add(1 - h, h) == 0.0                       # wraps to exactly 0
    assert add(1 - h, 1 - h) == np.float32(1 - 2 * h)  # largest possible sum: exact in [1,2), then - 1
    assert add(0.5, 0.5 - h) == np.float32(1 - h)      # just below 1: no wrap


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_low_bit_sequence_has_the_trinomial_of_the_paper(kind):
    # mod 2 the recurrence is the shift register x_n = x_{n-r} ^ x_{n-s}; (r,s) of PAPER.md:122 are primitive
    # trinomials, so Berlekamp-Massey on 2r+64 low bits finds linear complexity r and exactly the taps {0,s,r}.
    # A swapped pair, an off-by-one lag or a wrong dealing order changes the complexity or the taps.
    r, s = LAGS[kind]
    n = (2 * r + 64 + T - 1) // T
    out = oracle.Rng(kind, T, 3).fill_u32(n).reshape(T, n)
    seq = out.T.reshape(-1)                                    # v_m in sequence order: m = j*T + t
    bits = [int(v >> 9) & 1 for v in seq[:2 * r + 64]]
    C, Lc = _berlekamp_massey(bits)
    assert Lc == r
    taps = [i for i in range(r + 1) if (C >> i) & 1]
    assert taps == [0, r - s, r] or taps == [0, s, r], taps
    # connection polynomial 1 + z^a + z^r means x_n = x_{n-a} + x_{n-r}: a must be s
    assert taps == [0, s, r]


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_continuation_state_and_shards(kind):
    r, s = LAGS[kind]
    S, seed = 3 * T, 11
    whole = oracle.Rng(kind, S, seed).fill_u32(30).reshape(S, 30)
    a = oracle.Rng(kind, S, seed)
    parts = [a.fill_u32(k).reshape(S, k) for k in (1, 7, 2, 20)]
    assert np.array_equal(np.concatenate(parts, axis=1), whole)
    # state = the last r numbers of each instance, oldest first, as float bit patterns
    st = a.get_state().view(np.float32).reshape(3, r)
    v = integer_sequence(kind, seed, 1, 30 * T)
    hist = (seed_ints(kind, seed, 1) + v)[-r:]
    assert np.array_equal(st[1], (np.array(hist, dtype=np.float64) * 2.0 ** -23).astype(np.float32))
    sh = oracle.Rng(kind, T, seed, first=T, n_total=S).fill_u32(30).reshape(T, 30)
    assert np.array_equal(sh, whole[T:2 * T])
    with pytest.raises(ValueError):
        oracle.Rng(kind, 100, 1)                                  # whole 256-stream instances only
    # draw_reduce = checksums of the same draws
    red = oracle.Rng(kind, S, seed).draw_reduce(30).reshape(S, 2)
    assert np.array_equal(red[:, 0], np.bitwise_xor.reduce(whole, axis=1))
    assert np.array_equal(red[:, 1], whole.sum(axis=1, dtype=np.uint64).astype(np.uint32))


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_uniformity(kind):
    f = oracle.Rng(kind, 4 * T, 1).fill_f32(2048).astype(np.float64)
    n = f.size
    assert abs(f.mean() - 0.5) < 3 * math.sqrt(1 / (12 * n))
    assert abs(f.var() - 1 / 12) < 3 * math.sqrt(1 / (180 * n))
    cnt = np.bincount((f * 256).astype(np.int64), minlength=256).astype(np.float64)
    chi2 = ((cnt - n / 256) ** 2 / (n / 256)).sum()
    assert 255 - 3 * math.sqrt(510) < chi2 < 255 + 3 * math.sqrt(510), chi2


def test_ising_consumer_accepts_the_float_generator():
    # one stream per 8 sites; energy after sweeps equals fill-then-apply through the generic oracle path
    L, S = 64, 256
    r = oracle.Rng(oracle.LFIB521, S, 2)
    sp = oracle.ising_init_random(L, 3)
    tr = r.ising_sweep(sp, L, 0.4, 4, trace=True)
    assert tr[-1] == oracle.ising_energy(sp, L) and r.draws_done == 4 * L * L // S
