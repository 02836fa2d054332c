"""Pins for the oracle's multiply-with-carry generator (Table 1 row "MWC, same a").  CPU only.

Pinned against number theory, not against itself: with b = m = 2^32 and p = a b - 1 the state value
s_n = x_n + b c_n obeys  s_{n+1} = b^{-1} s_n  (mod p)  (b s_{n+1} = a b x_n + b c_n = p x_n + s_n), so the
whole sequence is a Lehmer generator on Python integers; p = a m - 1 is the safe prime of PAPER.md:68, and the
period comes out as (a m - 2)/2, half of what the paper states."""
import numpy as np
import pytest

import oracle

A, B = 4294967118, 1 << 32
P = A * B - 1


def _is_probable_prime(n, bases=(2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37)):
    if n < 2:
        return False
    for q in bases:
        if n % q == 0:
            return n == q
    d, r = n - 1, 0
    while d % 2 == 0:
        d //= 2
        r += 1
    for a in bases:
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(r - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def test_multiplier_of_the_paper_gives_a_safe_prime_and_the_stated_period():
    # "one requires am-1 as well as (am-2)/2 to be prime"; "the period is found to be p = am - 2";
    # a = 4294967118 is "the largest safe prime am-1 with a less than 2^32"
    assert _is_probable_prime(P) and _is_probable_prime((P - 1) // 2)
    for a in range(A + 1, B):
        assert not (_is_probable_prime(a * B - 1) and _is_probable_prime((a * B - 2) // 2)), a
    # The period is the order of b modulo p.  It divides p - 1 = 2q (q prime) and is not 1 or 2; because
    # b = 2^32 = (2^16)^2 is a quadratic residue it is q = (a m - 2)/2 = 9.2e18, HALF of the "p = am - 2"
    # the paper states -- noted as reading R-M2 in DESIGN.md; nothing in the method depends on it.
    q = (P - 1) // 2
    assert B % P != 1 and pow(B, 2, P) != 1 and pow(B, q, P) == 1


def test_sequence_is_the_lehmer_generator_b_inverse_mod_p():
    S, seed, n = 6, 3, 200
    r = oracle.Rng(oracle.MWC, S, seed)
    st0 = r.get_state().reshape(S, 2).astype(object)
    out = r.fill_u32(n).reshape(S, n)
    binv = pow(B, -1, P)
    for s in range(S):
        v = int(st0[s, 0]) + B * int(st0[s, 1])
        for j in range(n):
            assert int(out[s, j]) == v % B, (s, j)              # the draw is x_n = s_n mod b
            v = v * binv % P
        end = r.get_state().reshape(S, 2)
        assert int(end[s, 0]) + B * int(end[s, 1]) == v
    # closed form far ahead: s_n = s_0 b^{-n} mod p
    v0 = int(st0[0, 0]) + B * int(st0[0, 1])
    assert v0 * pow(binv, n, P) % P == int(r.get_state()[0]) + B * int(r.get_state()[1])


def test_seeding_continuation_and_shards():
    S, seed = 5, 9
    r = oracle.Rng(oracle.MWC, S, seed)
    st = r.get_state().reshape(S, 2)
    for s in range(S):
        z = oracle.splitmix64(seed, s)
        assert int(st[s, 0]) == z & 0xFFFFFFFF and int(st[s, 1]) == (z >> 32) % A and int(st[s, 1]) < A
    whole = oracle.Rng(oracle.MWC, S, seed).fill_u32(20).reshape(S, 20)
    parts = [r.fill_u32(k).reshape(S, k) for k in (1, 6, 13)]
    assert np.array_equal(np.concatenate(parts, axis=1), whole)
    sh = oracle.Rng(oracle.MWC, 2, seed, first=2, n_total=S).fill_u32(20).reshape(2, 20)
    assert np.array_equal(sh, whole[2:4])
    # the two fixed points of the map are real: one step leaves them where they are
    for x, c in ((0, 0), (B - 1, A - 1)):
        t = A * x + c
        assert (t % B, t // B) == (x, c)


def test_uniformity():
    import math
    f = oracle.Rng(oracle.MWC, 1024, 1).fill_f32(4096).astype(np.float64)
    n = f.size
    assert abs(f.mean() - 0.5) < 3 * math.sqrt(1 / (12 * n))
    assert abs(f.var() - 1 / 12) < 3 * math.sqrt(1 / (180 * n))
    cnt = np.bincount((f * 256).astype(np.int64), minlength=256).astype(np.float64)
    chi2 = ((cnt - n / 256) ** 2 / (n / 256)).sum()
    assert 255 - 3 * math.sqrt(510) < chi2 < 255 + 3 * math.sqrt(510), chi2


# ---- "MWC, different a": one safe-prime multiplier per stream -----------------------------
def test_multipliers_are_the_safe_primes_counted_down_from_the_papers_value():
    mult = [int(a) for a in oracle.mwc_multipliers(0, 120)]
    assert mult[0] == A                                            # "which is just the a = 4294967118 above"
    assert mult == sorted(mult, reverse=True) and len(set(mult)) == len(mult)
    # every listed a qualifies, and NOTHING in between does (Python Miller-Rabin, independent of the C code)
    ok = lambda a: _is_probable_prime(a * B - 1) and _is_probable_prime((a * B - 2) // 2)  # noqa: E731
    listed = set(mult)
    for a in range(mult[-1], B):
        assert ok(a) == (a in listed), a
    # random access further down agrees with the scan from the top
    far = [int(a) for a in oracle.mwc_multipliers(3000, 5)]
    assert all(ok(a) for a in far) and far == [int(a) for a in oracle.mwc_multipliers(0, 3005)[3000:]]


def test_different_a_streams_are_lehmer_generators_with_their_own_modulus():
    S, seed, n = 40, 5, 60
    r = oracle.Rng(oracle.MWC_MULTI, S, seed)
    st0 = r.get_state().reshape(S, 3)
    mult = oracle.mwc_multipliers(0, S)
    assert np.array_equal(st0[:, 2], mult)
    out = r.fill_u32(n).reshape(S, n)
    for s in range(S):
        a = int(mult[s])
        p = a * B - 1
        z = oracle.splitmix64(seed, s)
        assert int(st0[s, 0]) == z & 0xFFFFFFFF and int(st0[s, 1]) == (z >> 32) % a
        v, binv = int(st0[s, 0]) + B * int(st0[s, 1]), pow(B, -1, p)
        for j in range(n):
            assert int(out[s, j]) == v % B
            v = v * binv % p
    # a shard uses the multipliers of its GLOBAL stream ids; continuation keeps them
    sh = oracle.Rng(oracle.MWC_MULTI, 8, seed, first=16, n_total=S)
    assert np.array_equal(sh.get_state().reshape(8, 3)[:, 2], mult[16:24])
    a1, a2 = sh.fill_u32(25).reshape(8, 25), sh.fill_u32(35).reshape(8, 35)
    assert np.array_equal(np.concatenate([a1, a2], axis=1), out[16:24])
