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


# ---- primality decided by PROOFS, not by the oracle's own algorithm ---------------------------------------
# The oracle decides primality with Miller-Rabin (as the paper says one does).  A pin that ran
# Miller-Rabin again would share any mistake of that route, so the checks below use none of it:
#  * "n is prime" is accepted only with a certificate.  Below 2^32: trial division by every prime up to 2^16.
#    Above: a Lucas / Pratt certificate -- the full factorisation of n - 1 (sympy only FINDS the factors; their
#    product is re-multiplied and each factor is itself proven by this same routine) and a g with
#    g^(n-1) = 1 and g^((n-1)/f) != 1 (mod n) for every prime factor f, i.e. an element of order n - 1.
#    For the safe primes p = 2q + 1, q proven prime: Pocklington's criterion with the single factor q > sqrt(p)
#    (some g with g^(p-1) = 1 and gcd(g^2 - 1, p) = 1).
#  * "n is composite" is accepted only with a witness: a prime factor below 2^16 (gcd with their product), or
#    a base b with b^(n-1) != 1 (mod n) (Fermat: no prime fails it), or, failing both, an explicit factor.
import math

_SMALL = None


def _small_primes():
    global _SMALL
    if _SMALL is None:
        sieve = np.ones(1 << 16, dtype=bool)
        sieve[:2] = False
        for i in range(2, 256):
            if sieve[i]:
                sieve[i * i::i] = False
        _SMALL = [int(q) for q in np.flatnonzero(sieve)]
    return _SMALL


_PRIMORIAL_1000 = math.prod(q for q in range(2, 1000) if all(q % d for d in range(2, int(q ** 0.5) + 1)))


def prove_prime(n: int) -> bool:
    """True only with a proof (trial division or a Pratt certificate); False if n has a factor or no certificate
    was found"""
    if n < 2:
        return False
    if n < 1 << 32:
        for q in _small_primes():
            if q * q > n:
                break
            if n % q == 0:
                return False
        return True
    if math.gcd(n, _PRIMORIAL_1000) != 1 or pow(2, n - 1, n) != 1:
        return False
    import sympy
    fs = sympy.factorint(n - 1)
    assert math.prod(f ** e for f, e in fs.items()) == n - 1
    if not all(prove_prime(int(f)) for f in fs):
        return False
    for g in range(2, 400):
        if pow(g, n - 1, n) == 1 and all(pow(g, (n - 1) // int(f), n) != 1 for f in fs):
            return True  # g has order n - 1: the multiplicative group has n - 1 elements, n is prime
    return False


def prove_safe_prime(p: int) -> bool:
    """p and q = (p - 1)/2 both prime, with proofs: q by prove_prime, p by Pocklington with the factor q"""
    q = (p - 1) // 2
    if p != 2 * q + 1 or not prove_prime(q) or q * q <= p:
        return False
    return any(pow(g, p - 1, p) == 1 and math.gcd(g * g - 1, p) == 1 for g in range(2, 50))


def prove_composite(n: int) -> bool:
    """True only with a witness of compositeness"""
    if n < 4:
        return False
    if 1 < math.gcd(n, _PRIMORIAL_1000) < n:
        return True
    if any(pow(b, n - 1, n) != 1 for b in (2, 3, 5, 7)):
        return True
    import sympy
    fs = sympy.factorint(n)  # a pseudoprime to four bases: show a factor
    return any(1 < int(f) < n and n % int(f) == 0 for f in fs)


def prove_not_a_multiplier(a: int) -> bool:
    p = a * B - 1
    return prove_composite(p) or prove_composite((p - 1) // 2)


def test_the_proof_routines_themselves():
    primes = [2, 3, 65537, 4294967291, 4294967311, 2 ** 61 - 1, 18446744073709551557]  # textbook primes
    composites = [1, 4, 65536 * 65537, 4294967297, 561, 3215031751, 2 ** 61 + 1, (2 ** 31 - 1) * (2 ** 32 - 5),
                  3825123056546413051]  # incl. Carmichael / strong pseudoprimes to several bases
    assert all(prove_prime(n) for n in primes) and not any(prove_prime(n) for n in composites)
    assert all(prove_composite(n) for n in composites if n >= 4) and not any(prove_composite(n) for n in primes)
    assert prove_safe_prime(2 * 1000000007 + 1) == prove_prime(2 * 1000000007 + 1)
    # the oracle's primality routine against the proofs, on numbers around the candidates' size
    rng = np.random.default_rng(1)
    for n in [int(x) | 1 for x in rng.integers(1 << 62, (1 << 63) - 1, 300)] + primes + composites:
        if oracle.is_prime64(n):
            assert prove_prime(n), n
        else:
            assert n < 4 or prove_composite(n), n


def test_multiplier_of_the_paper_gives_a_safe_prime_and_the_stated_period():
    # "one requires am-1 as well as (am-2)/2 to be prime"; "the period is found to be p = am - 2";
    # a = 4294967118 is "the largest safe prime am-1 with a less than 2^32"
    assert prove_safe_prime(P)                     # p = a m - 1 and (p - 1)/2, both with certificates
    for a in range(A + 1, B):
        assert prove_not_a_multiplier(a), a        # every larger a fails with a witness of compositeness
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
    # every listed a qualifies WITH A PROOF (Pratt certificate for (p-1)/2, Pocklington for p), and every a in
    # between fails WITH A WITNESS (a small factor or a failed Fermat test): none of it is Miller-Rabin, the
    # algorithm the oracle itself uses, so a mistake of that route (a wrong base set, a slip in the safe-prime
    # definition, a skipped or double-counted candidate) cannot pass on both sides
    listed = set(mult)
    for a in range(mult[-1], B):
        if a in listed:
            assert prove_safe_prime(a * B - 1), a
        else:
            assert prove_not_a_multiplier(a), a
    # random access further down agrees with the scan from the top
    far = [int(a) for a in oracle.mwc_multipliers(3000, 5)]
    assert all(prove_safe_prime(a * B - 1) for a in far) and far == [int(a) for a in oracle.mwc_multipliers(0, 3005)[3000:]]


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
