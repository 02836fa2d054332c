"""Exact references for the 2D Ising ferromagnet on a periodic L x L lattice.

Test helper (not product, not oracle).  Two independent routes:

* ``brute_force(L, beta)``: enumerate all 2^(L*L) states (L = 4 only).
* ``kaufman(L, beta)``: Kaufman's closed form for the finite torus, the formula
  behind the "exact" row of the paper's Table 1 (Ref.[9]):

      Z = 1/2 (2 sinh 2K)^(N/2) (Z1 + Z2 + Z3 + Z4),   K = beta, N = L*L
      Z1 = prod_{r<L} 2 cosh(L g_{2r+1}/2)   Z2 = prod_{r<L} 2 sinh(L g_{2r+1}/2)
      Z3 = prod_{r<L} 2 cosh(L g_{2r}/2)     Z4 = prod_{r<L} 2 sinh(L g_{2r}/2)
      cosh g_l = cosh 2K coth 2K - cos(l pi / L),  g_0 = 2K + ln tanh K  (signed)

  evaluated with mpmath at 60 digits; e = -(1/N) d ln Z / d beta and
  C_V = (beta^2 / N) d^2 ln Z / d beta^2 by mpmath's numerical differentiation.
"""
from __future__ import annotations

import numpy as np


def energies_all_states(L: int = 4) -> np.ndarray:
    """E = -sum_<ij> s_i s_j for every state; bit i of the state index = spin i up."""
    N = L * L
    idx = np.arange(1 << N, dtype=np.uint32)
    s = ((idx[:, None] >> np.arange(N, dtype=np.uint32)[None, :]) & 1).astype(np.int8) * 2 - 1
    s = s.reshape(-1, L, L)
    E = -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2)) - (s * np.roll(s, -1, axis=1)).sum(axis=(1, 2))
    return E.astype(np.int64)


def brute_force(L: int, beta: float):
    E = energies_all_states(L)
    w = np.exp(-beta * E.astype(np.float64))
    Z = w.sum()
    N = L * L
    m1 = (w * E).sum() / Z
    m2 = (w * E * E).sum() / Z
    dos = {int(e): int(c) for e, c in zip(*np.unique(E, return_counts=True))}
    return {"Z": float(Z), "e": float(m1 / N), "cv": float(beta * beta * (m2 - m1 * m1) / N), "dos": dos}


def _lnZ(L, K):
    import mpmath as mp

    N = L * L
    c = mp.cosh(2 * K) * mp.coth(2 * K)

    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))
        return mp.acosh(c - mp.cos(l * mp.pi / L))

    # products in logs, factoring out the largest term
    ln = [mp.mpf(0)] * 4
    sign = [1, 1, 1, 1]
    for r in range(L):
        go, ge = gamma(2 * r + 1), gamma(2 * r)
        ln[0] += mp.log(2 * mp.cosh(L * go / 2))
        ln[1] += mp.log(2 * mp.sinh(L * go / 2))
        ln[2] += mp.log(2 * mp.cosh(L * ge / 2))
        v = 2 * mp.sinh(L * ge / 2)
        if v < 0:
            sign[3] = -sign[3]
        ln[3] += mp.log(abs(v))
    m = max(ln)
    tot = sum(sg * mp.exp(x - m) for sg, x in zip(sign, ln))
    return -mp.log(2) + (mp.mpf(N) / 2) * mp.log(2 * mp.sinh(2 * K)) + m + mp.log(tot)


def kaufman(L: int, beta: float, digits: int = 60):
    import mpmath as mp

    with mp.workdps(digits):
        b = mp.mpf(repr(beta)) if not isinstance(beta, str) else mp.mpf(beta)
        N = L * L
        f = lambda k: _lnZ(L, k)
        d1 = mp.diff(f, b, 1, h=mp.mpf(10) ** (-digits // 4))
        d2 = mp.diff(f, b, 2, h=mp.mpf(10) ** (-digits // 4))
        return {"lnZ": float(f(b)), "e": float(-d1 / N), "cv": float(b * b * d2 / N)}
