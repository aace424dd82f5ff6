"""Exact results the oracle is pinned to.  Independent of oracle/ and of the CUDA path.

Nothing here simulates anything: these are closed forms and brute-force enumerations.

* ``dos_4x4(q)``            density of states g(M) of the 4x4 periodic Potts lattice by
                            enumerating all q^16 configurations (M = satisfied bonds, E = -M,
                            PAPER.md:46 Eq. 1).
* ``moments_from_dos``      <E>, <E^2> from Z = sum_M g(M) exp(M/T).
* ``kaufman_lnZ``           Kaufman's exact partition function of the m x n periodic Ising
                            lattice (B. Kaufman, Phys. Rev. 76, 1232 (1949)), used through the
                            q = 2 mapping J_Potts = 2 J_Ising (PAPER.md:238 footnote 3).
* ``onsager_energy_potts2`` Onsager's infinite-lattice internal energy in the same mapping.
* ``potts_tc`` / ``potts_eo_ed``  T_c (Eq. 2) and the ordered / disordered energies
                            at T_c (Eqs. 3, 6, with the garbled Eq. 3 read as in
                            DESIGN.md reading G1), checked against the paper's Table 2.
"""
from __future__ import annotations

import math

import mpmath as mp
import numpy as np


def dos_4x4(q: int) -> dict:
    """g(M) for the 4x4 periodic lattice; s[0] is fixed to 0 and the count multiplied by q."""
    n_free = 15
    total = q ** n_free
    g = np.zeros(33, dtype=np.int64)
    idx_right = [(r * 4 + (c + 1) % 4) for r in range(4) for c in range(4)]
    idx_down = [(((r + 1) % 4) * 4 + c) for r in range(4) for c in range(4)]
    chunk = 1 << 20
    for start in range(0, total, chunk):
        codes = np.arange(start, min(total, start + chunk), dtype=np.int64)
        s = np.zeros((codes.size, 16), dtype=np.uint8)
        c = codes.copy()
        for site in range(1, 16):
            s[:, site] = c % q
            c //= q
        M = (s == s[:, idx_right]).sum(axis=1) + (s == s[:, idx_down]).sum(axis=1)
        g += np.bincount(M, minlength=33)[:33]
    return {int(M): int(cnt) * q for M, cnt in enumerate(g) if cnt}


def moments_from_dos(g: dict, T: float):
    """(<E>, <E^2>) with E = -M, exact up to double rounding."""
    mp.mp.dps = 40
    Z = mp.mpf(0)
    s1 = mp.mpf(0)
    s2 = mp.mpf(0)
    for M, cnt in g.items():
        w = cnt * mp.e ** (mp.mpf(M) / mp.mpf(T))
        Z += w
        s1 += -M * w
        s2 += M * M * w
    return float(s1 / Z), float(s2 / Z)


def kaufman_lnZ(K, m: int, n: int):
    """ln Z of the m x n periodic Ising lattice, H = -J sum sigma sigma', K = J / T (mpmath)."""
    K = mp.mpf(K)
    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))
        c = mp.cosh(2 * K) * mp.coth(2 * K) - mp.cos(mp.pi * l / n)
        return mp.acosh(c)
    p1 = mp.mpf(1); p2 = mp.mpf(1); p3 = mp.mpf(1); p4 = mp.mpf(1)
    for r in range(n):
        go = gamma(2 * r + 1)
        ge = gamma(2 * r)
        p1 *= 2 * mp.cosh(m * go / 2)
        p2 *= 2 * mp.sinh(m * go / 2)
        p3 *= 2 * mp.cosh(m * ge / 2)
        p4 *= 2 * mp.sinh(m * ge / 2)
    Z = mp.mpf(0.5) * (2 * mp.sinh(2 * K)) ** (mp.mpf(m * n) / 2) * (p1 + p2 + p3 + p4)
    return mp.log(Z)


def potts2_exact_moments(L: int, T: float):
    """(<E>, Var E) of the q = 2 Potts model on the L x L periodic lattice.

    delta(s,s') = (1 + sigma sigma')/2, so H_Potts = -N + H_Ising(J_I = 1/2), K = 1/(2T):
    <E> = -N - (1/2) dlnZ/dK, Var E = (1/4) d^2 lnZ/dK^2.
    """
    mp.mp.dps = 60
    K0 = mp.mpf(1) / (2 * mp.mpf(T))
    f = lambda K: kaufman_lnZ(K, L, L)
    d1 = mp.diff(f, K0, 1)
    d2 = mp.diff(f, K0, 2)
    N = L * L
    return float(-N - d1 / 2), float(d2 / 4)


def onsager_energy_potts2(T: float) -> float:
    """Energy per spin of the q = 2 Potts model, L -> infinity (Onsager 1944, mapped J_I = 1/2)."""
    mp.mp.dps = 40
    K = mp.mpf(1) / (2 * mp.mpf(T))
    kappa = 2 * mp.sinh(2 * K) / mp.cosh(2 * K) ** 2
    u_over_J = -mp.coth(2 * K) * (1 + (2 / mp.pi) * (2 * mp.tanh(2 * K) ** 2 - 1) * mp.ellipk(kappa ** 2))
    return float(-1 + u_over_J / 2)


def potts_tc(q: int) -> float:
    return 1.0 / math.log(1.0 + math.sqrt(q))


def potts_eo_ed(q: int):
    """(e_o, e_d) at T_c for q > 4: Eq. 6 for the sum, Eq. 3 (Baxter) for the difference."""
    mp.mp.dps = 40
    theta = mp.acosh(mp.sqrt(q) / 2)
    prod = mp.mpf(1)
    for k in range(1, 400):
        prod *= mp.tanh(k * theta) ** 2
    latent = 2 * (1 + 1 / mp.sqrt(q)) * mp.tanh(theta / 2) * prod
    total = -2 * (1 + 1 / mp.sqrt(q))
    return float((total - latent) / 2), float((total + latent) / 2)
