"""Pins of the first + second neighbour oracle (oracle/potts8_oracle.c, reading S17).  -m "not gpu".

What can go wrong and which test catches it:
  wrong sign / acceptance rule / proposal, a neighbour dropped or counted twice   -> exact 3x3 enumeration (complete graph on 9 sites)
  wrong number of neighbours or a wrong wrap at a larger L                        -> single-bond high-temperature energy at L = 24
  bookkeeping, an update that reads a site of its own sub-network                 -> E_inc == recount with numpy rolls (test-side definition)
  sub-network order 0..8, counter (j, i, t, 16 + c), init domain, thresholds      -> site-by-site rebuild from the KAT-pinned Philox
"""
import itertools
import math

import numpy as np

import oracle


def _recount(s):
    """E = -(# equal pairs over first and second neighbours), each bond once: 4 directions per site."""
    e = 0
    for di, dj in ((0, 1), (1, 0), (1, 1), (1, -1)):
        e += int((s == np.roll(np.roll(s, -di, axis=0), -dj, axis=1)).sum())
    return -e


def _binned(x, nblocks=50):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nblocks) * nblocks
    b = x[:n].reshape(nblocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nblocks)


def test_thresholds8():
    for T in (0.5, 1.0, 2.5):
        thr = oracle.thresholds8(T)
        assert thr[:4] == oracle.thresholds(T) and thr[:6] == oracle.thresholds3(T)
        assert thr == [int(math.floor(math.ldexp(math.exp(-d / T), 32))) for d in range(1, 9)]


def test_exact_enumeration_3x3():
    L = 3
    for q, T, seed in ((2, 4.0, 1), (3, 3.0, 2), (3, 8.0, 3)):
        Z = m1 = m2 = 0.0
        for state in itertools.product(range(q), repeat=L * L):
            E = _recount(np.array(state, dtype=np.uint8).reshape(L, L))
            w = math.exp(-E / T)
            Z += w; m1 += w * E; m2 += w * E * E
        m1 /= Z; m2 /= Z
        o = oracle.OraclePotts8(L, q, seed, oracle.INIT_RANDOM)
        o.sweep(T, 20000)
        E, _ = o.sweep_measured(T, 400000, 1, hist=False)
        e1, s1 = _binned(E)
        e2, s2 = _binned(E.astype(np.float64) ** 2)
        assert abs(e1 - m1) < 4 * s1, (q, T, e1, m1, s1)
        assert abs(e2 - m2) < 4 * s2, (q, T, e2, m2, s2)


def test_high_temperature_energy_counts_four_bonds_per_site():
    """K = 1/T << 1: energy per bond = e^K / (e^K + q - 1) up to O(v^2) (triangles exist on this lattice),
    v = (e^K - 1)/(e^K + q - 1); 4 bonds per site."""
    L, q, T = 24, 3, 50.0
    K = 1.0 / T
    per_bond = math.exp(K) / (math.exp(K) + q - 1)
    v = (math.exp(K) - 1) / (math.exp(K) + q - 1)
    o = oracle.OraclePotts8(L, q, 4, oracle.INIT_RANDOM, threads=4)
    o.sweep(T, 100)
    E, _ = o.sweep_measured(T, 4000, 1, hist=False)
    e, err = _binned(E / (4.0 * L * L))
    assert abs(-e - per_bond) < 4 * err + 20 * v * v, (e, per_bond, err)
    assert err < 1e-3                       # a dropped or doubled neighbour direction would move e by 1/(4q) = 0.08


def test_invariants_and_threads_8():
    for L, q, T in ((6, 2, 3.0), (12, 9, 1.6), (24, 24, 1.2)):
        a = oracle.OraclePotts8(L, q, 7, oracle.INIT_RANDOM)
        b = oracle.OraclePotts8(L, q, 7, oracle.INIT_RANDOM, threads=4)
        assert a.energy() == _recount(a.spins())
        # the start state is the 2D model's (R9 unchanged)
        assert (a.spins() == oracle.OraclePotts(L, q, 7, oracle.INIT_RANDOM).spins()).all() if L % 2 == 0 else True
        Ea, Ha = a.sweep_measured(T, 12, 1)
        for k in range(3):
            b.sweep(T, 4)
        assert (a.spins() == b.spins()).all() and a.t == b.t == 12
        assert a.energy_incremental() == a.energy() == _recount(a.spins()) == int(Ea[-1])
        assert (Ha.sum(axis=1) == L * L).all()
        c = oracle.OraclePotts8(L, q, 7, oracle.INIT_ORDERED)
        c.set_state(a.spins(), a.t)
        a.sweep(T, 3); c.sweep(T, 3)
        assert (a.spins() == c.spins()).all()


def test_degenerate_temperatures_8():
    L, q = 12, 5
    o = oracle.OraclePotts8(L, q, 1, oracle.INIT_ORDERED)
    assert o.energy() == -4 * L * L
    E, H = o.sweep_measured(0.01, 20, 1)
    assert (E == -4 * L * L).all() and (H[:, 0] == L * L).all()
    r = oracle.OraclePotts8(L, q, 2, oracle.INIT_RANDOM)
    E, _ = r.sweep_measured(0.01, 30, 1, hist=False)
    assert (np.diff(E) <= 0).all()
    h = oracle.OraclePotts8(24, 4, 3, oracle.INIT_ORDERED, threads=4)
    E, H = h.sweep_measured(1e9, 60, 1)
    assert abs(E[5:].mean() / (4 * 24 * 24) + 0.25) < 0.02


def test_sweep_rebuilt_site_by_site_from_the_philox_words_8():
    L, q, seed = 6, 5, (3 << 32) | 41
    key = [seed & 0xFFFFFFFF, seed >> 32]
    T = 2.2
    thr = oracle.thresholds8(T)
    o = oracle.OraclePotts8(L, q, seed, oracle.INIT_RANDOM)
    s = np.zeros((L, L), dtype=int)
    for i, j in itertools.product(range(L), repeat=2):
        s[i, j] = (oracle.philox4x32_10([j, i, 0, 2], key)[0] * q) >> 32
    assert (s == o.spins()).all()
    rejected = 0
    for t in range(2):
        for c in range(9):
            a, b = divmod(c, 3)
            for i in range(a, L, 3):
                for j in range(b, L, 3):
                    w = oracle.philox4x32_10([j, i, t, 16 + c], key)
                    new = (w[0] * q) >> 32
                    nb = [s[(i + di) % L, (j + dj) % L] for di in (-1, 0, 1) for dj in (-1, 0, 1) if (di, dj) != (0, 0)]
                    d = sum(v == s[i, j] for v in nb) - sum(v == new for v in nb)
                    if d <= 0 or w[1] < thr[d - 1]:
                        s[i, j] = new
                    else:
                        rejected += 1
        o.sweep(T, 1)
        assert (s == o.spins()).all(), t
    assert rejected > 5
