"""Pins of the 3D oracle (oracle/potts3d_oracle.c, reading S16).  All -m "not gpu".

What can go wrong and which test catches it:
  wrong sign / acceptance rule / proposal, a neighbour dropped or counted twice  -> exact 2x2x2 enumeration (Boltzmann moments)
  wrong number of neighbours or a wrong wrap at a larger L                       -> single-bond high-temperature energy at L = 8
  energy bookkeeping, update reading the wrong plane                             -> E_inc == recount with numpy rolls (test-side definition)
  counter layout (x, y, t, colour + 4 z), init domain, threshold table           -> site-by-site rebuild from the KAT-pinned Philox
  threshold expression                                                           -> thresholds3 == floor(2^32 exp(-d/T)) in 50-digit arithmetic
"""
import itertools
import math

import numpy as np

import oracle
import workloads


def _recount(s):
    """Eq. 1 on the cubic lattice, written with rolls: E = -(# equal nearest-neighbour pairs), each bond once."""
    return -int(sum((s == np.roll(s, -1, axis=a)).sum() for a in range(3)))


def _binned(x, nblocks=50):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nblocks) * nblocks
    b = x[:n].reshape(nblocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nblocks)


def test_thresholds3_against_high_precision():
    import mpmath
    mpmath.mp.dps = 50
    for T in (0.3, 0.7177, 1.0, 1.8163, 2.5, 40.0):
        thr = oracle.thresholds3(T)
        for d in range(1, 7):
            exact = mpmath.floor(mpmath.mpf(2) ** 32 * mpmath.exp(-mpmath.mpf(d) / mpmath.mpf(T)))
            assert abs(thr[d - 1] - int(exact)) <= 1          # libm exp is within an ulp of the true value
        assert thr == sorted(thr, reverse=True)
    assert oracle.thresholds3(0.5)[:4] == oracle.thresholds(0.5)          # the 2D table is its prefix


def test_exact_enumeration_2x2x2():
    """Boltzmann moments of the 2 x 2 x 2 periodic lattice (every neighbour pair is a double bond there) by brute
    force over all q^8 states, against the chain's long-run <E>, <E^2> within 4 sigma."""
    L = 2
    for q, T, seed in ((2, 3.0, 1), (3, 2.0, 2), (3, 5.0, 3)):
        Z = m1 = m2 = 0.0
        for state in itertools.product(range(q), repeat=L ** 3):
            s = np.array(state, dtype=np.uint8).reshape(L, L, L)
            E = _recount(s)
            w = math.exp(-E / T)
            Z += w; m1 += w * E; m2 += w * E * E
        m1 /= Z; m2 /= Z
        o = oracle.OraclePotts3D(L, q, seed, oracle.INIT_RANDOM)
        o.sweep(T, 20000)
        E, _ = o.sweep_measured(T, 400000, 1, hist=False)
        e1, s1 = _binned(E)
        e2, s2 = _binned(E.astype(np.float64) ** 2)
        assert abs(e1 - m1) < 4 * s1, (q, T, e1, m1, s1)
        assert abs(e2 - m2) < 4 * s2, (q, T, e2, m2, s2)


def test_high_temperature_energy_is_the_single_bond_value():
    """At K = 1/T << 1 the energy per bond is that of an isolated bond, e^K / (e^K + q - 1), up to terms of the order of
    v^3 with v = (e^K - 1)/(e^K + q - 1) (the shortest loop of the cubic lattice has four bonds): 3 bonds per site."""
    L, q, T = 8, 3, 12.0
    K = 1.0 / T
    per_bond = math.exp(K) / (math.exp(K) + q - 1)
    v = (math.exp(K) - 1) / (math.exp(K) + q - 1)
    o = oracle.OraclePotts3D(L, q, 4, oracle.INIT_RANDOM, threads=4)
    o.sweep(T, 200)
    E, _ = o.sweep_measured(T, 6000, 1, hist=False)
    e, err = _binned(E / (3.0 * L ** 3))
    assert abs(-e - per_bond) < 4 * err + 8 * v ** 3, (e, per_bond, err, v ** 3)
    assert err < 2e-3 and abs(per_bond - 1.0 / q) > 10 * err       # the test resolves the temperature dependence


def test_invariants_and_threads():
    for L, q, T in ((4, 2, 2.2), (6, 9, 1.4), (8, 24, 0.9)):
        a = oracle.OraclePotts3D(L, q, 7, oracle.INIT_RANDOM)
        b = oracle.OraclePotts3D(L, q, 7, oracle.INIT_RANDOM, threads=4)
        assert a.energy() == _recount(a.spins())
        Ea, Ha = a.sweep_measured(T, 12, 1)
        for k in range(3):
            b.sweep(T, 4)
        assert (a.spins() == b.spins()).all() and a.t == b.t == 12
        assert a.energy_incremental() == a.energy() == _recount(a.spins()) == int(Ea[-1])
        assert (Ha.sum(axis=1) == L ** 3).all()
        assert (Ha[-1] == np.bincount(a.spins().ravel(), minlength=q)).all()
        c = oracle.OraclePotts3D(L, q, 7, oracle.INIT_ORDERED)
        c.set_state(a.spins(), a.t)
        a.sweep(T, 3); c.sweep(T, 3)
        assert (a.spins() == c.spins()).all()


def test_degenerate_temperatures_3d():
    L, q = 6, 5
    o = oracle.OraclePotts3D(L, q, 1, oracle.INIT_ORDERED)
    assert o.energy() == -3 * L ** 3                                # ordered: every bond satisfied
    E, H = o.sweep_measured(0.01, 20, 1)
    assert (E == -3 * L ** 3).all() and (H[:, 0] == L ** 3).all()   # T -> 0: frozen
    r = oracle.OraclePotts3D(L, q, 2, oracle.INIT_RANDOM)
    E, _ = r.sweep_measured(0.01, 30, 1, hist=False)
    assert (np.diff(E) <= 0).all()                                  # only d <= 0 is accepted
    h = oracle.OraclePotts3D(8, 4, 3, oracle.INIT_ORDERED, threads=4)
    E, H = h.sweep_measured(1e9, 40, 1)                             # T -> infinity: every proposal accepted
    assert abs(E[5:].mean() / (3 * 8 ** 3) + 1.0 / 4) < 0.02
    assert abs(H[5:].mean(axis=0) / 8 ** 3 - 0.25).max() < 0.02


def test_sweep_rebuilt_site_by_site_from_the_philox_words():
    """R2', R3', R9': colour order, counter (x, y, t, colour + 4 z), init counter (x, y, 0, 2 + 4 z), through the
    KAT-pinned Philox routine and the threshold table."""
    L, q, seed = 4, 5, (9 << 32) | 77
    key = [seed & 0xFFFFFFFF, seed >> 32]
    T = 1.3
    thr = oracle.thresholds3(T)
    o = oracle.OraclePotts3D(L, q, seed, oracle.INIT_RANDOM)
    s = np.zeros((L, L, L), dtype=int)
    for z, y, x in itertools.product(range(L), repeat=3):
        s[z, y, x] = (oracle.philox4x32_10([x, y, 0, 2 + 4 * z], key)[0] * q) >> 32
    assert (s == o.spins()).all()
    rejected = 0
    for t in range(2):
        for colour in (0, 1):
            src = s.copy()
            for z, y, x in itertools.product(range(L), repeat=3):
                if (x + y + z) % 2 != colour:
                    continue
                w = oracle.philox4x32_10([x, y, t, colour + 4 * z], key)
                new = (w[0] * q) >> 32
                nb = [src[z, y, (x - 1) % L], src[z, y, (x + 1) % L], src[z, (y - 1) % L, x], src[z, (y + 1) % L, x],
                      src[(z - 1) % L, y, x], src[(z + 1) % L, y, x]]
                d = sum(v == src[z, y, x] for v in nb) - sum(v == new for v in nb)
                if d <= 0 or w[1] < thr[d - 1]:
                    s[z, y, x] = new
                else:
                    rejected += 1
        o.sweep(T, 1)
        assert (s == o.spins()).all(), t
    assert rejected > 10
