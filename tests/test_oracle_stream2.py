"""Pins of the oracle's stream-spec v2 mode (R3', S15): one Philox4x32-10 block per pair of
same-colour sites.  All -m "not gpu".

What can go wrong in v2 and which test catches it:
  wrong words for the second site of a pair / wrong partner counter   -> test_word_selection (against the KAT-pinned
                                                                         Philox routine and the threshold table)
  first site of a pair no longer draws what v1 draws                   -> test_first_site_of_a_pair_is_v1
  the chain no longer samples the Boltzmann distribution               -> exact 4x4 moments (brute-force density of
     (e.g. correlated acceptance inside a pair)                           states), Kaufman's exact Ising energy at L = 32
  bookkeeping / threading                                              -> invariants
"""
import math

import numpy as np
import pytest

import exact_physics as ep
import oracle
import workloads


def _binned_mean_err(x, nblocks=50):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nblocks) * nblocks
    b = x[:n].reshape(nblocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nblocks)


def test_first_site_of_a_pair_is_v1():
    rng = np.random.default_rng(1)
    for _ in range(300):
        q = int(rng.integers(2, 40))
        i, k = int(rng.integers(0, 500)), 2 * int(rng.integers(0, 250))        # k even: first of its pair
        c = int(rng.integers(0, 2))
        j = 2 * k + ((i + c) & 1)
        nb = [int(x) for x in rng.integers(0, q, 4)]
        args = (i, j, int(rng.integers(0, 2 ** 32)), c, int(rng.integers(0, 2 ** 63)), q, float(rng.uniform(0.3, 2.0)),
                int(rng.integers(0, q)), nb)
        assert oracle.update_site(*args, stream=2) == oracle.update_site(*args, stream=1)


def test_word_selection_for_the_second_site_of_a_pair():
    rng = np.random.default_rng(2)
    for _ in range(300):
        q = int(rng.integers(2, 40))
        i, k = int(rng.integers(0, 500)), 2 * int(rng.integers(0, 250)) + 1    # k odd: second of its pair
        c = int(rng.integers(0, 2))
        j = 2 * k + ((i + c) & 1)
        t, seed = int(rng.integers(0, 2 ** 32)), int(rng.integers(0, 2 ** 63))
        w = oracle.philox4x32_10([j - 2, i, t, c], [seed & 0xFFFFFFFF, seed >> 32])   # the partner's v1 block
        prop = (w[2] * q) >> 32
        # accept-all temperature: the new spin IS the proposal, drawn from word 2
        assert oracle.update_site(i, j, t, c, seed, q, 1e15, 0, [0, 0, 0, 0], stream=2) == prop
        # d = 4 (four equal neighbours, proposal different): accepted iff word 3 < thr(4)
        if prop != 0:
            T = float(rng.uniform(1.0, 8.0))
            want = prop if w[3] < oracle.thresholds(T)[3] else 0
            assert oracle.update_site(i, j, t, c, seed, q, T, 0, [0, 0, 0, 0], stream=2) == want


@pytest.mark.parametrize("q,T,seed", [(2, 1.0, 31), (3, 0.99497262208, 32), (3, 1.5, 33)])
def test_long_run_moments_match_the_4x4_partition_function(q, T, seed):
    want_E, want_E2 = ep.moments_from_dos(ep.dos_4x4(q), T)
    o = oracle.OraclePotts(4, q, seed, oracle.INIT_RANDOM, stream=2)
    o.sweep(T, 200_000)
    E, _ = o.sweep_measured(T, 2_000_000, 1, hist=False)
    m1, e1 = _binned_mean_err(E)
    m2, e2 = _binned_mean_err(E.astype(np.float64) ** 2)
    assert abs(m1 - want_E) < 4 * e1, (m1, want_E, e1)
    assert abs(m2 - want_E2) < 4 * e2, (m2, want_E2, e2)
    assert e1 < 0.03


def test_q2_energy_matches_exact_ising():
    L, T = 32, 1.0
    want_E, want_var = ep.potts2_exact_moments(L, T)
    o = oracle.OraclePotts(L, 2, 41, oracle.INIT_ORDERED, stream=2)
    o.sweep(T, 5_000)
    E, _ = o.sweep_measured(T, 60_000, 1, hist=False)
    m1, e1 = _binned_mean_err(E)
    assert abs(m1 - want_E) < 4 * e1, (m1, want_E, e1)
    v, ev = _binned_mean_err((E.astype(np.float64) - want_E) ** 2)
    assert abs(v - want_var) < 4 * ev, (v, want_var, ev)


def test_invariants_threads_split_and_golden(golden_dir):
    T = 0.99 * workloads.t_c(9)
    a = oracle.OraclePotts(64, 9, 5, oracle.INIT_RANDOM, stream=2)
    b = oracle.OraclePotts(64, 9, 5, oracle.INIT_RANDOM, threads=4, stream=2)
    Ea, Ha = a.sweep_measured(T, 30, 1, hist=True)               # raises if E_inc != E or sum(hist) != L^2
    b.sweep(T, 13)
    b.sweep(T, 17)
    assert (a.spins() == b.spins()).all() and Ea[-1] == b.energy()
    v1 = oracle.OraclePotts(64, 9, 5, oracle.INIT_RANDOM)
    assert (v1.sweep_measured(T, 30, 1, hist=False)[0] != Ea).any()     # v2 really is another chain
    with pytest.raises(ValueError):
        oracle.OraclePotts(6, 3, 1, oracle.INIT_RANDOM, stream=2)        # L % 4 != 0
    # regression record written by tests/golden/make_stream2_golden.py (oracle only)
    case = None
    for line in open(f"{golden_dir}/trajectories_stream2.txt"):
        tok = line.split()
        if not tok or tok[0].startswith("#"):
            continue
        if tok[0] == "case":
            case = (int(tok[1]), int(tok[2]), int(tok[3]), oracle.INIT_RANDOM if tok[4] == "random" else oracle.INIT_ORDERED, float(tok[5]))
        elif tok[0] == "E":
            L, q, seed, init, f = case
            o = oracle.OraclePotts(L, q, seed, init, stream=2)
            t = 0
            for item in tok[1:]:
                at, want = item.split(":")
                o.sweep(f * workloads.t_c(q), int(at) - t)
                t = int(at)
                assert o.energy() == int(want), (case, at)


def test_stream2_sweep_is_the_site_rule_applied_in_checkerboard_order():
    """Pins the stream-2 branch of the oracle's half_sweep (which word and which partner counter each site of a
    full sweep takes): one sweep rebuilt site by site with oracle.update_site(stream=2) -- itself pinned above
    against the KAT-pinned Philox routine -- must equal OraclePotts(stream=2).sweep.  L % 4 == 0, several q, and a
    temperature at which many proposals are rejected, so a wrong word shows up as a different accept decision."""
    for L, q, seed, f in ((16, 7, 9, 0.9), (8, 3, 42, 0.7), (12, 24, 5, 1.0)):
        T = f * workloads.t_c(q)
        o = oracle.OraclePotts(L, q, seed, oracle.INIT_RANDOM, stream=2)
        o.sweep(T, 3)
        before, t = o.spins(), o.t
        o.sweep(T, 1)
        after = o.spins()
        mid = before.copy()
        rejected = 0
        for colour in (0, 1):
            src = mid.copy()
            for i in range(L):
                for j in range(L):
                    if (i + j) % 2 == colour:
                        nb = [src[(i - 1) % L, j], src[(i + 1) % L, j], src[i, (j - 1) % L], src[i, (j + 1) % L]]
                        mid[i, j] = oracle.update_site(i, j, t, colour, seed, q, T, src[i, j], nb, stream=2)
                        # what the site would have taken had every proposal been accepted
                        rejected += int(oracle.update_site(i, j, t, colour, seed, q, 1e15, src[i, j], nb, stream=2) != mid[i, j])
        assert (mid == after).all()
        assert rejected > L * L // 8                    # the case does exercise the acceptance word
        # and the stream-1 chain from the same state is a different one
        o1 = oracle.OraclePotts(L, q, seed, oracle.INIT_RANDOM, stream=1)
        o1.set_state(before, t)
        o1.sweep(T, 1)
        assert (o1.spins() != after).any()


def test_stream2_sweep_from_the_philox_words():
    """The same sweep once more from the definition R3' itself: Philox words through the KAT-pinned routine,
    thresholds through the P2-pinned routine, word (0,1) for even k, (2,3) of the partner's block for odd k."""
    L, q, seed = 8, 5, 77
    T = 0.8 * workloads.t_c(q)
    thr = oracle.thresholds(T)
    o = oracle.OraclePotts(L, q, seed, oracle.INIT_RANDOM, stream=2)
    o.sweep(T, 2)
    s, t = o.spins().astype(int), o.t
    o.sweep(T, 1)
    for colour in (0, 1):
        src = s.copy()
        for i in range(L):
            for j in range(L):
                if (i + j) % 2 != colour:
                    continue
                k = j >> 1
                jb = j if k % 2 == 0 else j - 2
                w = oracle.philox4x32_10([jb, i, t, colour], [seed & 0xFFFFFFFF, seed >> 32])
                w_prop, w_acc = (w[0], w[1]) if k % 2 == 0 else (w[2], w[3])
                new = (w_prop * q) >> 32
                nb = [src[(i - 1) % L, j], src[(i + 1) % L, j], src[i, (j - 1) % L], src[i, (j + 1) % L]]
                d = sum(x == src[i, j] for x in nb) - sum(x == new for x in nb)
                if d <= 0 or w_acc < thr[d - 1]:
                    s[i, j] = new
    assert (s == o.spins()).all()
