"""Pins of the CPU oracle to things other than itself (CPU only, -m "not gpu").

Each test names the pin (P1..P10 of DESIGN.md section 4) and the rule(s) it would catch a
mistake in.  Expected values come from tests/golden/ (the paper's printed numbers and the
SURVEY's independently computed vectors) or from tests/exact_physics.py (closed forms and
brute-force enumeration); none come from oracle/ or from the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import exact_physics as ep
import oracle
import workloads
from oracle import observables as obs


def _lines(golden_dir, name):
    with open(os.path.join(golden_dir, name)) as f:
        return [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]


# ---------------------------------------------------------------- P1: Philox (R3)
def test_p1_philox_known_answers(golden_dir):
    rows = _lines(golden_dir, "philox_kat.txt")
    assert len(rows) == 3
    for ln in rows:
        v = [int(x, 16) for x in ln.split()]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


# ---------------------------------------------------------------- P2: thresholds, T_c (R6, S12)
def test_p2_thresholds_and_tc(golden_dir):
    for ln in _lines(golden_dir, "thresholds.txt"):
        q, f, T, *thr = ln.split()
        q, f, T = int(q), float(f), float(T)
        assert f * workloads.t_c(q) == T            # same double as the survey's program
        assert oracle.thresholds(T) == [int(x) for x in thr]
    # thresholds are floor(2^32 p): check against an independent high-precision evaluation
    import mpmath as mp
    mp.mp.dps = 50
    for T in (0.3, 0.7141340452400369, 1.0, 2.5, 40.0):
        want = [int(mp.floor(mp.mpf(2) ** 32 * mp.e ** (-mp.mpf(d) / mp.mpf(T)))) for d in range(1, 5)]
        got = oracle.thresholds(T)
        # libm exp is not correctly rounded: allow the last unit, demand monotone decrease
        assert all(abs(a - b) <= 1 for a, b in zip(got, want))
        assert got[0] >= got[1] >= got[2] >= got[3]


def test_paper_printed_tc(golden_dir):
    vals = {}
    for ln in _lines(golden_dir, "paper_constants.txt"):
        p = ln.split()
        if p[0] != "table2":
            vals[p[0]] = float(p[1])
    assert math.floor(workloads.t_c(6) * 1e7) / 1e7 == vals["Tc_q6"]       # "0.8076068..."
    assert math.floor(workloads.t_c(2) * 1e7) / 1e7 == vals["Tc_q2"]       # "1.1345926..."
    assert vals["Tmin_profile_q9"] < workloads.t_c(9) < vals["Tmax_profile_q9"] + 1e-6
    assert ep.potts_tc(9) == workloads.t_c(9)


def test_exact_helpers_reproduce_paper_table2(golden_dir):
    """Validates tests/exact_physics (not the oracle): Table 2's exact columns."""
    for ln in _lines(golden_dir, "paper_constants.txt"):
        p = ln.split()
        if p[0] == "table2":
            q, eo, ed = int(p[1]), float(p[2]), float(p[3])
            got_eo, got_ed = ep.potts_eo_ed(q)
            assert abs(-got_eo - eo) < 1.1e-6 and abs(-got_ed - ed) < 1.1e-6


# ---------------------------------------------------------------- P3: exact enumeration 4x4
@pytest.fixture(scope="module")
def dos(golden_dir):
    table = {}
    for ln in _lines(golden_dir, "dos_4x4.txt"):
        q, *items = ln.split()
        table[int(q)] = {int(a.split(":")[0]): int(a.split(":")[1]) for a in items}
    return table


def test_p3_dos_fixture_matches_brute_force(dos):
    for q in (2, 3):
        g = ep.dos_4x4(q)
        assert g == dos[q]
        assert sum(g.values()) == q ** 16


def _binned_mean_err(x, nblocks=50):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nblocks) * nblocks
    b = x[:n].reshape(nblocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nblocks)


@pytest.mark.parametrize("q,T,seed", [(2, 1.0, 11), (2, 2.0, 12), (3, 0.8, 13),
                                      (3, 0.99497262208, 14), (3, 1.5, 15)])
def test_p3_long_run_moments_match_partition_function(dos, q, T, seed):
    """R1, R2, R4-R7: the chain samples the Boltzmann distribution of the 4x4 lattice."""
    want_E, want_E2 = ep.moments_from_dos(dos[q], T)
    o = oracle.OraclePotts(4, q, seed, oracle.INIT_RANDOM)
    o.sweep(T, 200_000)                                   # burn-in, 10 %
    E, _ = o.sweep_measured(T, 2_000_000, 1, hist=False)
    m1, e1 = _binned_mean_err(E)
    m2, e2 = _binned_mean_err(E.astype(np.float64) ** 2)
    assert abs(m1 - want_E) < 4 * e1, (m1, want_E, e1)
    assert abs(m2 - want_E2) < 4 * e2, (m2, want_E2, e2)
    assert e1 < 0.03                                       # the test has resolving power


# ---------------------------------------------------------------- P4: Onsager / Kaufman (q = 2)
def test_p4_kaufman_helper_is_exact_on_4x4(dos):
    for T in (1.0, 2.0):
        E, var = ep.potts2_exact_moments(4, T)
        want_E, want_E2 = ep.moments_from_dos(dos[2], T)
        assert abs(E - want_E) < 1e-10 and abs(var + E * E - want_E2) < 1e-8


def test_p4_onsager_limit_values():
    # SURVEY 8(c) P4 values; e(T_c) = -(1 + 1/sqrt 2) also follows from PAPER.md:67 Eq. 6
    for T, want in ((0.9, -1.929651902863), (1.0, -1.872782287656), (1.3, -1.514146819005),
                    (1.5, -1.408654796251), (2.0, -1.278636120314)):
        assert abs(ep.onsager_energy_potts2(T) - want) < 1e-11
    assert abs(ep.onsager_energy_potts2(workloads.t_c(2)) + (1 + 1 / math.sqrt(2))) < 1e-7
    for T in (1.0, 1.3):                                   # finite-size shift < 1e-7 at L = 64
        assert abs(ep.potts2_exact_moments(64, T)[0] / 4096 - ep.onsager_energy_potts2(T)) < 1e-7


@pytest.mark.parametrize("T,seed,init", [(1.0, 21, oracle.INIT_ORDERED), (1.3, 22, oracle.INIT_RANDOM)])
def test_p4_q2_energy_and_fluctuations_match_exact_ising(T, seed, init):
    """R1-R7 at scale: L = 32, q = 2 against Kaufman's exact finite-lattice <E> and Var E."""
    L = 32
    want_E, want_var = ep.potts2_exact_moments(L, T)
    o = oracle.OraclePotts(L, 2, seed, init)
    o.sweep(T, 5_000)
    E, _ = o.sweep_measured(T, 60_000, 1, hist=False)
    m1, e1 = _binned_mean_err(E)
    assert abs(m1 - want_E) < 4 * e1, (m1, want_E, e1)
    assert e1 / (L * L) < 5e-4
    dev2 = (E.astype(np.float64) - want_E) ** 2
    v, ev = _binned_mean_err(dev2)
    assert abs(v - want_var) < 4 * ev, (v, want_var, ev)
    # and against the infinite-lattice Onsager value (finite-size shift is below the error bar)
    assert abs(m1 / (L * L) - ep.onsager_energy_potts2(T)) < 4 * e1 / (L * L) + 1e-5


# ---------------------------------------------------------------- P5: T_c as specific-heat peak drift
def test_p5_specific_heat_peak_drifts_to_tc():
    """q = 2: exact finite-L C_v peaks approach T_c = 1/ln(1+sqrt 2) as L grows (PAPER.md:52,
    :225), and the oracle's measured C_v follows the exact L = 8 and L = 16 curves, peak included."""
    Tc = workloads.t_c(2)
    grid = [Tc * f for f in (0.92, 0.97, 1.02, 1.07, 1.12, 1.20)]

    def exact_cv(L, T):
        return ep.potts2_exact_moments(L, T)[1] / (L * L * T * T)

    peaks = {}
    for L in (4, 8, 16, 32):
        fine = np.linspace(0.9 * Tc, 1.35 * Tc, 91)
        peaks[L] = fine[int(np.argmax([exact_cv(L, T) for T in fine]))]
    d = [abs(peaks[L] - Tc) for L in (4, 8, 16, 32)]
    assert d[0] > d[1] > d[2] > d[3] and d[3] < 0.03 * Tc

    for L, nsw in ((8, 300_000), (16, 200_000)):
        measured, exact = [], []
        for k, T in enumerate(grid):
            o = oracle.OraclePotts(L, 2, 100 + 10 * L + k, oracle.INIT_RANDOM)
            o.sweep(T, 5_000)
            E, _ = o.sweep_measured(T, nsw, 1, hist=False)
            want_E, want_var = ep.potts2_exact_moments(L, T)
            v, ev = _binned_mean_err((E.astype(np.float64) - want_E) ** 2)
            assert abs(v - want_var) < 4.5 * ev, (L, T, v, want_var, ev)
            cv = obs.specific_heat(E, L * L, T)
            measured.append(cv)
            exact.append(want_var / (L * L * T * T))
            assert abs(cv - exact[-1]) < 0.06 * exact[-1]
        assert int(np.argmax(measured)) == int(np.argmax(exact))


# ---------------------------------------------------------------- P6: bookkeeping invariants (R7, R8)
@pytest.mark.parametrize("L,q,init,f", [(16, 6, oracle.INIT_RANDOM, 0.9), (32, 9, oracle.INIT_ORDERED, 1.05),
                                        (2, 5, oracle.INIT_RANDOM, 1.0), (6, 256, oracle.INIT_RANDOM, 1.0)])
def test_p6_incremental_energy_and_histogram_sum(L, q, init, f):
    o = oracle.OraclePotts(L, q, 5, init)
    assert o.energy() == o.energy_incremental()
    E, H = o.sweep_measured(f * workloads.t_c(q), 200, 1)       # raises if an invariant breaks
    assert (H.sum(axis=1) == L * L).all()
    assert o.energy() == E[-1] == o.energy_incremental()
    s = o.spins()
    # Eq. 1 recomputed with numpy rolls (an independent expression of the same sum)
    bonds = int((s == np.roll(s, -1, axis=1)).sum() + (s == np.roll(s, -1, axis=0)).sum())
    assert E[-1] == -bonds
    assert (np.bincount(s.ravel(), minlength=q) == H[-1]).all()
    assert s.max() < q


def test_p6_sweep_split_and_restart_and_threads():
    T = 0.99 * workloads.t_c(9)
    a = oracle.OraclePotts(32, 9, 3, oracle.INIT_RANDOM)
    b = oracle.OraclePotts(32, 9, 3, oracle.INIT_RANDOM)
    c = oracle.OraclePotts(32, 9, 3, oracle.INIT_RANDOM, threads=4)
    a.sweep(T, 30)
    b.sweep(T, 11); b.sweep(T, 19)
    c.sweep(T, 30)
    assert (a.spins() == b.spins()).all() and a.t == b.t == 30
    assert (a.spins() == c.spins()).all() and a.energy_incremental() == c.energy_incremental()
    d = oracle.OraclePotts(32, 9, 3, oracle.INIT_ORDERED)
    d.set_state(b.spins(), b.t)
    a.sweep(T, 7); d.sweep(T, 7)
    assert (a.spins() == d.spins()).all()
    # a different seed or a shifted sweep counter gives a different trajectory
    e = oracle.OraclePotts(32, 9, 4, oracle.INIT_RANDOM)
    assert (e.spins() != oracle.OraclePotts(32, 9, 3, oracle.INIT_RANDOM).spins()).any()


def test_update_site_matches_full_sweep():
    """oracle_update_site (used by the full-size sampled GPU checks) is the same rule as the sweep."""
    L, q, seed = 16, 7, 9
    T = 1.01 * workloads.t_c(q)
    o = oracle.OraclePotts(L, q, seed, oracle.INIT_RANDOM)
    o.sweep(T, 3)
    before = o.spins()
    t = o.t
    o.sweep(T, 1)
    after = o.spins()
    mid = before.copy()
    for colour in (0, 1):
        src = mid.copy()
        for i in range(L):
            for j in range(L):
                if (i + j) % 2 == colour:
                    nb = [src[(i - 1) % L, j], src[(i + 1) % L, j], src[i, (j - 1) % L], src[i, (j + 1) % L]]
                    mid[i, j] = oracle.update_site(i, j, t, colour, seed, q, T, src[i, j], nb)
    assert (mid == after).all()


# ---------------------------------------------------------------- P7: degenerate temperatures (R6)
def test_p7_zero_temperature_limit():
    L, q = 32, 6
    assert oracle.thresholds(0.01) == [0, 0, 0, 0]
    o = oracle.OraclePotts(L, q, 1, oracle.INIT_ORDERED)
    E, H = o.sweep_measured(0.01, 50, 1)
    assert (E == -2 * L * L).all() and (H[:, 0] == L * L).all() and (H[:, 1:] == 0).all()
    o = oracle.OraclePotts(L, q, 2, oracle.INIT_RANDOM)
    E0 = o.energy()
    E, _ = o.sweep_measured(0.01, 100, 1)
    assert E[0] <= E0 and (np.diff(E) <= 0).all()


def test_p7_infinite_temperature_limit():
    L, q = 64, 8
    T = 1e12
    assert all(t >= 2 ** 32 - 2 for t in oracle.thresholds(T))
    o = oracle.OraclePotts(L, q, 3, oracle.INIT_ORDERED)
    E, H = o.sweep_measured(T, 400, 1)
    e = E[20:].mean() / (L * L)
    # i.i.d. uniform spins: <e> = -2/q, Var(E) = 2N (1/q)(1 - 1/q)
    se = math.sqrt(2 * (1 / q) * (1 - 1 / q) / (L * L) / 380)
    assert abs(e + 2 / q) < 5 * se
    assert abs(H[20:].mean(axis=0) - L * L / q).max() < 5 * math.sqrt(L * L / q / 380) + 1


# ---------------------------------------------------------------- P8: proposal uniformity (R4, R9)
@pytest.mark.parametrize("q", [6, 9, 24, 256])
def test_p8_proposal_uniformity(q):
    L = 2048
    o = oracle.OraclePotts(L, q, 77, oracle.INIT_RANDOM)       # R9 uses the same mulhi(w0, q)
    h = o.histogram().astype(np.float64)
    exp = L * L / q
    chi2 = ((h - exp) ** 2 / exp).sum()
    dof = q - 1
    assert chi2 < dof + 5 * math.sqrt(2 * dof)
    assert h.min() > 0
    s = o.spins()
    # neighbouring sites are uncorrelated: satisfied-bond fraction = 1/q
    frac = ((s == np.roll(s, 1, 0)).mean() + (s == np.roll(s, 1, 1)).mean()) / 2
    assert abs(frac - 1 / q) < 5 * math.sqrt((1 / q) * (1 - 1 / q) / (2 * L * L))


# ---------------------------------------------------------------- P10: golden trajectories (R2, R3, R9)
def test_p10_golden_trajectories(golden_dir):
    cases, cur = [], None
    for ln in _lines(golden_dir, "trajectories.txt"):
        p = ln.split()
        if p[0] == "case":
            cur = {"L": int(p[1]), "q": int(p[2]), "seed": int(p[3]), "init": p[4], "f": float(p[5]),
                   "row0": None, "E": {}, "hist": {}}
            cases.append(cur)
        elif p[0] == "row0":
            cur["row0"] = [int(x) for x in p[1:]]
        elif p[0] == "hist":
            cur["hist"][int(p[1])] = [int(x) for x in p[2:]]
        elif p[0] == "E":
            cur["E"] = {int(a.split(":")[0]): int(a.split(":")[1]) for a in p[1:]}
    assert len(cases) == 3
    for c in cases:
        init = oracle.INIT_RANDOM if c["init"] == "random" else oracle.INIT_ORDERED
        o = oracle.OraclePotts(c["L"], c["q"], c["seed"], init)
        T = c["f"] * workloads.t_c(c["q"])
        if c["row0"]:
            assert list(o.spins()[0, :len(c["row0"])]) == c["row0"]
        tmax = max(list(c["E"]) + list(c["hist"]))
        E = {0: o.energy()}
        H = {0: list(o.histogram())}
        for t in range(1, tmax + 1):
            o.sweep(T, 1)
            if t in c["E"]:
                E[t] = o.energy()
            if t in c["hist"]:
                H[t] = list(o.histogram())
        for t, want in c["E"].items():
            assert E[t] == want, (c, t)
        for t, want in c["hist"].items():
            assert H[t] == want, (c, t)


# ---------------------------------------------------------------- R10: derived observables
def test_r10_observables_closed_cases():
    # two-valued series: mean/variance/4th moment known in closed form
    E = [-10] * 50 + [-30] * 50
    N, T = 16, 2.0
    assert obs.specific_heat(E, N, T) == 100.0 / (16 * 4.0)
    assert obs.binder_cumulant(E) == pytest.approx(1 - 410000.0 / (3 * 250000.0), rel=2e-16)   # = 34/75
    assert obs.binder_cumulant([-7] * 9) == 2 / 3
    assert obs.magnetisation([16, 0, 0], 3) == 1.0
    assert obs.magnetisation([5, 5, 5, 5], 4) == 0.0
    assert obs.energy_per_spin(-32, 16) == -2.0
    # huge energies (L = 32768 scale): the exact-integer path does not lose the variance
    base = -(2 ** 31) + 12345
    big = [base + d for d in (0, 1, 2, 3, 4)]
    assert obs.specific_heat(big, 2 ** 30, 1.0) == 2.0 / 2 ** 30


# ---------------------------------------------------------------- derived observables: closed cases
def test_mean_energy_per_spin_closed_cases():
    from oracle import observables as ob
    N = 64 * 64
    assert ob.mean_energy_per_spin([-2 * N] * 7, N) == -2.0                 # ordered state, Eq. 1: 2N satisfied bonds
    assert ob.mean_energy_per_spin([-2 * N, 0], N) == -1.0
    assert ob.mean_energy_per_spin([-3, -5, -4], 4) == -1.0                 # (-12 / 3) / 4
    assert ob.mean_energy_per_spin([-1, -2], 3) == -0.5                     # (-3 / 2) / 3
    # mean of per-sample energies per spin, the definition e = <E> / N (PAPER.md:209 uses e = E/N)
    rng = np.random.default_rng(0)
    E = rng.integers(-2 * N, 0, size=1000)
    assert abs(ob.mean_energy_per_spin(E, N) - float(np.mean(E.astype(np.float64)) / N)) < 1e-12
    # consistent with the single-sample form
    assert ob.mean_energy_per_spin([-4582], N) == ob.energy_per_spin(-4582, N)


def test_susceptibility_and_magnetisation_moments_closed_cases():
    """chi = N/T (<m^2> - <m>^2) (Eq. 11) with m of Eq. 7."""
    from oracle import observables as ob
    q, N = 4, 400
    ordered = [N, 0, 0, 0]                      # m = 1
    uniform = [100, 100, 100, 100]              # m = 0
    half = [250, 50, 50, 50]                    # Nmax/N = 5/8: m = (4 * 5/8 - 1) / 3 = 1/2
    assert ob.magnetisation_moments([ordered] * 5, q) == (1.0, 1.0)
    assert ob.susceptibility([ordered] * 5, q, 0.7) == 0.0                  # no fluctuation
    assert ob.magnetisation_moments([ordered, uniform], q) == (0.5, 0.5)
    assert ob.susceptibility([ordered, uniform], q, 2.0) == N / 2.0 * 0.25  # variance 1/4
    m1, m2 = ob.magnetisation_moments([half, half, uniform, ordered], q)
    assert m1 == 0.5 and m2 == (0.25 + 0.25 + 0.0 + 1.0) / 4
    assert abs(ob.susceptibility([half, half, uniform, ordered], q, 0.5) - N / 0.5 * (0.375 - 0.25)) < 1e-12
    # which state holds the majority does not matter (Eq. 7 uses the maximum)
    assert ob.magnetisation_moments([[50, 250, 50, 50]], q) == (0.5, 0.25)
