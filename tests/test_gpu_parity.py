"""GPU parity: the CUDA path through the C-ABI against the CPU oracle, bit for bit (-m gpu).

Same seeded inputs on both sides (workloads.py); spins, energy series and histograms must be
identical after every sweep (north_star: "bit-exactly, with identical spin configurations,
energy series and histograms after every sweep").  Integer work, so the bar is equality.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pb():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible")
    import paper_1101_0876_b200 as pb
    pb.load_library()
    return pb


# How the sweep is launched never changes what it computes (P6: "any GPU tile/launch shape ... same bits"):
# streaming = one launch per half-sweep; resident = one persistent launch, lattice in shared memory,
# split over `ctas` CTAs that exchange boundary rows (0 = the library's own choice).
LAUNCH_SHAPES = {
    "streaming": {"variant": 1},
    "resident": {"variant": 2},
    "resident1": {"variant": 2, "resident_ctas": 1},
    "resident2": {"variant": 2, "resident_ctas": 2},
    "resident3": {"variant": 2, "resident_ctas": 3},
    "resident7": {"variant": 2, "resident_ctas": 7},
    "resident148": {"variant": 2, "resident_ctas": 148},
    "resident_w1": {"variant": 2, "resident_words": 1},          # one 4-site word per thread and row visit
    "resident_w1_5": {"variant": 2, "resident_words": 1, "resident_ctas": 5},
    "resident_w2": {"variant": 2, "resident_words": 2},          # an 8-site chunk per thread and row visit
    "cluster": {"variant": 3},                                   # one thread-block cluster, boundary rows through DSMEM
    "cluster1": {"variant": 3, "cluster_ctas": 1},
    "cluster3": {"variant": 3, "cluster_ctas": 3},
    "cluster8": {"variant": 3, "cluster_ctas": 8},
    "cluster16": {"variant": 3, "cluster_ctas": 16},             # beyond the portable cluster size
    "auto": {"variant": 0},
}


def _pair(pb, L, q, seed, init, layout=0, shape=None):
    g = pb.Potts(L, q, seed, init, layout=layout)
    for k, v in LAUNCH_SHAPES[shape or "streaming"].items():
        g.potts_set_option(k, v)
    sh = shape or "streaming"
    if (sh.startswith("resident") and g.potts_get_option("resident_active") == 0) or \
            (sh.startswith("cluster") and g.potts_get_option("cluster_active") == 0):
        with pytest.raises(pb.PottsError) as e:          # a forced shape that cannot hold the lattice is refused
            g.potts_sweep(1.0, 1)
        assert e.value.code == pb.ERR_UNSUPPORTED
        pytest.skip(f"L={L} does not fit the shared memory of shape {shape}")
    o = oracle.OraclePotts(L, q, seed, init)
    return g, o


@pytest.mark.parametrize("shape", ["streaming", "resident", "resident2", "resident7", "cluster", "auto"])
def test_cfg1_full_run_series_and_spins(pb, shape):
    """BASELINE configs[0] in full: q=9, L=64, random start, 0.99 T_c, 1000 sweeps, E+hist every sweep."""
    w = workloads.CONFIGS[1]
    g, o = _pair(pb, w.L, w.q, w.seed, w.init, shape=shape)
    assert g.potts_energy() == o.energy()
    assert (g.potts_histogram() == o.histogram()).all()
    assert (g.potts_download() == o.spins()).all()
    T = w.temperatures[0]
    Eg, Hg = g.potts_sweep_measured(T, w.sweeps_per_t, w.every, hist=True)
    Eo, Ho = o.sweep_measured(T, w.sweeps_per_t, w.every, hist=True)
    assert (Eg == Eo).all()
    assert (Hg == Ho).all()
    assert (g.potts_download() == o.spins()).all()
    assert g.potts_sweep_count() == o.t == 1000
    # derived observables, host double, 1e-12 relative (north_star)
    from oracle import observables as obs
    me, cv, bl = pb.potts_observables(Eg, w.L * w.L, T)
    for got, want in ((me, obs.mean_energy_per_spin(Eo, w.L * w.L)), (cv, obs.specific_heat(Eo, w.L * w.L, T)),
                      (bl, obs.binder_cumulant(Eo))):
        assert abs(got - want) <= 1e-12 * abs(want)
    assert abs(pb.potts_magnetisation(Hg[-1], w.q) - obs.magnetisation(Ho[-1], w.q)) <= 1e-12


@pytest.mark.parametrize("L,q,init,f,seed", [
    (32, 2, workloads.INIT_RANDOM, 1.0, 11),        # smallest supported L, Ising limit
    (64, 6, workloads.INIT_ORDERED, 1.005, 7),      # cfg2's parameters at small L
    (96, 24, workloads.INIT_ORDERED, 1.002, 4),     # L not a power of two, several blocks + ragged tail
    (160, 9, workloads.INIT_RANDOM, 0.98, 3),
    (224, 128, workloads.INIT_RANDOM, 1.0, 5),      # largest q on the 7-bit compare path
    (64, 129, workloads.INIT_RANDOM, 1.0, 6),       # first q on the 8-bit compare path
    (96, 256, workloads.INIT_RANDOM, 1.1, 8),       # maximum q
    (64, 3, workloads.INIT_RANDOM, 50.0, 9),        # hot: nearly every proposal accepted
    (64, 5, workloads.INIT_RANDOM, 0.05, 10),       # cold: thresholds ~ 0
    (512, 9, workloads.INIT_RANDOM, 0.995, 5),      # many blocks
])
@pytest.mark.parametrize("shape", ["streaming", "resident", "resident1", "resident3", "resident148", "resident_w1",
                                   "resident_w1_5", "resident_w2", "cluster", "cluster1", "cluster3", "cluster8", "cluster16", "auto"])
def test_every_sweep_spins_energy_histogram(pb, L, q, init, f, seed, shape):
    g, o = _pair(pb, L, q, seed, init, shape=shape)
    T = f * workloads.t_c(q)
    assert (g.potts_download() == o.spins()).all()
    for _ in range(6):
        g.potts_sweep(T, 1)
        o.sweep(T, 1)
        assert (g.potts_download() == o.spins()).all()
        assert g.potts_energy() == o.energy()
        assert (g.potts_histogram() == o.histogram()).all()
    Eg, Hg = g.potts_sweep_measured(T, 24, 3, hist=True)
    Eo, Ho = o.sweep_measured(T, 24, 3, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts_download() == o.spins()).all()


def test_sweep_split_equals_single_call_and_seed_high_bits(pb):
    L, q, seed = 128, 9, (0xDEADBEEF << 32) | 12345       # key1 != 0
    T = 0.99 * workloads.t_c(q)
    a, o = _pair(pb, L, q, seed, workloads.INIT_RANDOM)
    b = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
    a.potts_sweep(T, 20)
    b.potts_sweep(T, 7)
    b.potts_sweep(T, 13)
    o.sweep(T, 20)
    sa = a.potts_download()
    assert (sa == b.potts_download()).all() and (sa == o.spins()).all()


@pytest.mark.parametrize("kind", ["domains", "stripes", "uniform"])
def test_upload_restart_matches_oracle(pb, kind):
    L, q = 96, 7
    s0 = workloads.synthetic_spins(L, q, 123, kind)
    g = pb.Potts(L, q, 99, workloads.INIT_ORDERED)
    o = oracle.OraclePotts(L, q, 99, workloads.INIT_ORDERED)
    g.potts_upload(s0)
    g.potts_set_sweep_count(1000)
    o.set_state(s0, 1000)
    assert (g.potts_download() == s0).all()
    assert g.potts_energy() == o.energy()
    T = 1.0 * workloads.t_c(q)
    Eg, Hg = g.potts_sweep_measured(T, 10, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, 10, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all() and (g.potts_download() == o.spins()).all()


def test_degenerate_temperatures(pb):
    L, q = 64, 6
    g = pb.Potts(L, q, 1, workloads.INIT_ORDERED)
    E, H = g.potts_sweep_measured(0.01, 20, 1, hist=True)
    assert (E == -2 * L * L).all() and (H[:, 0] == L * L).all()
    g, o = _pair(pb, L, q, 2, workloads.INIT_RANDOM)
    Eg, _ = g.potts_sweep_measured(1e12, 10, 1, hist=False)
    Eo, _ = o.sweep_measured(1e12, 10, 1, hist=False)
    assert (Eg == Eo).all()


def test_errors_on_device(pb):
    g = pb.Potts(64, 4, 1)
    with pytest.raises(pb.PottsError) as e:
        g.potts_sweep(-1.0, 1)
    assert e.value.code == pb.ERR_ARG
    with pytest.raises(pb.PottsError):
        g.potts_sweep(float("nan"), 1)
    with pytest.raises(pb.PottsError):
        g.potts_sweep_measured(1.0, 10, 3)            # every does not divide nsweeps
    bad = np.zeros((64, 64), dtype=np.uint8)
    bad[5, 7] = 4                                      # >= q
    before = g.potts_download()
    with pytest.raises(pb.PottsError):
        g.potts_upload(bad)
    assert (g.potts_download() == before).all()        # rejected upload leaves the lattice untouched
    g.potts_set_sweep_count(2 ** 32 - 2)
    g.potts_sweep(1.0, 1)
    with pytest.raises(pb.PottsError):
        g.potts_sweep(1.0, 1)                          # counter would pass 2^32 - 1
    E, _ = g.potts_sweep_measured(1.0, 0, 1)           # empty run is fine
    assert E.size == 0


# ---- sub-byte packed layout (BASELINE configs[3] is q=24 "sub-byte-packed ... (q<32)") ----------
@pytest.mark.parametrize("L,q,init,f,seed", [
    (64, 24, workloads.INIT_ORDERED, 1.002, 4),     # cfg4's parameters at the smallest packed L (5 bits)
    (128, 24, workloads.INIT_RANDOM, 1.0, 4),
    (192, 9, workloads.INIT_RANDOM, 0.99, 1),       # 4 bits, L not a power of two
    (64, 16, workloads.INIT_RANDOM, 1.0, 2),        # largest q on 4 bits
    (128, 17, workloads.INIT_RANDOM, 1.0, 3),       # first q on 5 bits
    (64, 32, workloads.INIT_RANDOM, 1.05, 5),       # largest packed q
    (64, 2, workloads.INIT_RANDOM, 1.0, 6),
    (2048, 24, workloads.INIT_ORDERED, 1.002, 4),   # several blocks, more than one row per thread
])
def test_packed_layout_every_sweep(pb, L, q, init, f, seed):
    g, o = _pair(pb, L, q, seed, init, layout=pb.LAYOUT_PACKED)
    T = f * workloads.t_c(q)
    assert (g.potts_download() == o.spins()).all()
    assert g.potts_energy() == o.energy() and (g.potts_histogram() == o.histogram()).all()
    nstep = 6 if L <= 256 else 2
    for _ in range(nstep):
        g.potts_sweep(T, 1)
        o.sweep(T, 1)
        assert (g.potts_download() == o.spins()).all()
        assert g.potts_energy() == o.energy()
        assert (g.potts_histogram() == o.histogram()).all()
    n = 12 if L <= 256 else 3
    Eg, Hg = g.potts_sweep_measured(T, n, 3, hist=True)
    Eo, Ho = o.sweep_measured(T, n, 3, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts_download() == o.spins()).all()


def test_packed_upload_and_layout_invariance(pb):
    L, q = 128, 24
    s0 = workloads.synthetic_spins(L, q, 77, "domains")
    T = 1.002 * workloads.t_c(q)
    outs = []
    for layout in (pb.LAYOUT_U8, pb.LAYOUT_PACKED):
        g = pb.Potts(L, q, 4, workloads.INIT_ORDERED, layout=layout)
        g.potts_upload(s0)
        assert (g.potts_download() == s0).all()
        E, H = g.potts_sweep_measured(T, 10, 1, hist=True)
        outs.append((E, H, g.potts_download()))
    for a, b in zip(outs[0], outs[1]):
        assert (a == b).all()
    o = oracle.OraclePotts(L, q, 4, workloads.INIT_ORDERED)
    o.set_state(s0, 0)
    Eo, Ho = o.sweep_measured(T, 10, 1, hist=True)
    assert (outs[1][0] == Eo).all() and (outs[1][1] == Ho).all() and (outs[1][2] == o.spins()).all()


def test_packed_limits(pb):
    for L, q in ((64, 33), (96, 9)):
        with pytest.raises(pb.PottsError) as e:
            pb.Potts(L, q, 1, layout=pb.LAYOUT_PACKED)
        assert e.value.code == pb.ERR_UNSUPPORTED
    assert pb.potts_workspace_bytes(8192, 24, pb.LAYOUT_PACKED) < 0.7 * pb.potts_workspace_bytes(8192, 24, pb.LAYOUT_U8)


def test_ladder_protocol_matches_oracle_and_call_sequence(pb):
    """T ladder with transient + measured sweeps, state carried over (here: a short cooling ladder)."""
    L, q, seed = 128, 9, 3
    Ts = [f * workloads.t_c(q) for f in (1.02, 1.0, 0.98)]
    g, o = _pair(pb, L, q, seed, workloads.INIT_RANDOM, shape="resident")
    E, H = g.potts_ladder(Ts, 7, 12, 4, hist=True)
    assert E.shape == (3, 3) and H.shape == (3, 3, q)
    g2 = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
    g2.potts_set_option("variant", 1)
    for k, T in enumerate(Ts):
        o.sweep(T, 7)
        Eo, Ho = o.sweep_measured(T, 12, 4, hist=True)
        g2.potts_sweep(T, 7)
        E2, H2 = g2.potts_sweep_measured(T, 12, 4, hist=True)
        assert (E[k] == Eo).all() and (H[k] == Ho).all() and (E2 == Eo).all() and (H2 == Ho).all()
    assert (g.potts_download() == o.spins()).all() and g.potts_sweep_count() == o.t == 57
    with pytest.raises(pb.PottsError):
        g.potts_ladder(Ts, 1, 10, 3)
    with pytest.raises(pb.PottsError):
        g.potts_ladder([0.7, -1.0], 1, 10, 5)


# ---- replica batch: lattice r of a batch == a single handle with (seed_r, T_r) ---------------------------
@pytest.mark.parametrize("L,q,n", [(64, 9, 5), (32, 2, 3), (128, 24, 4), (96, 200, 2), (256, 6, 3),
                                   (160, 12, 2),      # 1024 / (L/8) thread rows would be odd: made even (one parity per thread)
                                   (416, 9, 2)])      # the largest lattice a CTA holds beside the 32 KB accept table: 18 thread rows over 416 rows, uneven
def test_batch_replicas_match_oracle(pb, L, q, n):
    seeds = [1000 + 7 * r + (r << 40) for r in range(n)]
    Ts = [(0.9 + 0.1 * r) * workloads.t_c(q) for r in range(n)]
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
    E, H = b.potts_batch_sweep_measured(Ts, 12, 3)
    E2, _ = b.potts_batch_sweep_measured(Ts, 5, 1, hist=False)          # the counter carries over
    assert b.potts_batch_sweep_count() == 17
    for r in range(n):
        o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_RANDOM)
        Eo, Ho = o.sweep_measured(Ts[r], 12, 3, hist=True)
        assert (E[r] == Eo).all() and (H[r] == Ho).all(), r
        Eo2, _ = o.sweep_measured(Ts[r], 5, 1, hist=False)
        assert (E2[r] == Eo2).all() and (b.potts_batch_download(r) == o.spins()).all(), r


def test_batch_larger_than_one_launch_and_ordered_start(pb):
    L, q, n = 32, 6, 1030                                              # > 1024 lattices: two launches per call
    seeds = list(range(5, 5 + n))
    T = 1.005 * workloads.t_c(q)
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_ORDERED)
    E, _ = b.potts_batch_sweep_measured(T, 6, 2, hist=False)
    assert b.potts_batch_launch_count() == 2
    for r in (0, 1, 511, 1023, 1024, 1029):
        o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_ORDERED)
        Eo, _ = o.sweep_measured(T, 6, 2, hist=False)
        assert (E[r] == Eo).all() and (b.potts_batch_download(r) == o.spins()).all(), r
    with pytest.raises(pb.PottsError):
        pb.PottsBatch(512, 6, [1, 2])                                  # does not fit one CTA


# ---- stream-spec v2 (S15): one Philox block per pair of same-colour sites ------------------
@pytest.mark.parametrize("L,q,init,f,seed,layout,shape", [
    (64, 9, workloads.INIT_RANDOM, 0.99, 1, 0, "streaming"),
    (64, 9, workloads.INIT_RANDOM, 0.99, 1, 0, "resident"),
    (96, 6, workloads.INIT_ORDERED, 1.005, 7, 0, "resident3"),
    (256, 24, workloads.INIT_RANDOM, 1.0, 4, 0, "resident_w2"),
    (512, 200, workloads.INIT_RANDOM, 1.0, 9, 0, "resident_w1"),
    (1024, 6, workloads.INIT_ORDERED, 1.005, 7, 0, "resident"),
    (128, 129, workloads.INIT_RANDOM, 1.2, 5, 0, "streaming"),
    (128, 9, workloads.INIT_RANDOM, 0.99, 3, 0, "cluster"),
    (128, 24, workloads.INIT_ORDERED, 1.002, 4, 1, "streaming"),       # packed, 5 bits
    (192, 9, workloads.INIT_RANDOM, 0.99, 2, 1, "streaming"),          # packed, 4 bits
])
def test_stream_spec_2_matches_oracle(pb, L, q, init, f, seed, layout, shape):
    g = pb.Potts(L, q, seed, init, layout=layout)
    for k, v in LAUNCH_SHAPES[shape].items():
        g.potts_set_option(k, v)
    g.potts_set_stream_spec(2)
    assert g.potts_get_stream_spec() == 2
    o = oracle.OraclePotts(L, q, seed, init, stream=2, threads=4)
    T = f * workloads.t_c(q)
    Eg, Hg = g.potts_sweep_measured(T, 12, 3, hist=True)
    Eo, Ho = o.sweep_measured(T, 12, 3, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    g.potts_sweep(T, 3)
    o.sweep(T, 3)
    assert (g.potts_download() == o.spins()).all() and g.potts_energy() == o.energy()
    with pytest.raises(pb.PottsError):
        g.potts_set_stream_spec(3)


def test_stream_spec_2_batch_and_default_unchanged(pb):
    L, q, seeds, T = 64, 9, [11, 12, 13], 0.99 * workloads.t_c(9)
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
    b.potts_batch_set_stream_spec(2)
    E, H = b.potts_batch_sweep_measured(T, 8, 2)
    for r, s in enumerate(seeds):
        o = oracle.OraclePotts(L, q, s, workloads.INIT_RANDOM, stream=2)
        Eo, Ho = o.sweep_measured(T, 8, 2, hist=True)
        assert (E[r] == Eo).all() and (H[r] == Ho).all() and (b.potts_batch_download(r) == o.spins()).all()
    g = pb.Potts(L, q, 11, workloads.INIT_RANDOM)
    assert g.potts_get_stream_spec() == 1                  # the default chain is north_star's per-site stream


def test_batch_ladder_matches_single_handle_ladders_and_oracle(pb):
    """potts_batch_ladder (PAPER.md:96 for every replica at once): replica r == potts_ladder of a single handle with
    (seed_r, ladder_r) == the oracle driven through the same call sequence."""
    L, q, n = 64, 6, 4
    seeds = [900 + r for r in range(n)]
    Tc = workloads.t_c(q)
    ladders = np.array([[(1.03 - 0.01 * r) * Tc, 1.0 * Tc, (0.97 + 0.005 * r) * Tc] for r in range(n)])
    t_tran, t_max, dt = 6, 12, 3
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
    E, H = b.potts_batch_ladder(ladders, t_tran, t_max, dt)
    assert E.shape == (n, 3, t_max // dt) and H.shape == (n, 3, t_max // dt, q)
    for r in range(n):
        g = pb.Potts(L, q, seeds[r], pb.INIT_RANDOM)
        Eg, Hg = g.potts_ladder(list(ladders[r]), t_tran, t_max, dt, hist=True)
        assert (np.asarray(Eg).reshape(3, -1) == E[r]).all() and (np.asarray(Hg).reshape(3, -1, q) == H[r]).all()
        o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_RANDOM)
        for k in range(3):
            o.sweep(float(ladders[r, k]), t_tran)
            Eo, Ho = o.sweep_measured(float(ladders[r, k]), t_max, dt, hist=True)
            assert (Eo == E[r, k]).all() and (Ho == H[r, k]).all()
        assert (b.potts_batch_download(r) == o.spins()).all()
    assert b.potts_batch_sweep_count() == 3 * (t_tran + t_max)


def test_susceptibility_of_a_gpu_series_against_exact_rationals(pb):
    """chi, <m>, <m^2> (Eq. 11) of a histogram series recorded on the GPU: the library's host function
    against the oracle-side exact rational arithmetic, 1e-12 relative."""
    from oracle import observables as ob
    L, q = 128, 2
    T = 1.0 * workloads.t_c(q)
    g = pb.Potts(L, q, 17, pb.INIT_RANDOM)
    _, H = g.potts_sweep_measured(T, 200, 1, hist=True)
    m1, m2, chi = pb.potts_susceptibility(H, q, T)
    w1, w2 = ob.magnetisation_moments(H, q)
    wchi = ob.susceptibility(H, q, T)
    for got, want in ((m1, w1), (m2, w2), (chi, wchi)):
        assert abs(got - want) <= 1e-12 * abs(want)
    assert 0.0 < m1 < 1.0 and chi > 0.0


def test_every_beyond_2_30_is_rejected(pb):
    """The persistent kernels count samples in 32 bits: `every` > 2^30 is an argument error (not an endless loop)."""
    g = pb.Potts(64, 9, 1, pb.INIT_RANDOM)
    with pytest.raises(pb.PottsError) as e:
        g.potts_sweep_measured(1.0, 2 ** 31, 2 ** 31, hist=False)
    assert e.value.code == pb.ERR_ARG
    assert g.potts_sweep_count() == 0


def test_persistent_kernels_are_deterministic_under_repetition(pb):
    """compute-sanitizer is closed on this pool (profiles/r02c_sanitizer.md), so the hand-rolled inter-CTA packet
    protocol and the DSMEM exchange are exercised instead: the same run repeated on many grid shapes must give the
    same bits every time (a race shows up as run-to-run differences), and those bits are the oracle's."""
    L, q, seed, n = 256, 9, 4, 60
    T = 0.99 * workloads.t_c(q)
    o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM, threads=4)
    Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
    want = o.spins()
    shapes = [{"variant": 2, "resident_ctas": c} for c in (2, 5, 16, 37, 64, 148)] + \
             [{"variant": 2, "resident_ctas": 148, "resident_words": 2}, {"variant": 3, "cluster_ctas": 16}, {"variant": 3, "cluster_ctas": 8}]
    for shape in shapes:
        for rep in range(4):
            g = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
            for k, v in shape.items():
                g.potts_set_option(k, v)
            Eg, Hg = g.potts_sweep_measured(T, n, 1, hist=True)
            assert (Eg == Eo).all() and (Hg == Ho).all(), (shape, rep)
            assert (g.potts_download() == want).all(), (shape, rep)
            g.close()


@pytest.mark.parametrize("L,q,ctas", [(64, 9, 4), (64, 9, 1), (32, 6, 2), (128, 24, 16), (96, 3, 3), (64, 200, 8)])
def test_cluster_kernel_exchange_over_many_launches(pb, L, q, ctas):
    """The cluster kernel's neighbour exchange (8-byte packets {4 spins | half-sweep number} into the neighbour's inbox in
    its shared memory, polled by the thread that needs them, potts_cluster.cuh) numbers its half-sweeps per launch:
    launches of 1, 2, 3, ... sweeps (the packet-free first half-sweep, odd and even counts, an inbox that starts zeroed
    every time), with every measurement form in turn, must follow the oracle's chain bit for bit, and repeat it."""
    seed = 21
    T = 0.99 * workloads.t_c(q)
    for rep in range(2):
        g = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
        g.potts_set_option("variant", 3)
        g.potts_set_option("cluster_ctas", ctas)
        assert g.potts_get_option("cluster_active") == ctas
        o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM)
        for k, n in enumerate([1, 1, 2, 3, 1, 4, 7, 2, 5, 16, 1]):
            kind = k % 4
            if kind == 0:
                g.potts_sweep(T, n)
                o.sweep(T, n)
            elif kind == 1:
                Eg, Hg = g.potts_sweep_measured(T, n, 1, hist=True)
                Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
                assert (Eg == Eo).all() and (Hg == Ho).all(), (rep, k, n)
            elif kind == 2:
                e0 = o.energy()
                d = g.potts_sweep_delta(T, n)
                es = []
                for _ in range(n):
                    o.sweep(T, 1)
                    es.append(o.energy())
                assert (d == np.diff(np.array([e0] + es, dtype=np.int64))).all(), (rep, k, n)
            else:
                every = 2 if n % 2 == 0 else 1
                Eg, Hg = g.potts_sweep_measured(T, n, every, hist=False)
                Eo, Ho = o.sweep_measured(T, n, every, hist=False)
                assert (Eg == Eo).all(), (rep, k, n)
            assert g.potts_energy() == o.energy(), (rep, k, n)
        assert (g.potts_download() == o.spins()).all()
        assert (g.potts_histogram() == o.histogram()).all()
        g.close()


@pytest.mark.parametrize("L,q,seed,rows", [(1024, 9, 3, 0), (2048, 6, 8, 4), (1024, 24, 5, 16), (1024, 200, 2, 2)])
def test_streaming_kernel_with_bulk_staged_rows(pb, L, q, seed, rows):
    """Option stream_stage = 1 (cp.async.bulk staging of the other-colour rows, an experiment kept for its A/B record)
    is one more launch shape of the same chain."""
    T = 0.99 * workloads.t_c(q)
    g = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
    g.potts_set_option("variant", 1)
    g.potts_set_option("stream_stage", 1)
    if rows:
        g.potts_set_option("stream_rows", rows)
    o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM, threads=8)
    g.potts_sweep(T, 3)
    Eg, Hg = g.potts_sweep_measured(T, 2, 1, hist=True)      # sampled sweeps take the unstaged kernel
    g.potts_sweep(T, 2)
    o.sweep(T, 3)
    Eo, Ho = o.sweep_measured(T, 2, 1, hist=True)
    o.sweep(T, 2)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts_download() == o.spins()).all()


def test_batch_series_on_the_device_equal_the_host_series(pb):
    """potts_batch_sweep_measured_dev leaves the series on the device: same numbers as the host variant / the oracle."""
    import torch
    L, q, n, ns = 64, 9, 4, 12
    seeds = [70 + r for r in range(n)]
    Ts = [(0.95 + 0.03 * r) * workloads.t_c(q) for r in range(n)]
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
    E_dev = torch.full((n, ns // 2), 123, dtype=torch.int64, device="cuda")     # stale contents must be cleared by the call
    H_dev = torch.full((n, ns // 2, q), 7, dtype=torch.int64, device="cuda")
    b.potts_batch_sweep_measured_dev(Ts, ns, 2, E_dev, H_dev)
    torch.cuda.synchronize()
    for r in range(n):
        o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_RANDOM)
        Eo, Ho = o.sweep_measured(Ts[r], ns, 2, hist=True)
        assert (E_dev[r].cpu().numpy() == Eo).all() and (H_dev[r].cpu().numpy() == Ho).all()
