"""GPU parity at BASELINE.json's full lattice sizes, in the launch configuration bench.py times (-m gpu).

The oracle (row-parallel mode, same bits as serial: tests/test_oracle_pins.py) can afford a few full sweeps even at
L = 32768, so the first sweeps are compared element by element; later times are covered by (a) restarting the oracle
from a downloaded GPU state (state = spins + t, the RNG is stateless) and (b) checking sampled sites one by one with the
oracle's single-site rule against the GPU's configurations before and after a sweep.
"""
import os

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu
THREADS = len(os.sched_getaffinity(0))


@pytest.fixture(scope="module")
def pb():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible")
    import paper_1101_0876_b200 as pb
    pb.load_library()
    return pb


def _gpu(pb, w):
    return pb.Potts(w.L, w.q, w.seed, w.init, layout=pb.LAYOUT_PACKED if w.packed else pb.LAYOUT_U8)


def _check_sampled_sites(w, T, t, S0, S1, n=1500, seed=11):
    """S0 / S1 = configurations before / after sweep t.  Whites were updated from S0, blacks from the new whites."""
    rng = np.random.default_rng(seed)
    L = w.L
    for i, j in zip(rng.integers(0, L, n), rng.integers(0, L, n)):
        i, j = int(i), int(j)
        c = (i + j) & 1
        src = S0 if c == 0 else S1          # the other colour as the site saw it
        nb = [src[(i - 1) % L, j], src[(i + 1) % L, j], src[i, (j - 1) % L], src[i, (j + 1) % L]]
        want = oracle.update_site(i, j, t, c, w.seed, w.q, T, int(S0[i, j]), nb)
        assert int(S1[i, j]) == want, (i, j, t)


def test_cfg2_full_size_resident_launch_and_late_restart(pb):
    w = workloads.CONFIGS[2]
    T = w.temperatures[0]
    g, o = _gpu(pb, w), oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=THREADS)
    assert g.potts_get_option("resident_active") > 1            # the configuration bench.py times: many CTAs, shared memory
    Eg, _ = g.potts_sweep_measured(T, 40, 1, hist=False)
    Eo, _ = o.sweep_measured(T, 40, 1, hist=False)
    assert (Eg == Eo).all() and (g.potts_download() == o.spins()).all()
    g.potts_sweep(T, 2000)                                       # one persistent launch
    S = g.potts_download()
    o.set_state(S, 2040)
    assert g.potts_sweep_count() == 2040 and g.potts_energy() == o.energy()
    Eg, Hg = g.potts_sweep_measured(T, 5, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, 5, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all() and (g.potts_download() == o.spins()).all()
    assert Eg[-1] > -2 * w.L * w.L                               # the superheated ordered state has started to decay


def test_cfg3_full_size_scan_start(pb):
    w = workloads.CONFIGS[3]
    g, o = _gpu(pb, w), oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=THREADS)
    assert (g.potts_download() == o.spins()).all()
    for T in w.temperatures[:2]:                                 # the ladder carries configuration and t over
        Eg, Hg = g.potts_sweep_measured(T, 3, 1, hist=True)
        Eo, Ho = o.sweep_measured(T, 3, 1, hist=True)
        assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts_download() == o.spins()).all()


@pytest.mark.parametrize("L,q,opts", [
    (3072, 9, {"variant": 2}),                                       # 192 chunks per halo row over 64 comm threads: three each
    (2304, 6, {"variant": 2, "resident_ctas": 37}),                  # 144 chunks: sixteen comm threads get three, the rest two
    (4096, 24, {"variant": 2, "resident_ctas": 148, "resident_rows": 1}),
    (2560, 200, {"variant": 2, "resident_words": 2, "resident_ctas": 100}),
])
def test_resident_comm_threads_share_the_halo_chunks(pb, L, q, opts):
    """Beyond L = 2048 the resident kernel's 64 comm threads each receive several 8-site chunks of a halo row
    (potts_resident.cuh): every sweep of a short run against the oracle, on even and uneven chunk splits."""
    g = pb.Potts(L, q, 31, workloads.INIT_RANDOM)
    for k, v in opts.items():
        g.potts_set_option(k, v)
    assert g.potts_get_option("resident_active") > 1
    o = oracle.OraclePotts(L, q, 31, workloads.INIT_RANDOM, threads=len(os.sched_getaffinity(0)))
    T = 0.99 * workloads.t_c(q)
    Eg, Hg = g.potts_sweep_measured(T, 4, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, 4, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    g.potts_sweep(T, 3)
    o.sweep(T, 3)
    assert (g.potts_download() == o.spins()).all() and g.potts_energy() == o.energy()


def test_cfg4_full_size_packed(pb):
    w = workloads.CONFIGS[4]
    T = w.temperatures[0]
    g, o = _gpu(pb, w), oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=THREADS)
    Eg, _ = g.potts_sweep_measured(T, 3, 1, hist=False)
    Eo, _ = o.sweep_measured(T, 3, 1, hist=False)
    assert (Eg == Eo).all() and (g.potts_download() == o.spins()).all()
    g.potts_sweep(T, 30)
    S0 = g.potts_download()
    t = g.potts_sweep_count()
    g.potts_sweep(T, 1)
    _check_sampled_sites(w, T, t, S0, g.potts_download())
    assert int(g.potts_histogram().sum()) == w.L * w.L


def test_cfg5_full_size_streaming(pb):
    w = workloads.CONFIGS[5]
    T = w.temperatures[0]
    g = _gpu(pb, w)
    o = oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=THREADS)
    S = g.potts_download()
    assert (S == o.spins()).all()                                # random start, 2^30 sites
    assert g.potts_energy() == o.energy()
    Eg, Hg = g.potts_sweep_measured(T, 2, 2, hist=True)          # fused energy + histogram at full size
    o.sweep(T, 2)
    assert int(Eg[0]) == o.energy() == o.energy_incremental()
    assert (Hg[0] == o.histogram()).all()
    S0 = g.potts_download()
    assert (S0 == o.spins()).all()
    del S
    g.potts_sweep(T, 10)
    S0 = g.potts_download(S0)
    t = g.potts_sweep_count()
    E1, H1 = g.potts_sweep_measured(T, 1, 1, hist=True)
    S1 = g.potts_download()
    _check_sampled_sites(w, T, t, S0, S1)
    assert int(H1[0].sum()) == w.L * w.L and -2 * w.L * w.L <= int(E1[0]) < 0
    assert int(E1[0]) == g.potts_energy() and (H1[0] == g.potts_histogram()).all()   # fused == standalone reduction
    # mid-run restart: the oracle takes over the GPU's state at t = 13 (state = spins + t, the RNG is stateless) and
    # both run the next two sweeps of the workload's cadence in full; every spin, the energy and the histogram agree
    t1 = g.potts_sweep_count()
    o.set_state(S1, t1)
    del S0
    E2, H2 = g.potts_sweep_measured(T, 2, 2, hist=True)
    o.sweep(T, 2)
    assert int(E2[0]) == o.energy() == o.energy_incremental()
    assert (H2[0] == o.histogram()).all()
    assert (g.potts_download(S1) == o.spins()).all()


@pytest.mark.parametrize("q,want_eo,want_ed", [(9, -1.633167, -1.033499), (15, -1.765905, -0.750492)])
def test_p9_energies_of_the_coexisting_phases_at_tc(pb, q, want_eo, want_ed):
    """SURVEY pin P9, the paper's own validation (Table 2 at :213-221): at T_c the ordered branch
    (heated from the ordered start) sits at e_o and the disordered branch (cooled from a random start) at e_d.
    Values are Table 2's exact columns (tests/golden/paper_constants.txt); L = 1024 keeps both branches metastable
    for far longer than the run and finite-size shifts below the tolerance."""
    L, N = 1024, 1024 * 1024
    Tc = workloads.t_c(q)
    for init, want in ((workloads.INIT_ORDERED, want_eo), (workloads.INIT_RANDOM, want_ed)):
        g = pb.Potts(L, q, 17, init)
        E, _ = g.potts_ladder([Tc], 6000, 2000, 20, hist=False)
        e = float(E.mean()) / N
        assert abs(e - want) < 6e-3, (q, init, e, want)


def test_stream_spec_2_full_size(pb):
    """Stream-spec v2 at full sizes: packed L = 8192 element by element, L = 32768 on sampled sites."""
    w = workloads.CONFIGS[4]
    T = w.temperatures[0]
    g = _gpu(pb, w)
    g.potts_set_stream_spec(2)
    o = oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=THREADS, stream=2)
    Eg, _ = g.potts_sweep_measured(T, 3, 1, hist=False)
    Eo, _ = o.sweep_measured(T, 3, 1, hist=False)
    assert (Eg == Eo).all() and (g.potts_download() == o.spins()).all()
    del g, o
    w = workloads.CONFIGS[5]
    T = w.temperatures[0]
    g = _gpu(pb, w)
    g.potts_set_stream_spec(2)
    g.potts_sweep(T, 5)
    S0 = g.potts_download()
    t = g.potts_sweep_count()
    g.potts_sweep(T, 1)
    S1 = g.potts_download()
    rng = np.random.default_rng(3)
    L = w.L
    for i, j in zip(rng.integers(0, L, 1500), rng.integers(0, L, 1500)):
        i, j = int(i), int(j)
        c = (i + j) & 1
        src = S0 if c == 0 else S1
        nb = [src[(i - 1) % L, j], src[(i + 1) % L, j], src[i, (j - 1) % L], src[i, (j + 1) % L]]
        assert int(S1[i, j]) == oracle.update_site(i, j, t, c, w.seed, w.q, T, int(S0[i, j]), nb, stream=2), (i, j)
