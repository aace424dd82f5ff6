"""GPU parity of potts_sweep_delta (-m gpu): the per-sweep energy change accumulated on the fly from the accepted
moves against the oracle.

The oracle RECOUNTS Eq. 1 over the whole lattice after every sweep, so
E0 + cumsum(dE_gpu) == E_oracle is a comparison of two different computations of the same integers: it fails
if a single accepted move's d is dropped, double counted or has the wrong sign.  Spins must stay identical too
(the delta kernel is one more launch shape of the same chain, P6).
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


# (L, q, seed, init, T / T_c, sweeps): every compare mode (q <= 8, <= 16, <= 128, <= 256), several tiles and a
# ragged last warp (L = 96, 160), ordered and random starts, both sides of T_c
CASES = [
    (32, 2, 11, 1, 0.9, 40),
    (64, 9, 1, 1, 0.99, 60),
    (96, 6, 7, 0, 1.005, 40),
    (160, 24, 4, 1, 1.002, 25),
    (256, 15, 5, 1, 0.5, 20),
    (128, 200, 9, 1, 1.3, 20),
    (1088, 9, 3, 1, 0.995, 6),
]


# launch shapes of potts_sweep_delta: the library's choice (cluster kernel for L <= 288, resident kernel up to L = 4096,
# one launch per call), the streaming kernels (two launches per sweep), the resident kernel with forced grids, a cluster
VARIANTS = {
    "auto": {},
    "streaming": {"variant": 1},
    "resident": {"variant": 2},
    "resident3": {"variant": 2, "resident_ctas": 3},
    "resident_w2": {"variant": 2, "resident_words": 2, "resident_ctas": 7},
    "cluster8": {"variant": 3, "cluster_ctas": 8},
}


@pytest.mark.parametrize("variant", list(VARIANTS))
@pytest.mark.parametrize("stream", [1, 2])
@pytest.mark.parametrize("L,q,seed,init,f,n", CASES)
def test_delta_series_matches_recounted_energy(pb, L, q, seed, init, f, n, stream, variant):
    T = f * workloads.t_c(q)
    g = pb.Potts(L, q, seed, init)
    for k, v in VARIANTS[variant].items():
        g.potts_set_option(k, v)
    if variant == "cluster8" and not g.potts_get_option("cluster_active"):
        pytest.skip("the cluster kernel cannot hold this lattice")
    g.potts_set_stream_spec(stream)
    o = oracle.OraclePotts(L, q, seed, init, threads=4, stream=stream)
    E0 = o.energy()
    assert g.potts_energy() == E0
    try:
        dE = g.potts_sweep_delta(T, n)
    except pb.PottsError as e:
        if e.code == pb.ERR_UNSUPPORTED and variant not in ("auto", "streaming"):
            pytest.skip("forced launch shape cannot hold this lattice")
        raise
    Eo, _ = o.sweep_measured(T, n, 1, hist=False)
    assert dE.dtype == np.int64 and dE.shape == (n,)
    assert (E0 + np.cumsum(dE) == Eo).all()
    assert (g.potts_download() == o.spins()).all()
    assert g.potts_energy() == int(Eo[-1]) == o.energy_incremental()
    assert g.potts_sweep_count() == o.t == n


def test_delta_is_the_same_chain_as_the_other_launch_shapes(pb):
    """sweep(a); sweep_delta(b); sweep_measured(c) is the chain of sweep(a+b+c) (sweep counter lives in the handle)."""
    L, q, seed = 128, 9, 21
    T = 0.99 * workloads.t_c(q)
    g = pb.Potts(L, q, seed, pb.INIT_RANDOM)
    o = oracle.OraclePotts(L, q, seed, pb.INIT_RANDOM)
    g.potts_sweep(T, 7)
    Eo, _ = o.sweep_measured(T, 7, 1, hist=False)
    dE = g.potts_sweep_delta(T, 9)
    Eo2, _ = o.sweep_measured(T, 9, 1, hist=False)
    assert (int(Eo[-1]) + np.cumsum(dE) == Eo2).all()
    Eg3, _ = g.potts_sweep_measured(T, 5, 1, hist=False)
    Eo3, _ = o.sweep_measured(T, 5, 1, hist=False)
    assert (Eg3 == Eo3).all()
    assert (g.potts_download() == o.spins()).all()


def test_delta_degenerate_temperatures(pb):
    """P7: at T -> 0+ only d <= 0 is accepted: every dE <= 0, and the ordered state never moves."""
    g = pb.Potts(64, 6, 3, pb.INIT_RANDOM)
    dE = g.potts_sweep_delta(0.01, 30)
    assert (dE <= 0).all() and dE[0] < 0
    g = pb.Potts(64, 6, 3, pb.INIT_ORDERED)
    assert (g.potts_sweep_delta(0.01, 5) == 0).all()
    assert g.potts_energy() == -2 * 64 * 64


# packed layout: 4-bit (q <= 16) and 5-bit (q <= 32) codes, several chunks per row and a ragged last warp
PACKED_CASES = [
    (64, 9, 1, 1, 0.99, 40),
    (128, 24, 4, 0, 1.002, 30),
    (192, 16, 6, 1, 0.7, 25),
    (320, 32, 8, 1, 1.2, 15),
    (2112, 24, 2, 1, 0.995, 4),
]


@pytest.mark.parametrize("stream", [1, 2])
@pytest.mark.parametrize("L,q,seed,init,f,n", PACKED_CASES)
def test_delta_series_packed_layout(pb, L, q, seed, init, f, n, stream):
    T = f * workloads.t_c(q)
    g = pb.Potts(L, q, seed, init, layout=pb.LAYOUT_PACKED)
    g.potts_set_stream_spec(stream)
    o = oracle.OraclePotts(L, q, seed, init, threads=4, stream=stream)
    E0 = o.energy()
    dE = g.potts_sweep_delta(T, n)
    Eo, _ = o.sweep_measured(T, n, 1, hist=False)
    assert (E0 + np.cumsum(dE) == Eo).all()
    assert (g.potts_download() == o.spins()).all()
    assert g.potts_energy() == int(Eo[-1])
    assert g.potts_sweep_count() == o.t == n


def test_delta_arguments(pb):
    g = pb.Potts(64, 9, 1, pb.INIT_RANDOM)
    with pytest.raises(pb.PottsError) as e:
        g.potts_sweep_delta(-1.0, 1)
    assert e.value.code == pb.ERR_ARG
    assert g.potts_sweep_delta(1.0, 0).shape == (0,)
    assert g.potts_sweep_count() == 0


def test_delta_full_size_invariant(pb):
    """R7 / R8 at BASELINE configs[4]'s size (L = 32768, 2^30 spins), where the oracle cannot follow every sweep:
    E(0) + sum of the accepted moves' d == the recounted Eq. 1 energy (potts_energy, itself compared with the
    oracle at this size in test_gpu_fullsize.py), and the chain is the one the plain streaming kernel makes."""
    w = workloads.CONFIGS[5]
    T = w.temperatures[0]
    g = pb.Potts(w.L, w.q, w.seed, w.init)
    E0 = g.potts_energy()
    dE = g.potts_sweep_delta(T, 4)
    assert E0 + int(dE.sum()) == g.potts_energy()
    assert (dE < 0).all()                                   # cooling a random start below T_c: the energy falls
    r = pb.Potts(w.L, w.q, w.seed, w.init)
    r.potts_set_option("variant", 1)
    Er, _ = r.potts_sweep_measured(T, 4, 1, hist=False)
    assert (E0 + np.cumsum(dE) == Er).all()
    h = r.potts_histogram()
    assert (g.potts_histogram() == h).all() and int(h.sum()) == w.L * w.L


def test_delta_of_a_long_resident_call_is_one_launch(pb):
    """For lattices the persistent kernels hold, potts_sweep_delta is ONE launch per call (not two per sweep)."""
    g = pb.Potts(1024, 6, 7, pb.INIT_ORDERED)
    n0 = g.potts_launch_count()
    dE = g.potts_sweep_delta(1.005 * workloads.t_c(6), 300)
    assert g.potts_launch_count() - n0 == 1
    o = oracle.OraclePotts(1024, 6, 7, 0, threads=8)
    Eo, _ = o.sweep_measured(1.005 * workloads.t_c(6), 300, 1, hist=False)
    assert (-2 * 1024 * 1024 + np.cumsum(dE) == Eo).all()
    assert (g.potts_download() == o.spins()).all()


def test_batch_delta_every_replica(pb):
    """potts_batch_sweep_delta: every replica's series against its own oracle's recounted energies."""
    L, q, n, ns = 64, 9, 5, 30
    seeds = [50 + 3 * r for r in range(n)]
    Ts = [(0.9 + 0.05 * r) * workloads.t_c(q) for r in range(n)]
    b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
    dE = b.potts_batch_sweep_delta(Ts, ns)
    assert dE.shape == (n, ns)
    for r in range(n):
        o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_RANDOM)
        E0 = o.energy()
        Eo, _ = o.sweep_measured(Ts[r], ns, 1, hist=False)
        assert (E0 + np.cumsum(dE[r]) == Eo).all()
        assert (b.potts_batch_download(r) == o.spins()).all()
    assert b.potts_batch_sweep_count() == ns
