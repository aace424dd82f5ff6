"""GPU parity of the 3D generalisation (potts3_*, reading S16) against the 3D oracle (-m gpu).

Integer work only: the bar is equality of every spin, every energy and every histogram after every sweep.
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


# (L, q, init, T, seed, sweeps): every compare mode (q <= 8, <= 16, <= 128, <= 256), one chunk per row (L = 32), rows
# shorter than a warp (L = 64, 96: lanes of one warp sit in different rows and planes), L not a power of two, ordered
# and random starts, cold / hot / near the 3D transition (T_c(q=2) = 2.2558 with J_Potts = 2 J_Ising)
CASES = [
    (32, 2, 1, 2.25, 11, 12),
    (32, 9, 1, 1.2, 1, 12),
    (64, 6, 0, 1.6, 7, 8),
    (64, 24, 1, 1.0, 4, 8),
    (96, 3, 1, 1.8163, 3, 5),
    (64, 200, 1, 0.9, 9, 6),
    (32, 129, 1, 50.0, 6, 8),
    (32, 5, 1, 0.05, 10, 8),
    (128, 9, 1, 1.3, 5, 3),
]


@pytest.mark.parametrize("L,q,init,T,seed,n", CASES)
def test_3d_every_sweep_spins_energy_histogram(pb, L, q, init, T, seed, n):
    g = pb.Potts3D(L, q, seed, init)
    o = oracle.OraclePotts3D(L, q, seed, init, threads=8)
    assert (g.potts3_download() == o.spins()).all()                  # start state (R9')
    assert g.potts3_energy() == o.energy()
    assert (g.potts3_histogram() == o.histogram()).all()
    Eg, Hg = g.potts3_sweep_measured(T, n, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts3_download() == o.spins()).all()
    assert g.potts3_energy() == o.energy_incremental()
    assert g.potts3_sweep_count() == o.t == n


def test_3d_split_calls_cadence_upload_restart(pb):
    L, q, seed, T = 64, 9, (5 << 40) | 3, 1.25
    g = pb.Potts3D(L, q, seed, pb.INIT_RANDOM)
    o = oracle.OraclePotts3D(L, q, seed, pb.INIT_RANDOM, threads=8)
    g.potts3_sweep(T, 3)
    Eg, Hg = g.potts3_sweep_measured(T, 6, 3, hist=True)             # every third sweep
    o.sweep(T, 3)
    Eo, Ho = o.sweep_measured(T, 6, 3, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all() and Eg.shape == (2,)
    # restart another handle from the downloaded state: state = spins + t
    S = g.potts3_download()
    g2 = pb.Potts3D(L, q, seed, pb.INIT_ORDERED)
    g2.potts3_upload(S)
    g2.potts3_set_sweep_count(g.potts3_sweep_count())
    g.potts3_sweep(T, 2); g2.potts3_sweep(T, 2); o.sweep(T, 2)
    assert (g.potts3_download() == o.spins()).all() and (g2.potts3_download() == o.spins()).all()
    # synthetic upload (domains), then the chain from there
    s0 = np.stack([workloads.synthetic_spins(L, q, 20 + z // 16, "domains") for z in range(L)])
    g2.potts3_upload(s0)
    g2.potts3_set_sweep_count(100)
    o.set_state(s0, 100)
    assert g2.potts3_energy() == o.energy()
    g2.potts3_sweep(T, 2); o.sweep(T, 2)
    assert (g2.potts3_download() == o.spins()).all()


def test_3d_arguments(pb):
    for L, q, code in ((30, 9, pb.ERR_UNSUPPORTED), (33, 9, pb.ERR_ARG), (32, 1, pb.ERR_ARG), (32, 257, pb.ERR_ARG)):
        with pytest.raises(pb.PottsError) as e:
            pb.Potts3D(L, q, 1)
        assert e.value.code == code
    g = pb.Potts3D(32, 9, 1, pb.INIT_ORDERED)
    assert g.potts3_energy() == -3 * 32 ** 3
    for bad in (dict(T=-1.0, n=1, every=1), dict(T=1.0, n=5, every=2), dict(T=1.0, n=-1, every=1)):
        with pytest.raises(pb.PottsError) as e:
            g.potts3_sweep_measured(bad["T"], bad["n"], bad["every"])
        assert e.value.code == pb.ERR_ARG
    assert g.potts3_sweep_count() == 0
    E, H = g.potts3_sweep_measured(0.01, 4, 1)                        # T -> 0: the ordered state never moves
    assert (E == -3 * 32 ** 3).all() and (H[:, 0] == 32 ** 3).all()
    bad = np.zeros((32, 32, 32), dtype=np.uint8); bad[3, 4, 5] = 9
    with pytest.raises(pb.PottsError):
        g.potts3_upload(bad)


def test_3d_large_lattice_prefix(pb):
    """L = 256 (1.7e7 sites): start state, two sweeps element by element, fused-free energy and histogram."""
    L, q, seed, T = 256, 9, 5, 1.3
    g = pb.Potts3D(L, q, seed, pb.INIT_RANDOM)
    o = oracle.OraclePotts3D(L, q, seed, pb.INIT_RANDOM, threads=16)
    assert (g.potts3_download() == o.spins()).all()
    Eg, Hg = g.potts3_sweep_measured(T, 2, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, 2, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts3_download() == o.spins()).all()


# the row-walking kernel k_sweep3_rows_u8 in every shape (several windows per warp at these sizes: the point is every template
# argument -- compare mode, colour, words per lane, exact / one-compare acceptance (T = 0.05 has zero thresholds) --
# and every rows-per-warp value against the oracle), and the one-chunk-per-thread kernel forced where the other is automatic
@pytest.mark.parametrize("words,rows", [(1, 2), (2, 4), (4, 8), (1, 32), (4, 0), (2, 16), (-1, 0)])
@pytest.mark.parametrize("L,q,init,T,seed,n", CASES[:8])
def test_3d_row_walking_kernel(pb, L, q, init, T, seed, n, words, rows):
    n = min(n, 6)
    g = pb.Potts3D(L, q, seed, init)
    g.potts3_set_option("stream_words", words)
    g.potts3_set_option("stream_rows", rows)
    o = oracle.OraclePotts3D(L, q, seed, init, threads=8)
    Eg, Hg = g.potts3_sweep_measured(T, n, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts3_download() == o.spins()).all()


def test_3d_options(pb):
    g = pb.Potts3D(32, 9, 1)
    for key, value in (("stream_words", 3), ("stream_rows", 5), ("nonsense", 1)):
        with pytest.raises(pb.PottsError) as e:
            g.potts3_set_option(key, value)
        assert e.value.code == pb.ERR_ARG


@pytest.mark.parametrize("L,q,words", [(256, 9, 0), (256, 24, 2), (512, 6, 0), (512, 9, 1)])
def test_3d_kernels_agree_where_lanes_are_full(pb, L, q, words):
    """L = 256 / 512: the automatic choice (4 words per lane: two / four windows per warp) and narrower lanes (words = 1
    at L = 512: two column blocks) against the one-chunk-per-thread kernel, which the cases above pin to the oracle."""
    T, seed = 1.3, 77
    a = pb.Potts3D(L, q, seed, pb.INIT_RANDOM)
    b = pb.Potts3D(L, q, seed, pb.INIT_RANDOM)
    a.potts3_set_option("stream_words", words)
    b.potts3_set_option("stream_words", -1)
    Ea, Ha = a.potts3_sweep_measured(T, 3, 1, hist=True)
    Eb, Hb = b.potts3_sweep_measured(T, 3, 1, hist=True)
    assert (Ea == Eb).all() and (Ha == Hb).all()
    assert a.potts3_launch_count() == b.potts3_launch_count()
    assert (a.potts3_download() == b.potts3_download()).all()
