"""GPU parity of the first + second neighbour generalisation (potts8_*, reading S17) against
its oracle (-m gpu).  Integer work only: equality of every spin, energy and histogram after every sweep."""
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


# (L, q, init, T, seed, sweeps): every compare mode, the smallest lattice (one word per plane row), L not a power of
# two, ordered / random starts, cold / hot
CASES = [
    (12, 2, 1, 4.0, 11, 20),
    (24, 9, 1, 2.0, 1, 16),
    (48, 6, 0, 2.6, 7, 12),
    (96, 24, 1, 1.6, 4, 10),
    (132, 3, 1, 3.0, 3, 8),
    (60, 200, 1, 1.5, 9, 8),
    (36, 129, 1, 80.0, 6, 8),
    (36, 5, 1, 0.05, 10, 8),
    (768, 9, 1, 2.0, 5, 3),
]


@pytest.mark.parametrize("L,q,init,T,seed,n", CASES)
def test_nnn_every_sweep_spins_energy_histogram(pb, L, q, init, T, seed, n):
    g = pb.Potts8(L, q, seed, init)
    o = oracle.OraclePotts8(L, q, seed, init, threads=8)
    assert (g.potts8_download() == o.spins()).all()
    assert g.potts8_energy() == o.energy()
    assert (g.potts8_histogram() == o.histogram()).all()
    Eg, Hg = g.potts8_sweep_measured(T, n, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts8_download() == o.spins()).all()
    assert g.potts8_energy() == o.energy_incremental()
    assert g.potts8_sweep_count() == o.t == n


def test_nnn_split_calls_upload_restart_and_arguments(pb):
    L, q, seed, T = 96, 9, (7 << 36) | 5, 2.1
    g = pb.Potts8(L, q, seed, pb.INIT_RANDOM)
    o = oracle.OraclePotts8(L, q, seed, pb.INIT_RANDOM, threads=8)
    g.potts8_sweep(T, 3)
    Eg, Hg = g.potts8_sweep_measured(T, 6, 3, hist=True)
    o.sweep(T, 3)
    Eo, Ho = o.sweep_measured(T, 6, 3, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all() and Eg.shape == (2,)
    s0 = workloads.synthetic_spins(L, q, 31, "domains")
    g.potts8_upload(s0)
    g.potts8_set_sweep_count(1000)
    o.set_state(s0, 1000)
    assert g.potts8_energy() == o.energy()
    g.potts8_sweep(T, 2); o.sweep(T, 2)
    assert (g.potts8_download() == o.spins()).all()
    for Lb, qb, code in ((10, 9, pb.ERR_ARG), (18, 9, pb.ERR_UNSUPPORTED), (24, 1, pb.ERR_ARG)):
        with pytest.raises(pb.PottsError) as e:
            pb.Potts8(Lb, qb, 1)
        assert e.value.code == code
    c = pb.Potts8(24, 9, 1, pb.INIT_ORDERED)
    assert c.potts8_energy() == -4 * 24 * 24
    E, H = c.potts8_sweep_measured(0.01, 4, 1)
    assert (E == -4 * 24 * 24).all() and (H[:, 0] == 24 * 24).all()
    with pytest.raises(pb.PottsError):
        c.potts8_sweep_measured(1.0, 5, 2)


# the row-walking kernel k_sweep8_rows_u8 (automatic for L % 48 == 0): every compare mode, the three column residues
# of every launch set, exact / one-compare acceptance (T = 0.05 has zero thresholds), rows narrower than a warp with
# idle lanes (L = 144: 3 chunks on 4 lanes), rows per window 1 .. 16, several column blocks (L = 3072: 64 chunks);
# words = -1: the one-word-per-thread kernel at the same sizes
ROWS_CASES = [
    (48, 2, 1, 4.0, 11, 8),
    (96, 9, 1, 2.0, 1, 6),
    (144, 6, 0, 2.6, 7, 6),
    (96, 24, 1, 1.6, 4, 6),
    (192, 200, 1, 1.5, 9, 4),
    (48, 129, 1, 80.0, 6, 6),
    (96, 5, 1, 0.05, 10, 6),
]


@pytest.mark.parametrize("words,rows", [(0, 0), (4, 1), (4, 2), (4, 8), (4, 16), (-1, 0)])
@pytest.mark.parametrize("L,q,init,T,seed,n", ROWS_CASES)
def test_nnn_row_walking_kernel(pb, L, q, init, T, seed, n, words, rows):
    g = pb.Potts8(L, q, seed, init)
    g.potts8_set_option("stream_words", words)
    g.potts8_set_option("stream_rows", rows)
    o = oracle.OraclePotts8(L, q, seed, init, threads=8)
    Eg, Hg = g.potts8_sweep_measured(T, n, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    assert (g.potts8_download() == o.spins()).all()


def test_nnn_options_and_kernels_agree_at_several_column_blocks(pb):
    g = pb.Potts8(48, 9, 1)
    for key, value in (("stream_words", 2), ("stream_rows", 3), ("nonsense", 1)):
        with pytest.raises(pb.PottsError) as e:
            g.potts8_set_option(key, value)
        assert e.value.code == pb.ERR_ARG
    L, q, T, seed = 3072, 9, 2.0, 21
    a = pb.Potts8(L, q, seed, pb.INIT_RANDOM)
    b = pb.Potts8(L, q, seed, pb.INIT_RANDOM)
    b.potts8_set_option("stream_words", -1)
    o = oracle.OraclePotts8(L, q, seed, pb.INIT_RANDOM, threads=16)
    Ea, Ha = a.potts8_sweep_measured(T, 2, 1, hist=True)
    Eb, Hb = b.potts8_sweep_measured(T, 2, 1, hist=True)
    Eo, Ho = o.sweep_measured(T, 2, 1, hist=True)
    assert (Ea == Eo).all() and (Ha == Ho).all() and (Eb == Eo).all() and (Hb == Ho).all()
    assert (a.potts8_download() == o.spins()).all() and (b.potts8_download() == o.spins()).all()
