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
