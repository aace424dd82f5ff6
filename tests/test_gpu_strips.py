"""GPU parity of the row-strip form of the streaming kernel (potts_strip_*), -m gpu: n strips of one
lattice in ONE process on one GPU (rows copied device to device between the strips' halos; no rank waits for
another) must follow the single-lattice oracle bit for bit, whatever n is."""
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


@pytest.mark.parametrize("L,q,seed,init,f,n,sweeps", [
    (128, 9, 1, 1, 0.99, 1, 6),
    (128, 9, 1, 1, 0.99, 2, 6),
    (128, 9, 1, 1, 0.99, 4, 6),
    (96, 6, 7, 0, 1.005, 3, 6),
    (256, 24, 4, 1, 1.002, 5, 4),
    (160, 200, 9, 1, 1.3, 2, 4),
    (2048, 9, 3, 1, 0.995, 3, 3),          # several column blocks, many tiles per strip
])
def test_strips_reproduce_the_single_lattice_chain(pb, L, q, seed, init, f, n, sweeps):
    from paper_1101_0876_b200 import strips
    T = f * workloads.t_c(q)
    o = oracle.OraclePotts(L, q, seed, init, threads=8)
    run = strips.LocalStrips(L, q, seed, init, n)
    assert (run.download() == o.spins()).all()
    E0, H0 = run.energy_histogram()
    assert E0 == o.energy() and (H0 == o.histogram()).all()
    E, H = run.sweep(T, sweeps, every=1)
    Eo, Ho = o.sweep_measured(T, sweeps, 1, hist=True)
    assert (E == Eo).all() and (H == Ho).all()
    run.sweep(T, 2)                                   # unsampled sweeps, then the standalone partial sums
    o.sweep(T, 2)
    assert (run.download() == o.spins()).all()
    E1, H1 = run.energy_histogram()
    assert E1 == o.energy() and (H1 == o.histogram()).all()
    run.close()


def test_strip_arguments(pb):
    from paper_1101_0876_b200 import strips
    with pytest.raises(pb.PottsError) as e:
        strips.GpuStrip(128, 9, 1, 1, 16, 32)        # row0 not a multiple of 32
    assert e.value.code == pb.ERR_ARG
    with pytest.raises(pb.PottsError):
        strips.GpuStrip(128, 9, 1, 1, 96, 64)        # past the end of the lattice
    s = strips.GpuStrip(128, 9, 1, 1, 32, 64)
    lib = pb.load_library()
    assert lib.potts_sweep(s._h, 1.0, 1) == pb.ERR_UNSUPPORTED     # a strip is advanced half-sweep by half-sweep
    s.close()
