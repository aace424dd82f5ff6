"""potts_measure_noalloc (include/potts.h, "no-allocation entry point") against the existing measurement path.

The entry point computes the energy and histogram of a device lattice with its scratch (colour planes, accumulators)
in one file-scope device array instead of a handle's cudaMalloc'ed workspace.  The existing path is potts_energy /
potts_histogram of a Potts handle holding the same spins; the oracle is asked as well.  Integer work: exact equality.
The calls share the array, so every case makes several calls in a row, of different L and q, and checks each.

This file sorts last on purpose (pytest -x: a failure here hides nothing after it) and must pass
alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

import oracle
import workloads


def test_sizes_beyond_the_static_array_are_rejected_before_any_cuda_call():
    """-m "not gpu": argument errors come back before the library touches CUDA."""
    import ctypes
    import paper_1101_0876_b200 as pb
    lib = pb.load_library()
    fake = ctypes.c_void_p(0x1000)                                    # never dereferenced: the checks come first
    for L, q, code in ((pb.NOALLOC_MAX_L + 32, 9, pb.ERR_UNSUPPORTED), (4096, 9, pb.ERR_UNSUPPORTED), (48, 9, pb.ERR_UNSUPPORTED),
                       (33, 9, pb.ERR_ARG), (64, 1, pb.ERR_ARG), (64, 257, pb.ERR_ARG), (0, 9, pb.ERR_ARG)):
        assert lib.potts_measure_noalloc(fake, L, q, fake, fake, None) == code
    assert lib.potts_measure_noalloc(None, 64, 9, fake, fake, None) == pb.ERR_ARG
    assert lib.potts_measure_noalloc(fake, 64, 9, None, None, None) == pb.ERR_ARG
    assert lib.potts_measure_noalloc(ctypes.c_void_p(0x1004), 64, 9, fake, fake, None) == pb.ERR_ARG      # alignment
    assert lib.potts_measure_noalloc(fake, pb.NOALLOC_MAX_L + 32, 9, fake, fake, None) == pb.ERR_UNSUPPORTED
    assert b"POTTS_NOALLOC_MAX_L" in lib.potts_last_error()


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible")
    import paper_1101_0876_b200 as pb
    pb.load_library()
    return pb, torch


def _existing_path(pb, L, q, seed, init, T, sweeps):
    """A lattice after a few sweeps, and its energy / histogram by the existing path (handle workspace)."""
    g = pb.Potts(L, q, seed, init)
    if sweeps:
        g.potts_sweep(T, sweeps)
    return g.potts_download(), g.potts_energy(), np.asarray(g.potts_histogram(), dtype=np.int64)


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path(gpu):
    pb, torch = gpu
    # large then small then large again: a call must not see what the previous one left in the array
    cases = [(1024, 9, 5, 1, 0.72, 3), (64, 6, 7, 0, 0.81, 5), (2048, 200, 3, 1, 0.4, 1), (96, 2, 1, 1, 1.1, 4), (1024, 9, 5, 1, 0.72, 3)]
    for L, q, seed, init, T, sweeps in cases:
        S, E_ref, H_ref = _existing_path(pb, L, q, seed, init, T, sweeps)
        spins = torch.from_numpy(S).cuda()
        E = torch.full((1,), 12345, dtype=torch.int64, device="cuda")           # stale values the call must overwrite
        H = torch.full((q,), -7, dtype=torch.int64, device="cuda")
        for _ in range(2):                                                        # the same call twice in a row
            pb.potts_measure_noalloc(spins, q, E, H)
            torch.cuda.synchronize()
            assert int(E.item()) == E_ref
            assert (H.cpu().numpy() == H_ref).all() and int(H.sum().item()) == L * L


@pytest.mark.gpu
def test_against_the_oracle_each_output_alone_and_on_a_side_stream(gpu):
    pb, torch = gpu
    L, q = 128, 24
    S = workloads.synthetic_spins(L, q, 11, "domains")
    o = oracle.OraclePotts(L, q, 1, workloads.INIT_ORDERED)
    o.set_state(S, 0)
    spins = torch.from_numpy(np.ascontiguousarray(S)).cuda()
    E = torch.zeros(1, dtype=torch.int64, device="cuda")
    H = torch.zeros(q, dtype=torch.int64, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    pb.potts_measure_noalloc(spins, q, E, None, stream=st.cuda_stream)            # energy alone
    pb.potts_measure_noalloc(spins, q, None, H, stream=st.cuda_stream)            # histogram alone, same stream: ordered
    st.synchronize()
    assert int(E.item()) == o.energy()
    assert (H.cpu().numpy() == o.histogram()).all()


@pytest.mark.gpu
def test_bad_spin_values_mark_the_outputs(gpu):
    pb, torch = gpu
    L, q = 64, 5
    S = workloads.synthetic_spins(L, q, 3, "uniform")
    S[17, 40] = q                                                                 # one value out of range
    spins = torch.from_numpy(np.ascontiguousarray(S)).cuda()
    E = torch.zeros(1, dtype=torch.int64, device="cuda")
    H = torch.zeros(q, dtype=torch.int64, device="cuda")
    pb.potts_measure_noalloc(spins, q, E, H)
    torch.cuda.synchronize()
    assert int(E.item()) == -2 ** 63 and (H.cpu().numpy() == -1).all()
    S[17, 40] = 0                                                                 # the next call starts from a cleared flag
    S2, o = np.ascontiguousarray(S), oracle.OraclePotts(L, q, 1, workloads.INIT_ORDERED)
    o.set_state(S2, 0)
    pb.potts_measure_noalloc(torch.from_numpy(S2).cuda(), q, E, H)
    torch.cuda.synchronize()
    assert int(E.item()) == o.energy() and (H.cpu().numpy() == o.histogram()).all()
