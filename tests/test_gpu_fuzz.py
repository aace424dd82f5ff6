"""Seeded random sweep over (L, q, T, seed, start, layout, launch shape): every case must equal the oracle bit for bit (-m gpu).

The fixed cases of test_gpu_parity.py pick the edges by hand; this one walks the space between them (all compare modes,
both histogram table kinds, row splits that leave CTAs with 1..many rows, lattices whose plane rows are not a multiple
of a warp, packed and byte layouts) with a fixed seed, so a failure is reproducible.
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


def _cases(n, seed):
    rng = np.random.default_rng(seed)
    qs = [2, 3, 4, 6, 8, 9, 12, 16, 17, 24, 32, 33, 48, 64, 65, 96, 128, 129, 192, 256]
    out = []
    for k in range(n):
        q = int(rng.choice(qs))
        packed = bool(q <= 32 and rng.random() < 0.3)
        L = int(rng.choice([64, 128, 192, 256, 320]) if packed else rng.choice([32, 64, 96, 128, 160, 224, 256, 288, 384, 512]))
        shape = {}
        if not packed:
            variant = int(rng.choice([1, 2, 2, 2, 3, 0]))
            shape["variant"] = variant
            if variant == 3:
                shape["cluster_ctas"] = int(rng.choice([0, 1, 2, 3, 5, 8, 11, 16]))
            if variant == 2:
                shape["resident_ctas"] = int(rng.choice([0, 1, 2, 3, 5, 8, 13, 31, 64, 148]))
                shape["resident_words"] = int(rng.choice([0, 1, 2]))
        out.append(dict(L=L, q=q, packed=packed, shape=shape, seed=int(rng.integers(0, 2 ** 63)),
                        init=int(rng.integers(0, 2)), f=float(rng.choice([0.05, 0.7, 0.95, 1.0, 1.05, 1.5, 30.0])),
                        nsweeps=int(rng.choice([4, 6, 9])), every=int(rng.choice([1, 1, 3]))))
    return out


@pytest.mark.parametrize("case", _cases(48, 20261104), ids=lambda c: f"L{c['L']}q{c['q']}{'p' if c['packed'] else 'u'}")
def test_random_case_matches_oracle(pb, case):
    L, q = case["L"], case["q"]
    g = pb.Potts(L, q, case["seed"], case["init"], layout=pb.LAYOUT_PACKED if case["packed"] else pb.LAYOUT_U8)
    for k, v in case["shape"].items():
        g.potts_set_option(k, v)
    if (case["shape"].get("variant") == 2 and g.potts_get_option("resident_active") == 0) or \
            (case["shape"].get("variant") == 3 and g.potts_get_option("cluster_active") == 0):
        pytest.skip("forced launch shape cannot hold this lattice")
    o = oracle.OraclePotts(L, q, case["seed"], case["init"])
    T = case["f"] * workloads.t_c(q)
    n = case["nsweeps"] // case["every"] * case["every"]
    Eg, Hg = g.potts_sweep_measured(T, n, case["every"], hist=True)
    Eo, Ho = o.sweep_measured(T, n, case["every"], hist=True)
    assert (Eg == Eo).all() and (Hg == Ho).all()
    g.potts_sweep(T, 2)
    o.sweep(T, 2)
    assert (g.potts_download() == o.spins()).all()
    assert g.potts_energy() == o.energy() and (g.potts_histogram() == o.histogram()).all()


@pytest.mark.slow
def test_cluster_kernel_soak(pb):
    """Randomised soak of the cluster kernel's lock-free packet exchange (potts_cluster.cuh): for POTTS_SOAK_SECONDS
    (default 60) seconds random (L <= 288, q, cluster size, stream definition, seed, temperature) runs of three calls of
    random length and kind (measured, plain, energy-change series) against the oracle, each followed by a second handle
    that repeats the chain in one call (determinism).  Collected but skipped unless POTTS_RUN_SLOW=1; record:
    profiles/r02h_cluster_exchange.md."""
    import os
    import time
    seconds = float(os.environ.get("POTTS_SOAK_SECONDS", "60"))
    rng = np.random.default_rng(12345)
    t0, n_ok = time.time(), 0
    while time.time() - t0 < seconds:
        L = int(rng.choice([32, 64, 96, 128, 160, 192, 256, 288]))
        q = int(rng.choice([2, 3, 6, 9, 16, 17, 24, 128, 129, 256]))
        G = int(rng.choice([0, 1, 2, 3, 4, 5, 7, 8, 12, 16]))
        st = int(rng.choice([1, 2]))
        seed = int(rng.integers(1, 2 ** 62))
        T = float(rng.choice([0.5, 0.9, 0.99, 1.0, 1.05, 2.0])) * workloads.t_c(q)
        case = (L, q, G, st, seed, T)

        def handle():
            g = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
            g.potts_set_option("variant", 3)
            g.potts_set_option("cluster_ctas", G)
            if st == 2:
                g.potts_set_stream_spec(2)
            return g
        g = handle()
        if g.potts_get_option("cluster_active") == 0:
            g.close()
            continue
        o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM, stream=st, threads=8)
        for _ in range(3):
            n, kind = int(rng.integers(1, 40)), int(rng.integers(0, 3))
            if kind == 0:
                Eg, Hg = g.potts_sweep_measured(T, n, 1, hist=True)
                Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
                assert (Eg == Eo).all() and (Hg == Ho).all(), case
            elif kind == 1:
                g.potts_sweep(T, n)
                o.sweep(T, n)
            else:
                e0, es = o.energy(), []
                d = g.potts_sweep_delta(T, n)
                for _ in range(n):
                    o.sweep(T, 1)
                    es.append(o.energy())
                assert (d == np.diff(np.array([e0] + es, dtype=np.int64))).all(), case
            assert g.potts_energy() == o.energy(), case
        assert (g.potts_download() == o.spins()).all(), case
        g2 = handle()
        g2.potts_sweep(T, int(o.t))
        assert (g2.potts_download() == o.spins()).all(), case
        g.close()
        g2.close()
        n_ok += 1
    print(f"CLUSTER SOAK OK: {n_ok} random cases identical to the oracle and repeatable, {time.time() - t0:.0f} s", flush=True)


@pytest.mark.slow
def test_resident_kernel_large_lattice_soak(pb):
    """Randomised soak of the resident kernel beyond L = 2048, where 64 comm threads share the chunks of a halo row
    (potts_resident.cuh): for POTTS_SOAK_SECONDS (default 60) seconds random (L, q, grid size, words per thread, thread
    rows, stream definition, seed) runs of a few measured sweeps against the oracle.  Collected but skipped unless
    POTTS_RUN_SLOW=1; record: profiles/r02i_occupancy.md."""
    import os
    import time
    seconds = float(os.environ.get("POTTS_SOAK_SECONDS", "60"))
    rng = np.random.default_rng(777)
    threads = len(os.sched_getaffinity(0))
    t0, n_ok = time.time(), 0
    while time.time() - t0 < seconds:
        L = int(rng.choice([2080, 2112, 2304, 2560, 3072, 3104, 3584, 4064, 4096]))
        q = int(rng.choice([2, 6, 9, 16, 24, 129]))
        G = int(rng.choice([0, 37, 64, 100, 111, 147, 148]))
        W = int(rng.choice([0, 2]))
        rows = int(rng.choice([0, 1, 2, 3]))
        st = int(rng.choice([1, 2]))
        seed = int(rng.integers(1, 2 ** 62))
        T = float(rng.choice([0.9, 1.0, 1.1])) * workloads.t_c(q)
        case = (L, q, G, W, rows, st, seed)
        g = pb.Potts(L, q, seed, workloads.INIT_RANDOM)
        for k, v in (("variant", 2), ("resident_ctas", G), ("resident_words", W), ("resident_rows", rows)):
            g.potts_set_option(k, v)
        if st == 2:
            g.potts_set_stream_spec(2)
        if g.potts_get_option("resident_active") == 0:
            g.close()
            continue
        o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM, stream=st, threads=threads)
        n = int(rng.integers(2, 5))
        Eg, Hg = g.potts_sweep_measured(T, n, 1, hist=True)
        Eo, Ho = o.sweep_measured(T, n, 1, hist=True)
        assert (Eg == Eo).all() and (Hg == Ho).all(), case
        assert (g.potts_download() == o.spins()).all(), case
        g.close()
        n_ok += 1
    print(f"RESIDENT SOAK OK: {n_ok} random cases beyond L = 2048 identical to the oracle, {time.time() - t0:.0f} s", flush=True)


@pytest.mark.slow
def test_batch_kernel_soak(pb):
    """Randomised soak of the replica-batch kernel's own body (potts_resident.cuh, k_resident_batch_u8): for
    POTTS_SOAK_SECONDS (default 60) seconds random (L <= 416, q, number of replicas, stream definition, seeds,
    temperatures) batches, a measured call, an energy-change call and the final spins of every replica against the
    oracle.  Collected but skipped unless POTTS_RUN_SLOW=1; record: profiles/r02i_occupancy.md."""
    import os
    import time
    seconds = float(os.environ.get("POTTS_SOAK_SECONDS", "60"))
    rng = np.random.default_rng(4242)
    t0, n_ok = time.time(), 0
    while time.time() - t0 < seconds:
        L = int(rng.choice([32, 64, 96, 128, 160, 192, 224, 256, 320, 416]))
        q = int(rng.choice([2, 3, 6, 9, 16, 17, 24, 129, 256]))
        n = int(rng.integers(1, 7))
        st = int(rng.choice([1, 2]))
        seeds = [int(x) for x in rng.integers(1, 2 ** 62, size=n)]
        Ts = [float(rng.choice([0.5, 0.99, 1.0, 1.05, 2.0])) * workloads.t_c(q) for _ in range(n)]
        case = (L, q, n, st, seeds[0])
        b = pb.PottsBatch(L, q, seeds, workloads.INIT_RANDOM)
        if st == 2:
            b.potts_batch_set_stream_spec(2)
        ns, nd = int(rng.integers(1, 9)), int(rng.integers(1, 6))
        E, H = b.potts_batch_sweep_measured(Ts, ns, 1)
        dE = b.potts_batch_sweep_delta(Ts, nd)
        for r in range(n):
            o = oracle.OraclePotts(L, q, seeds[r], workloads.INIT_RANDOM, stream=st, threads=8)
            Eo, Ho = o.sweep_measured(Ts[r], ns, 1, hist=True)
            assert (E[r] == Eo).all() and (H[r] == Ho).all(), (case, r)
            e0, es = o.energy(), []
            for _ in range(nd):
                o.sweep(Ts[r], 1)
                es.append(o.energy())
            assert (dE[r] == np.diff(np.array([e0] + es, dtype=np.int64))).all(), (case, r)
            assert (b.potts_batch_download(r) == o.spins()).all(), (case, r)
        b.close()
        n_ok += 1
    print(f"BATCH SOAK OK: {n_ok} random batches identical to the oracle, {time.time() - t0:.0f} s", flush=True)
