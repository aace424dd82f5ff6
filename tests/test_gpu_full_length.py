"""Full-length parity of the BASELINE.json configurations: every sweep of the run, GPU against the oracle (-m gpu).

Marked `slow` (hours of oracle time for the large lattices): collected, but skipped unless POTTS_RUN_SLOW=1, e.g.

    POTTS_RUN_SLOW=1 python -m pytest tests/test_gpu_full_length.py -m gpu -q -k cfg2
    POTTS_FULL_LENGTH_LIMIT=100 POTTS_RUN_SLOW=1 python -m pytest tests/test_gpu_full_length.py -m gpu -q -k cfg5

Both sides run the configuration's temperature ladder from its start state in chunks of `chunk` sweeps; after every
chunk the energy (and histogram) series of the chunk are compared entry by entry, and every `spin_every` chunks the whole
spin configuration.  The oracle runs in its row-parallel mode (same bits as serial, tests/test_oracle_pins.py).
POTTS_FULL_LENGTH_LIMIT bounds the number of sweeps.  Records: profiles/r01d_full_length_parity.md (round 1),
profiles/r02d_full_length_parity.md and r02j_full_length_parity.md (round 2; r02j: all five complete).
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402,F401
import pytest  # noqa: E402

import oracle  # noqa: E402
import workloads  # noqa: E402

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5], ids=lambda k: f"cfg{k}")
def test_full_length_parity(k):
    import paper_1101_0876_b200 as pb
    limit = int(os.environ["POTTS_FULL_LENGTH_LIMIT"]) if os.environ.get("POTTS_FULL_LENGTH_LIMIT") else None
    w = workloads.CONFIGS[k]
    threads = len(os.sched_getaffinity(0))
    g = pb.Potts(w.L, w.q, w.seed, w.init, layout=pb.LAYOUT_PACKED if w.packed else pb.LAYOUT_U8)
    o = oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=threads)
    chunk = max(w.every, (200 if w.L <= 1024 else 50 if w.L <= 8192 else 10) // w.every * w.every)
    spin_every = 10
    t0 = time.time()
    done = compared = spin_checks = 0
    assert (g.potts_download() == o.spins()).all()
    for T in w.temperatures:
        left = w.sweeps_per_t
        nchunk = 0
        while left > 0 and (limit is None or done < limit):
            n = min(chunk, left)
            Eg, Hg = g.potts_sweep_measured(T, n, w.every, hist=w.hist)
            Eo, Ho = o.sweep_measured(T, n, w.every, hist=w.hist)
            assert (Eg == Eo).all(), (T, done)
            if w.hist:
                assert (Hg == Ho).all(), (T, done)
            compared += len(Eg)
            left -= n
            done += n
            nchunk += 1
            if nchunk % spin_every == 0 or left == 0:
                assert (g.potts_download() == o.spins()).all(), (T, done)
                spin_checks += 1
                print(f"  t = {done}: E = {int(Eo[-1])}, {time.time() - t0:.0f} s", flush=True)
    print(f"FULL-LENGTH PARITY OK {w.name}: {done} sweeps ({done * w.L * w.L:.3e} updates), {compared} series samples "
          f"and {spin_checks} full configurations identical, kernel variant resident_ctas={g.potts_get_option('resident_active')}, "
          f"oracle threads={threads}, {time.time() - t0:.0f} s", flush=True)

