"""Writes tests/golden/trajectories_stream2.txt: reference energies of the stream-spec v2 chain (R3').

Calls only oracle/ (never the CUDA path).  These values are a regression record of the oracle's v2 mode;
what pins v2's correctness are the exact 4x4 moments, Kaufman's Ising energy and the word-selection checks in
tests/test_oracle_stream2.py.

    python tests/golden/make_stream2_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import math  # noqa: E402

import oracle  # noqa: E402

CASES = [(64, 9, 1, 1, 0.99), (64, 6, 7, 0, 1.005), (8, 3, 42, 1, 1.0)]      # the P10 cases, run with stream = 2
AT = [0, 1, 2, 3, 10, 100]


def main():
    lines = ["# Stream-spec v2 (one Philox block per pair of same-colour sites, DESIGN.md S15): energies at given sweep counts.",
             "# Written by tests/golden/make_stream2_golden.py from oracle/ alone.",
             "# case L q seed init T_factor"]
    for L, q, seed, init, f in CASES:
        T = f / math.log(1.0 + math.sqrt(float(q)))
        o = oracle.OraclePotts(L, q, seed, init, stream=2)
        out, t = [], 0
        for a in AT:
            o.sweep(T, a - t)
            t = a
            out.append(f"{a}:{o.energy()}")
        lines.append(f"case {L} {q} {seed} {'random' if init else 'ordered'} {f}")
        lines.append("E " + " ".join(out))
    with open(os.path.join(HERE, "trajectories_stream2.txt"), "w") as fh:
        fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
