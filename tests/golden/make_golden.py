"""Writes tests/golden/oracle_tiny_jacobian.txt: the oracle's own output on two seeded tiny mechanisms.

    python tests/golden/make_golden.py

This is a REGRESSION fixture for the oracle (it freezes oracle/oracle.c's arithmetic so that an
accidental change shows up), not a pin to the paper: the paper prints no worked numeric
example, so value-level parity with its runs stays "unpinned".  The script calls
only oracle/ and the seeded input generators; nothing here comes from the CUDA path.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.oracle import Oracle                      # noqa: E402
from paper_1605_03262_b200 import synth               # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny_jacobian.txt")
CASES = [(0, 3), (3, 2)]                              # (tiny mechanism seed, number of states)


def main():
    lines = ["# oracle regression fixture; written by tests/golden/make_golden.py (calls only oracle/)",
             "# per case: 'case <seed> <n_states> <n_species>', then per state one line of dPhi/dt (Ns+1 values)",
             "# and one line of the Jacobian ((Ns+1)^2 values, column-major), '%.17e'"]
    for seed, n in CASES:
        m = synth.make_tiny_mechanism(seed)
        T, P, Y = synth.make_states(m.n_species, n, 4242 + seed)
        o = Oracle(m)
        src = o.source(T, P, Y)
        J = o.jacobian(T, P, Y)
        lines.append("case %d %d %d" % (seed, n, m.n_species))
        for s in range(n):
            lines.append(" ".join("%.17e" % v for v in src["dydt"][s]))
            lines.append(" ".join("%.17e" % v for v in J[s]))
    with open(OUT, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("wrote", OUT)


if __name__ == "__main__":
    main()
