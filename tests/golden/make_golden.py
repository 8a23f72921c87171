"""Writes tests/golden/dhop_2x2x2x2.txt: the oracle's Dhop and Dhop^dagger on a seeded 2^4 x Ls=1
lattice, antiperiodic in time.  Calls only dwf_inputs/ (seeded generators) and oracle/; never the
CUDA path.  The paper prints no worked values for the operator -- it never writes the
operator down -- so this fixture is not a paper value: it freezes the pinned
oracle (tests/test_oracle_pins.py) against accidental change.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import dwf_inputs as gen   # noqa: E402
import oracle              # noqa: E402

DIMS, LS, SEED = (2, 2, 2, 2), 1, 2203


def compute():
    U = gen.gauge_random(DIMS, SEED)
    psi = gen.spinor_gaussian(gen.volume(DIMS), LS, SEED)
    return (oracle.dhop(DIMS, LS, oracle.ANTIPERIODIC_T, U, psi),
            oracle.dhop(DIMS, LS, oracle.ANTIPERIODIC_T, U, psi, dagger=True))


if __name__ == "__main__":
    d, dd = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "dhop_2x2x2x2.txt")
    with open(path, "w") as f:
        f.write("# oracle Dhop (column 1) and Dhop^dagger (column 2), canonical order [site][s][spin][colour][reim]\n")
        f.write(f"# dims {DIMS} Ls {LS} antiperiodic time, gauge_random / spinor_gaussian seed {SEED}; written by make_golden.py\n")
        for a, b in zip(d.ravel(), dd.ravel()):
            f.write(f"{float(a)!r} {float(b)!r}\n")
    print("wrote", path, d.size, "rows")
