"""Writes tests/golden/c0_oracle.txt: the oracle's results for BASELINE config 0 (n = 104 real, 32 electrons, seed 0).

    python tests/golden/make_golden.py

Calls only oracle/ and the seeded input generator (which holds none of the method's arithmetic); never the CUDA path.  The
stored values are what the oracle computes for Eq. 5, the Fermi level of the occupations f_i
and D = C diag(f) C^H (Eq. 8; reading C3 of DESIGN.md).  They pin the oracle against silent changes: a
later change of its arithmetic must regenerate this file on purpose and say why in the commit message."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_09058_b200.synth import make_config  # noqa: E402

SAMPLES = [(0, 0), (1, 0), (13, 5), (52, 51), (103, 103), (103, 0), (77, 20), (40, 40)]


def main():
    prob = make_config(0)
    ref = oracle.solve_problem(prob)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c0_oracle.txt")
    with open(path, "w") as f:
        f.write("# config 0 (BASELINE.json configs[0]): n=104 real, 1 item, g=2, 32 electrons, kT=9.5e-4 Ha, seed 0\n")
        f.write("# written by tests/golden/make_golden.py from oracle/ only (Cholesky reduction + cyclic Jacobi, long double)\n")
        f.write("mu %.17e\n" % ref["mu"])
        f.write("trace_DS %.17e\n" % float(np.trace(ref["D"][0] @ prob.S_full(0))))
        f.write("norm_D_F %.17e\n" % float(np.linalg.norm(ref["D"][0])))
        for (i, j) in SAMPLES:
            f.write("D %d %d %.17e\n" % (i, j, ref["D"][0][i, j]))
        for k, e in enumerate(ref["e"][0]):
            f.write("e %d %.17e\n" % (k, e))
    print(path)


if __name__ == "__main__":
    main()
