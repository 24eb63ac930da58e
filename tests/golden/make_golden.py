"""Writes tests/golden/tiny_image.txt from the FP64 oracle ALONE (never from the CUDA path).

Run:  python tests/golden/make_golden.py
The paper prints no numeric example (PAPER.md has timing tables only), so this file is a
regression fixture for the oracle, not an external pin: it catches an accidental change of
the oracle's arithmetic.  Input = pdm_inputs.tiny_random_problem(seed=101, nx=12, nz=4, nw=3, L=2, ntab=8).
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle          # noqa: E402
import pdm_inputs      # noqa: E402

if __name__ == "__main__":
    c = pdm_inputs.tiny_random_problem(101, nx=12, nz=4, nw=3, L=2, ntab=8)
    img = oracle.migrate(c)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_image.txt")
    with open(out, "w") as fh:
        fh.write("# oracle image [nz=4][nx=12], tiny_random_problem(101,12,4,3,2,8); "
                 "Eq.(1) PAPER.md:45 + Alg.1 :59-70; written by make_golden.py (oracle only)\n")
        for row in img:
            fh.write(" ".join(float(v).hex() for v in row) + "\n")
    print("wrote", out)
