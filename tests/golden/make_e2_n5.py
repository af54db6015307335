"""Writes tests/golden/e2_n5_single_helicity.txt: (A, B, D) of g g -> t t~ g g g for ONE helicity configuration from the
oracle's explicit-colour engine E2 (8^5 x 9 colour assignments, no colour basis, no recursion; about five minutes on one
core). Calls only oracle/ and the seeded input generator. tests/test_oracle_colour.py compares the colour-ordered engine
E1 (the one every parity test uses at n = 5) with these numbers.

  python tests/golden/make_e2_n5.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as O  # noqa: E402
from trex_inputs import default_theta, make_config  # noqa: E402

HEL, EVENT = 77, 0


def main():
    w = make_config(5, n=8)
    th = default_theta()
    b = O.abd(4, w.momenta[:, :, EVENT:EVENT + 1], th, engine=2, hel_only=HEL)[0]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "e2_n5_single_helicity.txt")
    with open(out, "w") as fh:
        fh.write("# (A, B, D) of |M|^2 = A + kappa B + kappa^2 D, g g > t t~ g g g, helicity index %d, event %d of make_config(5, n=8),\n" % (HEL, EVENT))
        fh.write("# default_theta(); oracle engine E2 (explicit colour). Written by tests/golden/make_e2_n5.py (oracle only).\n")
        fh.write(" ".join(repr(float(x)) for x in b) + "\n")
    print(out, b)


if __name__ == "__main__":
    main()
