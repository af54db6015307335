"""Writes profiles/oracle_flops_per_event.json: the floating-point operations per reweighted event of the oracle's plain
algorithm (explicit 4 x 4 Dirac matrices, every helicity and every ordering from scratch, old and new parameter point
evaluated separately), counted by instantiating it on a counting scalar type. Calls only oracle/ and the seeded input
generators.  `python -m oracle.count_flops`"""
import json
import os

import numpy as np

from oracle import oracle as O
from trex_inputs import make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    out = {"_comment": "oracle/oracle.py count_flops on the first event of each class (seeded configs of trex_inputs); "
                       "add/mul/div/sqrt are operations on real numbers, flop = their sum; written by oracle/count_flops.py"}
    for cfg in (1, 2, 3, 4, 5):
        w = make_config(cfg, n=64)
        for sp in w.classes:
            i = int(np.where(w.keys == sp.key)[0][0])
            c = O.count_flops(sp.sid, w.momenta[:, :, i], w.theta_old, w.theta_new)
            out["cfg%d %s" % (cfg, sp.name)] = c
    with open(os.path.join(ROOT, "profiles", "oracle_flops_per_event.json"), "w") as fh:
        json.dump(out, fh, indent=1)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
