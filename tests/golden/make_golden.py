"""Writes tests/golden/oracle_config1.txt: energy, virial and the first forces of BASELINE.json config 1 (seeded synthetic
input of gen/, PaiNN weights of its seed) as the fp64 oracle computes them.  Calls only gen/ and oracle/ (never the CUDA
path).  The file is a regression guard for the oracle itself: a change to the oracle's arithmetic must re-run this script
and name, in its commit message, the passage of PAPER.md or the DESIGN.md reading that justifies the change.  (PAPER.md
prints no worked numerical example of the PaiNN forward pass -- its numbers are timings and error statistics on datasets
that are not in the container -- so there is no paper-printed fixture; the oracle's pins are the closed forms, invariants
and brute-force checks of tests/test_oracle_pins.py.)

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import gen      # noqa: E402
import oracle   # noqa: E402


def evaluate():
    c = gen.make_config(1)
    m = c["model"]
    blob = gen.make_weights(m["n_species"], m["F"], m["K"], m["T"], m["rc"], seed=m["wseed"])
    r = oracle.compute(blob, c["pos"], c["types"], c["box"], c["n_local"], c["n_ghost"], c["ghost_owner"])
    return c, r


def main():
    c, r = evaluate()
    with open(os.path.join(HERE, "oracle_config1.txt"), "w") as f:
        f.write("# oracle (fp64) on BASELINE.json config 1; written by tests/golden/make_golden.py -- do not edit\n")
        f.write(f"n_atoms {len(c['pos'])}\nn_edges {int(r['n_edges'])}\n")
        f.write(f"energy {float(r['energy']):.17e}\n")
        f.write("virial " + " ".join(f"{x:.17e}" for x in np.asarray(r["virial"]).ravel()) + "\n")
        for a in range(8):
            f.write(f"force {a} " + " ".join(f"{x:.17e}" for x in r["forces"][a]) + "\n")


if __name__ == "__main__":
    main()
