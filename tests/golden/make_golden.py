"""Writes tests/golden/*.txt.  Calls ONLY lattice_inputs (the seeded generator) and oracle/ --
never the CUDA path.  The paper (arXiv 1105.2279) prints no worked numerical example, field
value or checksum, so there is no paper-cited fixture; these files freeze the
pinned oracle's output on BASELINE.json configs[0] (4^4, fp64, Haar SU(3), seed 1, a=0.5) so that
a later change to the oracle's arithmetic or to the generator cannot go unnoticed.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import lattice_inputs as li  # noqa: E402
import oracle as orc  # noqa: E402


def main():
    dims = li.CONFIGS["c1"]["dims"]
    u = [t.numpy() for t in li.gauge_field(li.CONFIGS["c1"]["seed"], dims, "f64", "haar")]
    out = orc.smear_step(dims, u, 0.5, "t64")
    lines = ["# BASELINE.json configs[0]: 4^4 fp64 Haar SU(3) seed 1, one smear step a=0.5; oracle variant t64",
             "# written by tests/golden/make_golden.py (oracle only); values are C99 hex floats",
             "plaq_avg_in %s" % float(orc.plaquette_avg(dims, u, "t64")).hex(),
             "plaq_avg_out %s" % float(orc.plaquette_avg(dims, out, "t64")).hex()]
    for (s, mu) in [(0, 0), (37, 1), (129, 2), (255, 3)]:
        vals = " ".join(float(v).hex() for v in out[mu][s].ravel())
        lines.append("uout site=%d mu=%d %s" % (s, mu, vals))
        vals = " ".join(float(v).hex() for v in u[mu][s].ravel())
        lines.append("uin site=%d mu=%d %s" % (s, mu, vals))
    with open(os.path.join(HERE, "c1_smear_step.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
