"""The frozen oracle outputs of tests/golden/ (written by tests/golden/make_golden.py, which
calls only oracle/).  The paper prints no worked example, so no fixture cites the paper."""
import os

import numpy as np

import lattice_inputs as li
import oracle as orc

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c1_smear_step.txt")


def _read():
    rows = {}
    for line in open(GOLD):
        if line.startswith("#"):
            continue
        p = line.split()
        if p[0].startswith("plaq"):
            rows[p[0]] = float.fromhex(p[1])
        else:
            rows[(p[0], int(p[1].split("=")[1]), int(p[2].split("=")[1]))] = np.array([float.fromhex(v) for v in p[3:]])
    return rows


def test_c1_generator_and_oracle_match_golden():
    rows = _read()
    dims = li.CONFIGS["c1"]["dims"]
    u = [t.numpy() for t in li.gauge_field(1, dims, "f64", "haar")]
    out = orc.smear_step(dims, u, 0.5, "t64")
    # the generator uses libm log/sin/cos: allow a few ulp across libm versions, nothing more
    assert abs(orc.plaquette_avg(dims, u, "t64") - rows["plaq_avg_in"]) < 1e-14
    assert abs(orc.plaquette_avg(dims, out, "t64") - rows["plaq_avg_out"]) < 1e-14
    for key, want in rows.items():
        if isinstance(key, tuple):
            which, s, mu = key
            got = (out if which == "uout" else u)[mu][s].ravel()
            assert np.abs(got - want).max() < 1e-14
