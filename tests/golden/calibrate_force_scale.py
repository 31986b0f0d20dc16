"""Writes tests/golden/force_scale.txt: the per-family multiplier on scale_Z that makes the RMS
force of the random-weight model 1 eV/Ang on the family's own initial positions (DESIGN.md
reading R17).  Calls only oracle/ and workloads/ (never the CUDA path).  The constants are then
copied by hand into workloads/inputs.py FORCE_SCALE; tests/test_workloads.py checks they agree.

Run:  python tests/golden/calibrate_force_scale.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402
from oracle import gmnn_oracle as orc  # noqa: E402


def rms_force_at_unit_scale(w):
    w.model.scale[:] = 1.0
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, w.model.r_cut)
    res = orc.energy_forces(m, w.positions, w.species, w.cell, pairs)
    return float(np.sqrt((res.forces ** 2).mean())), len(pairs) / w.n_atoms


def main():
    rows = []
    for fam, w in (("tiny", wl.tiny_box()), ("ionic_liquid", wl.ionic_liquid_box()),
                   ("li3po4", wl.li3po4_box(1024)), ("li3po4_check_8192", wl.li3po4_box(8192))):
        rms, nbr = rms_force_at_unit_scale(w)
        rows.append((fam, rms, 1.0 / rms, nbr))
        print(fam, rms, 1.0 / rms, nbr)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "force_scale.txt")
    with open(out, "w") as f:
        f.write("# family  rms_force_at_scale_1[eV/Ang]  force_scale=1/rms  mean_neighbours\n")
        f.write("# written by tests/golden/calibrate_force_scale.py (oracle only); reading R17 in DESIGN.md\n")
        for r in rows:
            f.write("%s %.9e %.9e %.4f\n" % r)


if __name__ == "__main__":
    main()
