"""Writes tests/golden/cfg1_oracle_sample.txt by calling ONLY oracle/ (and the seeded
input generator).  Regression fixture: guards the oracle against accidental change.
Not a paper value -- the paper prints no H element.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2603_21835_b200 import workloads  # noqa: E402

w = workloads.make("si8_sz")
H, (bi, bj, bR, off) = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V)
sel = np.random.default_rng(123).choice(len(bi), 12, replace=False)
path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle_sample.txt")
with open(path, "w") as f:
    f.write("# oracle (gint_oracle.c) output on workload si8_sz (BASELINE.json configs[0]), Eq. 45 PAPER.md:393-398\n")
    f.write("# input sha256 %s\n" % w.sha256())
    f.write("# nblocks %d hlen %d\n" % (len(bi), off[-1]))
    f.write("# I J R1 R2 R3 mu nu H\n")
    for b in sorted(sel):
        blk = H[off[b]:off[b + 1]].reshape(4, 4)
        for mu, nu in ((0, 0), (0, 2), (1, 3), (3, 1)):
            f.write("%d %d %d %d %d %d %d %.17e\n" % (bi[b], bj[b], bR[b, 0], bR[b, 1], bR[b, 2], mu, nu, blk[mu, nu]))
print(path)
