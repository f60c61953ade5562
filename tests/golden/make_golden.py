"""Writes tests/golden/cfg1_oracle_sample.txt by calling ONLY oracle/ (and the seeded
input generator).  Regression fixture: guards the oracle against accidental change.
Not a paper value -- the paper prints no H element.

The sample is taken where H has signal (the self-image blocks (I,I,R != 0) of this workload are
below 1e-13 max|H| and carry none): the 4 largest on-site blocks (I,I,0) and the 8 largest
neighbour blocks with I < J, four elements each --
the largest diagonal one, the largest off-diagonal one and two more chosen by a seeded draw among the
elements above 1e-4 max|H| -- so that every stored value is >= 1e-4 max|H|.

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
scale = np.abs(H).max()
bmax = np.array([np.abs(H[off[b]:off[b + 1]]).max() for b in range(len(bi))])
zeroR = np.all(bR == 0, axis=1)
groups = [(np.nonzero((bi == bj) & zeroR)[0], 4), (np.nonzero(bi < bj)[0], 8)]
sel = np.concatenate([g[np.argsort(-bmax[g], kind="stable")[:n]] for g, n in groups])
rng = np.random.default_rng(123)
path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle_sample.txt")
with open(path, "w") as f:
    f.write("# oracle (gint_oracle.c) output on workload si8_sz (BASELINE.json configs[0]), Eq. 45 PAPER.md:393-398\n")
    f.write("# input sha256 %s\n" % w.sha256())
    f.write("# nblocks %d hlen %d max|H| %.17e\n" % (len(bi), off[-1], scale))
    f.write("# I J R1 R2 R3 mu nu H\n")
    for b in sorted(sel):
        blk = H[off[b]:off[b + 1]].reshape(4, 4)
        a = np.abs(blk)
        offd = a.copy()
        offd[np.arange(4), np.arange(4)] = 0.0
        big = [(int(np.argmax(np.diag(a))),) * 2, tuple(int(x) for x in np.unravel_index(np.argmax(offd), a.shape))]
        cand = [(int(m), int(n)) for m, n in zip(*np.nonzero(a >= 1e-4 * scale)) if (int(m), int(n)) not in big]
        for i in rng.choice(len(cand), 2, replace=False):
            big.append(cand[int(i)])
        for mu, nu in big:
            assert a[mu, nu] >= 1e-4 * scale
            f.write("%d %d %d %d %d %d %d %.17e\n" % (bi[b], bj[b], bR[b, 0], bR[b, 1], bR[b, 2], mu, nu, blk[mu, nu]))
print(path)
