"""Small test-side utilities (no method arithmetic)."""
import numpy as np

from paper_2603_21835_b200 import workloads as wl


def gaussian_species(shells, rcut, dr=0.01, name="g"):
    """Species whose radial tables are pure r^l exp(-alpha r^2) (for closed-form pins)."""
    ls = np.array([s[0] for s in shells], dtype=np.int32)
    tab = np.stack([wl.gaussian_table(float(a), rcut, dr, l=int(l)) for l, a in shells])
    return wl.Species(name=name, rcut=float(rcut), dr=float(dr), l=ls, table=np.ascontiguousarray(tab))


def mesh_points(lattice, ngrid):
    """Cartesian coordinates [N1*N2*N3][3] of the mesh points of one cell, C order."""
    n1, n2, n3 = (int(x) for x in ngrid)
    f = np.stack(np.meshgrid(np.arange(n1) / n1, np.arange(n2) / n2, np.arange(n3) / n3, indexing="ij"), axis=-1)
    return f.reshape(-1, 3) @ np.asarray(lattice)


def block_dict(H, blocks, norb_atom):
    """{(I,J,R1,R2,R3): ndarray[nI][nJ]} view of a flat block buffer."""
    bi, bj, bR, off = blocks
    out = {}
    for b in range(len(bi)):
        nI, nJ = int(norb_atom[bi[b]]), int(norb_atom[bj[b]])
        out[(int(bi[b]), int(bj[b]), int(bR[b, 0]), int(bR[b, 1]), int(bR[b, 2]))] = \
            H[off[b]:off[b] + nI * nJ].reshape(nI, nJ)
    return out


def norb_per_atom(w):
    return np.array([w.species[s].norb for s in w.atom_species], dtype=np.int64)
