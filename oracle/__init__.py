"""CPU oracle for gint_vlocal / gint_rho / gint_fvl / gint_fold_k / gint_snap_psibeta -- TEST INFRASTRUCTURE ONLY.

Thin ctypes binding of oracle/gint_oracle.c (which holds all the arithmetic and
cites the paper).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; it imports nothing
from the product package except nothing at all -- inputs arrive as numpy arrays.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence, Tuple

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_ip = ctypes.POINTER(ctypes.c_int)
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        c_i64p = ctypes.POINTER(ctypes.c_int64)
        lib.orc_phi.restype = ctypes.c_int
        lib.orc_phi.argtypes = [ctypes.c_int, c_dp, c_dp, c_ip, c_ip, c_ip, c_dp, ctypes.c_int, ctypes.c_int, c_dp, c_dp]
        lib.orc_enumerate_blocks.restype = ctypes.c_int64
        lib.orc_enumerate_blocks.argtypes = [c_dp, ctypes.c_int, c_dp, c_dp, ctypes.c_int64, c_i32p, c_i32p, c_i32p]
        lib.orc_vlocal.restype = ctypes.c_int
        lib.orc_vlocal.argtypes = [c_dp, c_ip, ctypes.c_int, c_dp, c_dp, c_ip, c_ip, c_ip, c_dp, ctypes.c_int, c_ip,
                                   c_dp, c_dp, ctypes.c_int64, c_i32p, c_i32p, c_i32p, c_i64p, c_dp, ctypes.c_int]
        lib.orc_rho.restype = ctypes.c_int
        lib.orc_rho.argtypes = [c_dp, c_ip, ctypes.c_int, c_dp, c_dp, c_ip, c_ip, c_ip, c_dp, ctypes.c_int, c_ip, c_dp,
                                ctypes.c_int64, c_i32p, c_i32p, c_i32p, c_i64p, c_dp, c_dp, ctypes.c_int]
        lib.orc_phi_grad.restype = ctypes.c_int
        lib.orc_phi_grad.argtypes = [ctypes.c_int, c_dp, c_dp, c_ip, c_ip, c_ip, c_dp, ctypes.c_int, ctypes.c_int, c_dp,
                                     c_dp, c_dp]
        lib.orc_fvl.restype = ctypes.c_int
        lib.orc_fvl.argtypes = [c_dp, c_ip, ctypes.c_int, c_dp, c_dp, c_ip, c_ip, c_ip, c_dp, ctypes.c_int, c_ip, c_dp,
                                c_dp, ctypes.c_int64, c_i32p, c_i32p, c_i32p, c_i64p, c_dp, c_dp, ctypes.c_int]
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


class _SpeciesPack:
    """Flatten a list of species (objects with rcut, dr, l, table) for the C side."""

    def __init__(self, species: Sequence):
        self.n = len(species)
        self.rcut = np.array([float(s.rcut) for s in species], dtype=np.float64)
        self.dr = np.array([float(s.dr) for s in species], dtype=np.float64)
        self.ntab = np.array([int(np.asarray(s.table).shape[1]) for s in species], dtype=np.intc)
        self.nrad = np.array([int(np.asarray(s.l).shape[0]) for s in species], dtype=np.intc)
        self.l = np.ascontiguousarray(np.concatenate([np.asarray(s.l, dtype=np.intc) for s in species]), dtype=np.intc)
        self.table = np.ascontiguousarray(np.concatenate([np.asarray(s.table, dtype=np.float64).ravel() for s in species]))
        self.norb = np.array([int(np.sum(2 * np.asarray(s.l) + 1)) for s in species], dtype=np.int64)

    def args(self):
        return (self.n, _p(self.rcut, ctypes.c_double), _p(self.dr, ctypes.c_double), _p(self.ntab, ctypes.c_int),
                _p(self.nrad, ctypes.c_int), _p(self.l, ctypes.c_int), _p(self.table, ctypes.c_double))


def phi(species: Sequence, which: int, d: np.ndarray) -> np.ndarray:
    """Orbital values phi_mu(d) of species `which` at displacements d[npts][3] (Eq. 1)."""
    lib = _load()
    sp = _SpeciesPack(species)
    d = np.ascontiguousarray(np.asarray(d, dtype=np.float64).reshape(-1, 3))
    out = np.empty((d.shape[0], int(sp.norb[which])), dtype=np.float64)
    rc = lib.orc_phi(*sp.args(), int(which), int(d.shape[0]), _p(d, ctypes.c_double), _p(out, ctypes.c_double))
    if rc < 0:
        raise RuntimeError("orc_phi failed: %d" % rc)
    return out


def enumerate_blocks(lattice, species, atom_species, atom_pos) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """All (I,J,R) with overlapping cutoff spheres, sorted by (I,J,R1,R2,R3).
    Returns (iat, jat, R[nblk][3], offset[nblk+1]) with offset the prefix sum of n_I*n_J."""
    lib = _load()
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    pos = np.ascontiguousarray(atom_pos, dtype=np.float64)
    asp = np.asarray(atom_species)
    rc_atom = np.ascontiguousarray([float(species[s].rcut) for s in asp], dtype=np.float64)
    natom = pos.shape[0]
    dummy = np.zeros(3, dtype=np.int32)
    n = lib.orc_enumerate_blocks(_p(lattice, ctypes.c_double), natom, _p(pos, ctypes.c_double),
                                 _p(rc_atom, ctypes.c_double), 0, _p(dummy, ctypes.c_int32),
                                 _p(dummy, ctypes.c_int32), _p(dummy, ctypes.c_int32))
    if n < 0:
        raise RuntimeError("orc_enumerate_blocks failed")
    bi = np.empty(max(n, 1), dtype=np.int32)
    bj = np.empty(max(n, 1), dtype=np.int32)
    bR = np.empty((max(n, 1), 3), dtype=np.int32)
    lib.orc_enumerate_blocks(_p(lattice, ctypes.c_double), natom, _p(pos, ctypes.c_double),
                             _p(rc_atom, ctypes.c_double), n, _p(bi, ctypes.c_int32), _p(bj, ctypes.c_int32),
                             _p(bR, ctypes.c_int32))
    bi, bj, bR = bi[:n], bj[:n], bR[:n]
    norb = np.array([int(np.sum(2 * np.asarray(species[s].l) + 1)) for s in asp], dtype=np.int64)
    off = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(norb[bi] * norb[bj], out=off[1:])
    return bi, bj, bR, off


def vlocal(lattice, ngrid, species, atom_species, atom_pos, V, blocks=None, nthreads: int = 0,
           return_threads: bool = False):
    """H blocks of Eq. 45 for `blocks` = (iat, jat, R) (default: all, sorted).
    Returns (H_flat, (iat, jat, R, offset)); H_flat holds the listed blocks back to back,
    each row-major n_I x n_J.  The listed blocks must be grouped by iat."""
    lib = _load()
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    ngrid_c = np.ascontiguousarray(ngrid, dtype=np.intc)
    pos = np.ascontiguousarray(atom_pos, dtype=np.float64)
    asp = np.ascontiguousarray(atom_species, dtype=np.intc)
    V = np.ascontiguousarray(V, dtype=np.float64)
    assert V.shape == tuple(int(x) for x in ngrid_c)
    sp = _SpeciesPack(species)
    if blocks is None:
        bi, bj, bR, off = enumerate_blocks(lattice, species, asp, pos)
    else:
        bi = np.ascontiguousarray(blocks[0], dtype=np.int32)
        bj = np.ascontiguousarray(blocks[1], dtype=np.int32)
        bR = np.ascontiguousarray(blocks[2], dtype=np.int32).reshape(-1, 3)
        norb = sp.norb[asp]
        off = np.zeros(bi.shape[0] + 1, dtype=np.int64)
        np.cumsum(norb[bi] * norb[bj], out=off[1:])
    out = np.zeros(int(off[-1]), dtype=np.float64)
    nb = int(bi.shape[0])
    if nb:
        rc = lib.orc_vlocal(_p(lattice, ctypes.c_double), _p(ngrid_c, ctypes.c_int), *sp.args(), int(pos.shape[0]),
                            _p(asp, ctypes.c_int), _p(pos, ctypes.c_double), _p(V, ctypes.c_double), nb,
                            _p(bi, ctypes.c_int32), _p(bj, ctypes.c_int32), _p(bR, ctypes.c_int32),
                            _p(off, ctypes.c_int64), _p(out, ctypes.c_double), int(nthreads))
        if rc < 0:
            raise RuntimeError("orc_vlocal failed: %d" % rc)
    else:
        rc = 0
    if return_threads:
        return out, (bi, bj, bR, off), rc
    return out, (bi, bj, bR, off)


def fold_k(H_flat, blocks, norb_atom, kfrac) -> np.ndarray:
    """H(k) = sum_R exp(i k.R) H(R)  -- PAPER.md:92-95 (Sec. 2.1, Eq. 5), the plain definition.

    k = kfrac[0] b1 + kfrac[1] b2 + kfrac[2] b3 with a_i . b_j = 2 pi delta_ij, R = n1 a1 + n2 a2 + n3 a3, so
    k.R = 2 pi (kfrac . n).  Returns the dense complex [norb_tot][norb_tot] matrix; rows are the orbitals of atom I
    (atoms in input order, orbitals in block order), columns those of atom J.  Pinned by
    tests/test_oracle_pins.py::test_bloch_sum_dense_gemm_cfg1 (Phi_k^dagger V dV Phi_k through a library GEMM).
    """
    bi, bj, bR, off = blocks
    norb_atom = np.asarray(norb_atom, dtype=np.int64)
    first = np.concatenate([[0], np.cumsum(norb_atom)])
    n = int(first[-1])
    Hk = np.zeros((n, n), dtype=np.complex128)
    kf = np.asarray(kfrac, dtype=np.float64)
    for b in range(len(bi)):
        I, J = int(bi[b]), int(bj[b])
        ph = np.exp(2j * np.pi * float(kf @ bR[b]))
        Hk[first[I]:first[I + 1], first[J]:first[J + 1]] += ph * np.asarray(H_flat[off[b]:off[b + 1]]).reshape(
            int(norb_atom[I]), int(norb_atom[J]))
    return Hk


def rho(lattice, ngrid, species, atom_species, atom_pos, D_flat, blocks, nthreads: int = 0) -> np.ndarray:
    """Charge density on the mesh from density-matrix blocks (Eq. 44).
    `blocks` = (iat, jat, R, offset) as returned by vlocal/enumerate_blocks; D_flat has the H layout."""
    lib = _load()
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    ngrid_c = np.ascontiguousarray(ngrid, dtype=np.intc)
    pos = np.ascontiguousarray(atom_pos, dtype=np.float64)
    asp = np.ascontiguousarray(atom_species, dtype=np.intc)
    sp = _SpeciesPack(species)
    bi = np.ascontiguousarray(blocks[0], dtype=np.int32)
    bj = np.ascontiguousarray(blocks[1], dtype=np.int32)
    bR = np.ascontiguousarray(blocks[2], dtype=np.int32).reshape(-1, 3)
    off = np.ascontiguousarray(blocks[3], dtype=np.int64)
    D = np.ascontiguousarray(D_flat, dtype=np.float64)
    assert D.shape[0] == int(off[-1])
    out = np.zeros(tuple(int(x) for x in ngrid_c), dtype=np.float64)
    rc = lib.orc_rho(_p(lattice, ctypes.c_double), _p(ngrid_c, ctypes.c_int), *sp.args(), int(pos.shape[0]),
                     _p(asp, ctypes.c_int), _p(pos, ctypes.c_double), int(bi.shape[0]), _p(bi, ctypes.c_int32),
                     _p(bj, ctypes.c_int32), _p(bR, ctypes.c_int32), _p(off, ctypes.c_int64), _p(D, ctypes.c_double),
                     _p(out, ctypes.c_double), int(nthreads))
    if rc < 0:
        raise RuntimeError("orc_rho failed: %d" % rc)
    return out


def phi_grad(species: Sequence, which: int, d: np.ndarray):
    """(phi[npts][norb], grad[npts][norb][3]) of species `which` at displacements d: Eq. 1 and its gradient with the
    radial derivative taken from the same cubic Lagrange interpolant (readings #19, #20)."""
    lib = _load()
    sp = _SpeciesPack(species)
    d = np.ascontiguousarray(np.asarray(d, dtype=np.float64).reshape(-1, 3))
    n = int(sp.norb[which])
    ph = np.empty((d.shape[0], n), dtype=np.float64)
    gr = np.empty((d.shape[0], n, 3), dtype=np.float64)
    rc = lib.orc_phi_grad(*sp.args(), int(which), int(d.shape[0]), _p(d, ctypes.c_double), _p(ph, ctypes.c_double),
                          _p(gr, ctypes.c_double))
    if rc < 0:
        raise RuntimeError("orc_phi_grad failed: %d" % rc)
    return ph, gr


def fvl(lattice, ngrid, species, atom_species, atom_pos, V, D_flat, blocks, nthreads: int = 0) -> np.ndarray:
    """Local Pulay force F[natom][3] (Eq. 46; reading #18):
    F_K = - sum_blocks D(I,J,R) : dH(I,J,R)/dtau_K at fixed V.  `blocks` = (iat, jat, R, offset), D_flat in the H layout."""
    lib = _load()
    lattice = np.ascontiguousarray(lattice, dtype=np.float64)
    ngrid_c = np.ascontiguousarray(ngrid, dtype=np.intc)
    pos = np.ascontiguousarray(atom_pos, dtype=np.float64)
    asp = np.ascontiguousarray(atom_species, dtype=np.intc)
    V = np.ascontiguousarray(V, dtype=np.float64)
    sp = _SpeciesPack(species)
    bi = np.ascontiguousarray(blocks[0], dtype=np.int32)
    bj = np.ascontiguousarray(blocks[1], dtype=np.int32)
    bR = np.ascontiguousarray(blocks[2], dtype=np.int32).reshape(-1, 3)
    off = np.ascontiguousarray(blocks[3], dtype=np.int64)
    D = np.ascontiguousarray(D_flat, dtype=np.float64)
    assert D.shape[0] == int(off[-1]) and V.shape == tuple(int(x) for x in ngrid_c)
    F = np.zeros((pos.shape[0], 3), dtype=np.float64)
    rc = lib.orc_fvl(_p(lattice, ctypes.c_double), _p(ngrid_c, ctypes.c_int), *sp.args(), int(pos.shape[0]),
                     _p(asp, ctypes.c_int), _p(pos, ctypes.c_double), _p(V, ctypes.c_double), int(bi.shape[0]),
                     _p(bi, ctypes.c_int32), _p(bj, ctypes.c_int32), _p(bR, ctypes.c_int32), _p(off, ctypes.c_int64),
                     _p(D, ctypes.c_double), _p(F, ctypes.c_double), int(nthreads))
    if rc < 0:
        raise RuntimeError("orc_fvl failed: %d" % rc)
    return F


# ---- spherical-grid integration of the velocity-gauge nonlocal overlaps (Sec. 3.3.2, Eq. 47) ------
def enumerate_snap_pairs(lattice, species, proj, atom_species, atom_pos):
    """Every (I, J, R): projectors of atom I (cutoff rb_I) against orbitals of the image of atom J at tau_J + R
    (cutoff rc_J) with |tau_J + R - tau_I| < rb_I + rc_J (strict), sorted by (I, J, R1, R2, R3); species without
    projectors (no radial function) host none.  Brute force over a box of images.  Returns (iat, jat, R[n][3],
    offset[n+1]); block b holds n_J x m_I complex numbers, n_J orbitals of J (rows), m_I projector components of I."""
    lat = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    pos = np.asarray(atom_pos, dtype=np.float64).reshape(-1, 3)
    asp = np.asarray(atom_species).reshape(-1)
    rmax = max(float(p.rcut) for p in proj) + max(float(s.rcut) for s in species)
    inv = np.linalg.inv(lat)
    heights = 1.0 / np.linalg.norm(inv, axis=0)          # distance between lattice planes along each axis
    frac = pos @ inv
    span = frac.max(axis=0) - frac.min(axis=0)
    nmax = [int(np.ceil(rmax / heights[k] + span[k])) + 1 for k in range(3)]
    out = []
    for I in range(pos.shape[0]):
        if np.asarray(proj[asp[I]].l).shape[0] == 0:
            continue
        for J in range(pos.shape[0]):
            cut = float(proj[asp[I]].rcut) + float(species[asp[J]].rcut)
            for r1 in range(-nmax[0], nmax[0] + 1):
                for r2 in range(-nmax[1], nmax[1] + 1):
                    for r3 in range(-nmax[2], nmax[2] + 1):
                        # (tau_J - tau_I) first: a self image sits at exactly |R|, so a tie with the cutoff stays a tie
                        d = (pos[J] - pos[I]) + (r1 * lat[0] + r2 * lat[1] + r3 * lat[2])
                        if float(d @ d) < cut * cut:
                            out.append((I, J, r1, r2, r3))
    out.sort()
    arr = np.array(out, dtype=np.int64).reshape(-1, 5)
    norb = np.array([int(np.sum(2 * np.asarray(s.l) + 1)) for s in species], dtype=np.int64)
    mproj = np.array([int(np.sum(2 * np.asarray(p.l) + 1)) for p in proj], dtype=np.int64)
    sizes = norb[asp[arr[:, 1]]] * mproj[asp[arr[:, 0]]] if len(out) else np.zeros(0, dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    return (arr[:, 0].astype(np.int32), arr[:, 1].astype(np.int32), np.ascontiguousarray(arr[:, 2:5].astype(np.int32)), off)


def snap_psibeta(lattice, species, proj, atom_species, atom_pos, A, rad_x, rad_w, ang_n, ang_w, pairs=None):
    """S(I, J, R)[mu][b] = < phi_mu(r - tau_J - R) | exp(-i A.r) | beta_b(r - tau_I) >     (Eq. 47)

    by quadrature on a grid centred on the projector's atom, as the paper states it: radial nodes
    r_i = rad_x[i] * rb_I with weights rad_w[i] * rb_I (Gauss-Legendre on [0, rb_I]), angular nodes ang_n[a] with
    weights ang_w[a] (Lebedev-Laikov, sum 4 pi):

        S = sum_i sum_a  rad_w_i rb r_i^2  ang_w_a  phi_mu(tau_I + r_i n_a - tau_J - R)
                         exp(-i A . (tau_I + r_i n_a))  beta_b(r_i n_a)

    phi real (so the bra needs no conjugate), r the absolute Cartesian position with the atoms where the caller put
    them, beta_{l m zeta}(r) = b_{l zeta}(|r|) Y_lm(r/|r|) with the same table interpolation and real Y_lm as the
    orbitals (orc_phi evaluates both).  Straight nested sums, one pair at a time; complex128.
    Returns (S_flat complex128[offset[-1]], pairs)."""
    lat = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    pos = np.asarray(atom_pos, dtype=np.float64).reshape(-1, 3)
    asp = np.asarray(atom_species).reshape(-1)
    A = np.asarray(A, dtype=np.float64).reshape(3)
    rad_x = np.asarray(rad_x, dtype=np.float64)
    rad_w = np.asarray(rad_w, dtype=np.float64)
    ang_n = np.asarray(ang_n, dtype=np.float64).reshape(-1, 3)
    ang_w = np.asarray(ang_w, dtype=np.float64)
    if pairs is None:
        pairs = enumerate_snap_pairs(lat, species, proj, asp, pos)
    iat, jat, R, off = pairs
    S = np.zeros(int(off[-1]), dtype=np.complex128)
    for b in range(len(iat)):
        I, J = int(iat[b]), int(jat[b])
        rb = float(proj[asp[I]].rcut)
        r = rad_x * rb                                                   # [nr]
        pts = (r[:, None, None] * ang_n[None, :, :]).reshape(-1, 3)      # [nr * na][3], relative to tau_I
        wq = ((rad_w * rb * r * r)[:, None] * ang_w[None, :]).reshape(-1)
        beta = phi(proj, int(asp[I]), pts)                               # [npts][m_I]
        centre = pos[J] + R[b, 0] * lat[0] + R[b, 1] * lat[1] + R[b, 2] * lat[2]
        ph = phi(species, int(asp[J]), pts + (pos[I] - centre))          # [npts][n_J]
        phase = np.exp(-1j * ((pts + pos[I]) @ A))
        blk = ph.T @ ((wq * phase)[:, None] * beta)                      # [n_J][m_I]
        S[off[b]:off[b + 1]] = blk.reshape(-1)
    return S, pairs
