"""Pins for oracle.snap_psibeta / oracle.enumerate_snap_pairs (Sec. 3.3.2, Eq. 47): closed forms for
Gaussian orbitals and projectors, invariants, an independent pair count.  CPU only.

Closed forms used (c = a + b, A = |A|):
  int_0^inf r^(2l+2) exp(-c r^2) dr                = Gamma(l + 3/2) / (2 c^(l+3/2))
  int_0^inf r^(l+2) exp(-c r^2) j_l(A r) dr        = sqrt(pi) A^l exp(-A^2 / 4c) / (2^(l+2) c^(l+3/2))
  exp(-i A.r) = sum_l (2l+1) (-i)^l j_l(A r) P_l(A^.r^)
  int exp(-a|r-P|^2 - b|r-Q|^2 - i A.r) d^3r       = (pi/c)^(3/2) exp(-ab|P-Q|^2/c) exp(-A^2/4c) exp(-i A.(aP+bQ)/c)
"""
import math

import numpy as np

import oracle
from paper_2603_21835_b200 import workloads as wl
from helpers import gaussian_species

BIG = np.eye(3) * 60.0   # a cell large enough that no image matters


def quad(nang=110, nrad=140):
    x, rw = wl.radial_quadrature(nrad)
    n, aw = wl.angular_quadrature(nang)
    return x, rw, n, aw


def test_quadrature_tables_are_what_the_paper_names():
    """140-point Gauss-Legendre, 110-point Lebedev-Laikov: sizes, weight sums, unit vectors, and the
    Lebedev rule's exactness for a degree-16 monomial (order 17)."""
    x, rw, n, aw = quad()
    assert x.shape == (140,) and n.shape == (110, 3)
    assert abs(rw.sum() - 1.0) < 1e-14 and abs(aw.sum() - 4 * math.pi) < 1e-12
    assert np.abs(np.linalg.norm(n, axis=1) - 1).max() < 1e-14
    assert abs(np.sum(aw * n[:, 2] ** 16) - 4 * math.pi / 17) < 1e-12          # int z^16 dOmega = 4 pi / 17
    assert abs(np.sum(rw * x ** 7) - 1.0 / 8) < 1e-14


def test_onsite_overlaps_without_field_are_radial_integrals():
    """A = 0, one atom: S[(l m), (l' m')] = delta delta int f_l b_l r^2 dr; wrong Y_lm normalisation, a missing r^2 or
    quadrature weight, or a transposed block shows here."""
    a, b = 0.8, 3.0
    pos = np.array([[1.3, -0.7, 2.1]])
    want = np.zeros((9, 9))
    k = 0
    for l in (0, 1, 2):
        for _ in range(2 * l + 1):
            want[k, k] = math.gamma(l + 1.5) / (2 * (a + b) ** (l + 1.5))
            k += 1
    # what is left is the error of the cubic table interpolation, O(dr^4): 2e-8 at dr = 0.01, 16 times less at 0.005
    for dr, tol in ((0.01, 1e-7), (0.005, 1e-8)):
        sp = gaussian_species([(0, a), (1, a), (2, a)], rcut=6.0, dr=dr)
        pj = gaussian_species([(0, b), (1, b), (2, b)], rcut=3.0, dr=dr, name="beta")
        S, pairs = oracle.snap_psibeta(BIG, [sp], [pj], [0], pos, (0, 0, 0), *quad())
        assert len(pairs[0]) == 1 and tuple(pairs[2][0]) == (0, 0, 0)
        S = S.reshape(9, 9)
        assert np.abs(S.imag).max() < 1e-14
        off_diag = S.real - np.diag(np.diag(S.real))
        assert np.abs(off_diag).max() < 1e-15
        assert np.abs(S.real - want).max() < tol * want.max(), (dr, np.abs(S.real - want).max() / want.max())


def test_onsite_plane_wave_terms_pin_the_phase_convention():
    """One atom away from the origin, A != 0: <s|e^{-iA.r}|s> = sqrt(pi)/(4 c^1.5) e^{-A^2/4c} e^{-iA.tau} and
    <s|e^{-iA.r}|p_m> = -i sqrt(3 pi) A_m / (8 c^2.5) e^{-A^2/4c} e^{-iA.tau}, m = (y, z, x): the sign of the exponent,
    the absolute-position reading and the m order are all fixed by this."""
    a, b = 0.7, 2.5
    sp = gaussian_species([(0, a)], rcut=6.5)
    pj = gaussian_species([(0, b), (1, b)], rcut=3.2, name="beta")
    tau = np.array([[0.9, 1.7, -2.3]])
    A = np.array([0.31, -0.22, 0.17])
    S, _ = oracle.snap_psibeta(BIG, [sp], [pj], [0], tau, A, *quad())
    c = a + b
    g = math.exp(-(A @ A) / (4 * c)) * np.exp(-1j * (A @ tau[0]))
    want = np.empty(4, dtype=complex)
    want[0] = math.sqrt(math.pi) / (4 * c ** 1.5) * g
    want[1:] = -1j * math.sqrt(3 * math.pi) * A[[1, 2, 0]] / (8 * c ** 2.5) * g
    assert np.abs(S - want).max() < 1e-7 * np.abs(want).max()      # table interpolation error, as above


def test_two_centre_gaussians_in_a_field():
    """Projector on atom 0, orbital on atom 1: the Gaussian product formula.  The 110-point rule resolves the orbital's
    angular variation around the projector's centre only approximately (that is the method's error, not the oracle's):
    1e-6 with the paper's grid, 1e-8 with a 590-point rule."""
    a, b = 0.45, 2.0
    sp = gaussian_species([(0, a)], rcut=9.0)
    pj = gaussian_species([(0, b)], rcut=3.5, name="beta")
    pos = np.array([[0.4, -0.3, 0.8], [1.9, 0.6, -0.5]])
    A = np.array([-0.15, 0.27, 0.2])
    c = a + b
    P, Q = pos[1], pos[0]
    want = (math.pi / c) ** 1.5 * math.exp(-a * b * float((P - Q) @ (P - Q)) / c) * math.exp(-(A @ A) / (4 * c)) \
        * np.exp(-1j * (A @ (a * P + b * Q)) / c) / (4 * math.pi)
    for nang, tol in ((110, 1e-6), (590, 1e-8)):       # the floor is the table interpolation error again
        S, pairs = oracle.snap_psibeta(BIG, [sp], [pj], [0, 0], pos, A, *quad(nang))
        iat, jat, R, off = pairs
        k = [i for i in range(len(iat)) if iat[i] == 0 and jat[i] == 1][0]
        assert abs(S[off[k]] - want) < tol * abs(want), (nang, abs(S[off[k]] - want) / abs(want))


def test_conjugation_translation_and_periodic_images():
    """phi and beta are real: S(-A) = conj S(A).  Moving every atom by t multiplies S by e^{-iA.t}.  A pair (I, J, R)
    of a small periodic cell equals the pair (I, J', 0) of a big cell with J' placed at tau_J + R."""
    w = wl.tiny(seed=3, natom=3)
    pj = [wl.make_species("beta", 2.0, [(0, 1.5), (1, 1.8)])]
    A = np.array([0.21, 0.13, -0.3])
    q = quad()
    S, pairs = oracle.snap_psibeta(w.lattice, w.species, pj, w.atom_species, w.atom_pos, A, *q)
    Sm, _ = oracle.snap_psibeta(w.lattice, w.species, pj, w.atom_species, w.atom_pos, -A, *q, pairs=pairs)
    assert np.abs(Sm - S.conj()).max() < 1e-15 * np.abs(S).max() + 1e-18
    t = np.array([0.37, -1.2, 0.55])
    St, pt = oracle.snap_psibeta(w.lattice, w.species, pj, w.atom_species, w.atom_pos + t, A, *q)
    assert all(np.array_equal(x, y) for x, y in zip(pairs, pt))
    assert np.abs(St - np.exp(-1j * (A @ t)) * S).max() < 1e-13 * np.abs(S).max()
    iat, jat, R, off = pairs
    far = [b for b in range(len(iat)) if np.any(R[b] != 0)]
    assert far, "the tiny cell must have image pairs"
    for b in far[:: max(1, len(far) // 6)]:
        I, J = int(iat[b]), int(jat[b])
        two = np.stack([w.atom_pos[I], w.atom_pos[J] + R[b] @ w.lattice])
        S2, p2 = oracle.snap_psibeta(BIG, w.species, pj, [0, 0], two, A, *q)
        k = [i for i in range(len(p2[0])) if p2[0][i] == 0 and p2[1][i] == 1][0]
        assert np.abs(S2[p2[3][k]:p2[3][k + 1]] - S[off[b]:off[b + 1]]).max() < 1e-14 * np.abs(S).max()


def test_pair_list_against_a_replicated_supercell():
    """(I, J, R) list: sorted, strict cutoff rb_I + rc_J, and complete -- counted independently with a k-d tree over a
    7 x 7 x 7 replication of a triclinic cell; species without projectors host no pair."""
    from scipy.spatial import cKDTree
    w = wl.tiny(seed=5, natom=4)
    sp2 = wl.make_species("B", 2.2, [(0, 0.9)])
    species = [w.species[0], sp2]
    asp = np.array([0, 1, 0, 1], dtype=np.int32)
    none = wl.Species(name="none", rcut=0.0, dr=0.01, l=np.zeros(0, np.int32), table=np.zeros((0, 8)))
    proj = [wl.make_species("beta", 1.8, [(0, 1.5)]), none]
    iat, jat, R, off = oracle.enumerate_snap_pairs(w.lattice, species, proj, asp, w.atom_pos)
    keys = list(zip(iat.tolist(), jat.tolist(), R[:, 0].tolist(), R[:, 1].tolist(), R[:, 2].tolist()))
    assert keys == sorted(keys) and len(set(keys)) == len(keys)
    assert set(iat.tolist()) <= {0, 2}
    rng = range(-3, 4)
    shifts = np.array([(i, j, k) for i in rng for j in rng for k in rng])
    images = (w.atom_pos[None, :, :] + (shifts @ w.lattice)[:, None, :]).reshape(-1, 3)
    tree = cKDTree(images)
    count = 0
    for I in (0, 2):
        for J in range(4):
            cut = 1.8 + float(species[asp[J]].rcut)
            near = tree.query_ball_point(w.atom_pos[I], cut)
            count += sum(1 for k in near if k % 4 == J and np.linalg.norm(images[k] - w.atom_pos[I]) < cut)
    assert count == len(keys)
    assert off[-1] == sum(int(species[asp[j]].norb) * 1 for j in jat)


def test_pair_cutoff_is_strict_for_a_self_image_exactly_at_the_cutoff():
    """|a1| = rb + rc exactly: the self images (0, 0, +-1, 0, 0) sit ON the cutoff and are not pairs (strict
    inequality, and the displacement is formed as (tau_J - tau_I) + R so that rounding cannot turn the tie)."""
    sp = wl.make_species("A", 3.0, [(0, 0.6)])
    pj = wl.make_species("beta", 2.0, [(0, 1.5)])
    lat = np.array([[5.0, 0.0, 0.0], [0.0, 9.0, 0.0], [0.0, 0.0, 9.0]])
    iat, jat, R, off = oracle.enumerate_snap_pairs(lat, [sp], [pj], [0], np.array([[0.123456789, 1.1, 2.2]]))
    assert [tuple(r) for r in R.tolist()] == [(0, 0, 0)]
    lat[0, 0] = 5.0 - 1e-9
    iat, jat, R, off = oracle.enumerate_snap_pairs(lat, [sp], [pj], [0], np.array([[0.123456789, 1.1, 2.2]]))
    assert [tuple(r) for r in R.tolist()] == [(-1, 0, 0), (0, 0, 0), (1, 0, 0)]
