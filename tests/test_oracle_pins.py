"""Pins for the CPU oracle (oracle/gint_oracle.c): everything here checks the
oracle against something OTHER than itself -- brute force through a different
code path, closed forms, invariants, library routines.  CPU only.

Citations: Eq. 45 = PAPER.md:393-398, Eq. 1 = PAPER.md:66-70, Eq. 5 = PAPER.md:92-95,
R convention = PAPER.md:104-106.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2603_21835_b200 import workloads as wl
from helpers import block_dict, gaussian_species, mesh_points, norb_per_atom


def run_oracle(w, V=None, blocks=None):
    return oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V if V is None else V,
                         blocks=blocks)


# ---------------------------------------------------------------------------
# 1. brute force on a tiny triclinic workload, through dense numpy algebra
# ---------------------------------------------------------------------------
def brute_force_block(w, I, J, R, window=3):
    """H block from Eq. 45 by a dense sum over an enlarged unwrapped window of mesh
    points (no sphere point lists, no block table, numpy matmul)."""
    n1, n2, n3 = (int(x) for x in w.ngrid)
    idx = np.stack(np.meshgrid(np.arange(-window * n1, (window + 1) * n1),
                               np.arange(-window * n2, (window + 1) * n2),
                               np.arange(-window * n3, (window + 1) * n3), indexing="ij"), axis=-1).reshape(-1, 3)
    r = (idx / np.array([n1, n2, n3])) @ w.lattice
    sI, sJ = int(w.atom_species[I]), int(w.atom_species[J])
    dI = r - w.atom_pos[I]
    keep = np.einsum("ij,ij->i", dI, dI) < (w.species[sI].rcut + 1e-9) ** 2
    idx, r, dI = idx[keep], r[keep], dI[keep]
    phiI = oracle.phi(w.species, sI, dI)
    phiJ = oracle.phi(w.species, sJ, r - w.atom_pos[J] - np.asarray(R) @ w.lattice)
    v = w.V[idx[:, 0] % n1, idx[:, 1] % n2, idx[:, 2] % n3]
    dV = abs(np.linalg.det(w.lattice)) / (n1 * n2 * n3)
    return (phiI * v[:, None]).T @ phiJ * dV


@pytest.mark.parametrize("seed", [7, 11])
def test_brute_force_tiny_triclinic(seed):
    w = wl.tiny(seed=seed)
    H, blocks = run_oracle(w)
    d = block_dict(H, blocks, norb_per_atom(w))
    assert len(d) > 20          # rc=3 in a ~5 bohr cell: many image blocks, incl. self-image (I,I,R!=0)
    assert any(k[0] == k[1] and k[2:] != (0, 0, 0) for k in d)
    scale = np.abs(H).max()
    rng = np.random.default_rng(seed)
    keys = list(d.keys())
    for k in [keys[i] for i in rng.choice(len(keys), size=12, replace=False)] + [keys[0], keys[-1]]:
        ref = brute_force_block(w, k[0], k[1], k[2:])
        assert np.abs(d[k] - ref).max() <= 1e-13 * scale, k


def test_brute_force_single_orbital_analytic_phi():
    """One atom, one s orbital, phi written out analytically in the test (no oracle code
    at all): H_00(0) by a triple loop over images.  Agreement limited by the table
    interpolation error (~1e-9 relative), so this pins the whole pipeline to 1e-7."""
    alpha, rc = 0.9, 5.0
    sp = gaussian_species([(0, alpha)], rc)
    L, n = 11.0, 22
    lattice = np.diag([L, L, L])
    pos = np.array([[2.3, 4.1, 7.7]])
    rng = np.random.default_rng(0)
    V = rng.normal(size=(n, n, n))
    H, blocks = oracle.vlocal(lattice, [n, n, n], [sp], [0], pos, V)
    d = block_dict(H, blocks, [1])
    y00 = 0.5 / math.sqrt(math.pi)
    acc = 0.0
    g = np.arange(-n, 2 * n)
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    rr = np.sqrt((X * L / n - pos[0, 0]) ** 2 + (Y * L / n - pos[0, 1]) ** 2 + (Z * L / n - pos[0, 2]) ** 2)
    ph = np.where(rr < rc, np.exp(-alpha * rr * rr) * y00, 0.0)
    acc = np.sum(ph * ph * V[X % n, Y % n, Z % n]) * (L / n) ** 3
    assert abs(d[(0, 0, 0, 0, 0)][0, 0] - acc) <= 1e-7 * abs(acc)


# ---------------------------------------------------------------------------
# 2. H_mu,nu(R)[I,J] = H_nu,mu(-R)[J,I]
# ---------------------------------------------------------------------------
def test_transpose_symmetry_cfg1(cfg1, cfg1_oracle):
    H, blocks = cfg1_oracle
    d = block_dict(H, blocks, norb_per_atom(cfg1))
    assert len(d) == 376 and H.size == 6016
    scale = np.abs(H).max()
    for (I, J, a, b, c), blk in d.items():
        other = d[(J, I, -a, -b, -c)]
        assert np.abs(blk - other.T).max() <= 1e-14 * scale


def test_blocks_sorted_and_complete(cfg1, cfg1_oracle):
    bi, bj, bR, off = cfg1_oracle[1]
    keys = [(int(bi[b]), int(bj[b]), int(bR[b, 0]), int(bR[b, 1]), int(bR[b, 2])) for b in range(len(bi))]
    assert keys == sorted(keys) and len(set(keys)) == len(keys)
    # independent enumeration of the strict sphere-overlap criterion
    w = cfg1
    want = set()
    for I in range(w.natom):
        for J in range(w.natom):
            for a in range(-3, 4):
                for b in range(-3, 4):
                    for c in range(-3, 4):
                        dvec = w.atom_pos[J] + np.array([a, b, c]) @ w.lattice - w.atom_pos[I]
                        if np.linalg.norm(dvec) < 12.0:
                            want.add((I, J, a, b, c))
    assert want == set(keys)


_SHEARED = np.array([[4.2, 0.0, 0.0], [3.1, 2.9, 0.0], [-1.3, 1.9, 3.4]])     # strongly sheared: a2 nearly along a1


@pytest.mark.parametrize("lattice", [None, _SHEARED])
def test_blocks_complete_on_triclinic_cells(lattice):
    """Block enumeration on non-orthogonal cells, pinned by something that shares nothing with its text (no inverse
    lattice, no search box derived from it): a plain loop over +-7 images per axis with the strict sphere-overlap
    criterion of reading #9, positions drawn outside the home cell as well."""
    w = wl.tiny(seed=13, natom=4, lattice=lattice)
    w.atom_pos[1] += np.array([2, -1, 1]) @ w.lattice          # atoms are never wrapped (reading #11)
    bi, bj, bR, off = oracle.enumerate_blocks(w.lattice, w.species, w.atom_species, w.atom_pos)
    keys = [(int(bi[b]), int(bj[b]), int(bR[b, 0]), int(bR[b, 1]), int(bR[b, 2])) for b in range(len(bi))]
    assert keys == sorted(keys) and len(set(keys)) == len(keys)
    reach = 2 * w.species[0].rcut
    m = 7
    assert np.abs(bR).max() < m - 1                              # the brute-force window is not the limit
    shifts = np.array([[a, b, c] for a in range(-m, m + 1) for b in range(-m, m + 1) for c in range(-m, m + 1)])
    want = set()
    for I in range(w.natom):
        for J in range(w.natom):
            d = np.linalg.norm(w.atom_pos[J] + shifts @ w.lattice - w.atom_pos[I], axis=1)
            for s in shifts[d < reach]:
                want.add((I, J, int(s[0]), int(s[1]), int(s[2])))
    assert want == set(keys)
    assert np.array_equal(np.diff(off), np.full(len(bi), w.species[0].norb ** 2))


@pytest.mark.parametrize("lattice", [None, _SHEARED])
@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.37, -0.21, 0.45)])
def test_bloch_sum_dense_gemm_triclinic(lattice, kfrac):
    """Same library-GEMM pin as test_bloch_sum_dense_gemm_cfg1, on triclinic cells whose reach (2 rc = 6 bohr)
    exceeds every cell edge: a block missing from the enumeration, or one counted twice, changes
    sum_R exp(ik.R) H(R) away from Phi_k^dagger V dV Phi_k (Eq. 5)."""
    w = wl.tiny(seed=17, natom=3, lattice=lattice)
    H, blocks = run_oracle(w)
    bi, bj, bR, off = blocks
    norb = norb_per_atom(w)
    first = np.concatenate([[0], np.cumsum(norb)])
    nb = int(first[-1])
    recip = 2 * np.pi * np.linalg.inv(w.lattice).T
    k = np.array(kfrac) @ recip
    pts = mesh_points(w.lattice, w.ngrid)
    Phi = np.zeros((pts.shape[0], nb), dtype=complex)
    m = 4          # rc = 3 bohr never reaches further than 4 cells on these lattices
    for a in range(-m, m + 1):
        for b_ in range(-m, m + 1):
            for c in range(-m, m + 1):
                Rv = np.array([a, b_, c]) @ w.lattice
                for I in range(w.natom):
                    ph = oracle.phi(w.species, int(w.atom_species[I]), pts - w.atom_pos[I] - Rv)
                    if np.any(ph):
                        assert max(abs(a), abs(b_), abs(c)) < m
                        Phi[:, first[I]:first[I + 1]] += np.exp(1j * (k @ Rv)) * ph
    dV = abs(np.linalg.det(w.lattice)) / pts.shape[0]
    ref = Phi.conj().T @ (Phi * (w.V.reshape(-1, 1) * dV))
    Hk = oracle.fold_k(H, blocks, norb, kfrac)
    assert np.abs(Hk - ref).max() <= 1e-13 * np.abs(ref).max()


# ---------------------------------------------------------------------------
# 3. V = c gives c * S_grid; linearity in V
# ---------------------------------------------------------------------------
def test_constant_and_linear_in_V(cfg1):
    w = cfg1
    S, _ = run_oracle(w, V=np.ones_like(w.V))
    Hc, _ = run_oracle(w, V=np.full_like(w.V, -0.37))
    assert np.abs(Hc - (-0.37) * S).max() <= 1e-14 * np.abs(S).max()
    rng = np.random.default_rng(5)
    V2 = rng.normal(size=w.V.shape)
    H1, _ = run_oracle(w)
    H2, _ = run_oracle(w, V=V2)
    H12, _ = run_oracle(w, V=w.V + V2)
    assert np.abs(H12 - H1 - H2).max() <= 1e-13 * np.abs(H12).max()


# ---------------------------------------------------------------------------
# 4./5./6. Gaussian closed forms (absolute scale, dV, Y_lm constants and m-order,
#          V index <-> coordinate mapping)
# ---------------------------------------------------------------------------
def two_gaussian_atoms(h, shellsA, shellsB, rc=7.0, L=16.0, A=(5.1, 6.3, 7.2), B=(5.9, 7.0, 6.1), dr=0.01):
    n = int(round(L / h))
    lattice = np.diag([L, L, L])
    spA = gaussian_species(shellsA, rc, dr)
    spB = gaussian_species(shellsB, rc, dr)
    pos = np.array([A, B], dtype=np.float64)
    return lattice, np.array([n, n, n]), [spA, spB], np.array([0, 1]), pos


def s0(alpha, beta, A, B):
    p = alpha + beta
    d2 = float(np.sum((np.asarray(A) - np.asarray(B)) ** 2))
    return (math.pi / p) ** 1.5 * math.exp(-alpha * beta * d2 / p)


def test_gaussian_s_overlap_converges_to_analytic():
    alpha, beta = 0.7, 0.8
    errs = {}
    for h in (1.0, 0.5, 0.4):
        lattice, ng, sp, asp, pos = two_gaussian_atoms(h, [(0, alpha)], [(0, beta)])
        H, blocks = oracle.vlocal(lattice, ng, sp, asp, pos, np.ones(tuple(ng)))
        d = block_dict(H, blocks, [1, 1])
        exact = s0(alpha, beta, pos[0], pos[1]) / (4 * math.pi)
        errs[h] = abs(d[(0, 1, 0, 0, 0)][0, 0] - exact) / exact
        # unit-normalised Gaussians: S = (2 sqrt(ab)/(a+b))^{3/2} exp(-ab d^2/(a+b))
        nA, nB = (2 * alpha / math.pi) ** 0.75, (2 * beta / math.pi) ** 0.75
        Snorm = d[(0, 1, 0, 0, 0)][0, 0] * 4 * math.pi * nA * nB
        closed = (2 * math.sqrt(alpha * beta) / (alpha + beta)) ** 1.5 * math.exp(
            -alpha * beta * np.sum((pos[0] - pos[1]) ** 2) / (alpha + beta))
        assert abs(Snorm - closed) / closed == pytest.approx(errs[h], abs=1e-12)
    assert 1e-6 < errs[1.0] < 1e-2          # quadrature error ~ exp(-pi^2/(h^2 (a+b))) = 1.4e-3
    assert errs[0.5] < 5e-8 and errs[0.4] < 5e-8   # interpolation floor ~1e-9


def test_interpolation_error_scales_as_dr4():
    """Halving dr must reduce the error floor ~16x (cubic Lagrange, reading #4)."""
    alpha, beta = 1.1, 1.3
    out = {}
    for dr in (0.04, 0.02):
        lattice, ng, sp, asp, pos = two_gaussian_atoms(0.4, [(0, alpha)], [(0, beta)], rc=6.0, dr=dr)
        H, blocks = oracle.vlocal(lattice, ng, sp, asp, pos, np.ones(tuple(ng)))
        d = block_dict(H, blocks, [1, 1])
        exact = s0(alpha, beta, pos[0], pos[1]) / (4 * math.pi)
        out[dr] = abs(d[(0, 1, 0, 0, 0)][0, 0] - exact) / exact
    ratio = out[0.04] / out[0.02]
    assert 8.0 < ratio < 32.0, (out, ratio)


def test_plane_wave_potential_axis_mapping():
    """V = cos(G.r), G = 2pi/L (1,2,3): H_ss = Y00^2 S0 exp(-G^2/4p) cos(G.P)."""
    alpha, beta, L = 0.7, 0.8, 16.0
    lattice, ng, sp, asp, pos = two_gaussian_atoms(0.4, [(0, alpha)], [(0, beta)], L=L)
    G = 2 * math.pi / L * np.array([1.0, 2.0, 3.0])
    pts = mesh_points(lattice, ng)
    V = np.cos(pts @ G).reshape(tuple(ng))
    H, blocks = oracle.vlocal(lattice, ng, sp, asp, pos, V)
    d = block_dict(H, blocks, [1, 1])
    p = alpha + beta
    P = (alpha * pos[0] + beta * pos[1]) / p
    exact = s0(alpha, beta, pos[0], pos[1]) / (4 * math.pi) * math.exp(-G @ G / (4 * p)) * math.cos(G @ P)
    assert abs(d[(0, 1, 0, 0, 0)][0, 0] - exact) <= 5e-8 * abs(s0(alpha, beta, pos[0], pos[1]) / (4 * math.pi))
    # a transposed V (wrong axis order) must NOT pass
    Hbad, _ = oracle.vlocal(lattice, ng, sp, asp, pos, np.ascontiguousarray(V.transpose(2, 1, 0)))
    assert abs(Hbad[blocks[3][1]] - exact) > 1e-3 * abs(exact)


def test_s_p_d_gaussian_overlaps_pin_ylm():
    """<s_A | r^l exp(-b r^2) Y_lm at B> closed forms: pins every Y_lm constant, the
    m-order (l=1: y,z,x; l=2: xy,yz,3z^2-1,xz,x^2-y^2) and the sign convention."""
    alpha, beta = 0.7, 0.8
    lattice, ng, sp, asp, pos = two_gaussian_atoms(0.4, [(0, alpha)], [(0, beta), (1, beta), (2, beta)])
    H, blocks = oracle.vlocal(lattice, ng, sp, asp, pos, np.ones(tuple(ng)))
    d = block_dict(H, blocks, [1, 9])
    blk = d[(0, 1, 0, 0, 0)][0]
    p = alpha + beta
    S0 = s0(alpha, beta, pos[0], pos[1])
    q = (alpha * pos[0] + beta * pos[1]) / p - pos[1]     # P - B
    x, y, z = q
    y00 = 0.5 / math.sqrt(math.pi)
    c1 = math.sqrt(3 / (4 * math.pi))
    c2a, c2b, c2c = 0.5 * math.sqrt(15 / math.pi), 0.25 * math.sqrt(5 / math.pi), 0.25 * math.sqrt(15 / math.pi)
    want = y00 * S0 * np.array([
        y00,
        c1 * y, c1 * z, c1 * x,
        c2a * x * y, c2a * y * z, c2b * (3 * z * z - (x * x + y * y + z * z)), c2a * x * z, c2c * (x * x - y * y)])
    assert np.abs(blk - want).max() <= 5e-8 * abs(want[0])
    assert np.abs(want[1:]).min() > 1e-4 * abs(want[0])   # every component is actually exercised


# ---------------------------------------------------------------------------
# 7. unit impulse: V = delta at one mesh point
# ---------------------------------------------------------------------------
def test_unit_impulse(cfg1):
    w = cfg1
    g = (5, 17, 30)
    V = np.zeros_like(w.V)
    V[g] = 1.0
    H, blocks = run_oracle(w, V=V)
    d = block_dict(H, blocks, norb_per_atom(w))
    n = w.ngrid
    rg = (np.array(g) / n) @ w.lattice
    dV = abs(np.linalg.det(w.lattice)) / np.prod(n)
    shifts = np.array([[a, b, c] for a in range(-3, 4) for b in range(-3, 4) for c in range(-3, 4)])
    rng = np.random.default_rng(1)
    keys = list(d.keys())
    for k in [keys[i] for i in rng.choice(len(keys), 25, replace=False)]:
        I, J, R = k[0], k[1], np.array(k[2:])
        pI = oracle.phi(w.species, 0, rg - w.atom_pos[I] - shifts @ w.lattice)          # over images R'
        pJ = oracle.phi(w.species, 0, rg - w.atom_pos[J] - (shifts + R) @ w.lattice)
        ref = dV * np.einsum("rm,rn->mn", pI, pJ)
        assert np.abs(d[k] - ref).max() <= 1e-14 * max(np.abs(ref).max(), 1e-3)


# ---------------------------------------------------------------------------
# 8. translate all atoms by one mesh vector and roll V
# ---------------------------------------------------------------------------
def test_shift_atoms_roll_V(cfg1, cfg1_oracle):
    w = cfg1
    H0, blocks0 = cfg1_oracle
    step = np.array([1, 2, -3])
    shift = (step / w.ngrid) @ w.lattice
    V2 = np.roll(w.V, shift=tuple(int(s) for s in step), axis=(0, 1, 2))
    H1, blocks1 = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos + shift, V2)
    assert np.array_equal(blocks0[2], blocks1[2]) and np.array_equal(blocks0[0], blocks1[0])
    assert np.abs(H1 - H0).max() <= 1e-12 * np.abs(H0).max()


# ---------------------------------------------------------------------------
# 9. Bloch-sum dense cross-check through a library GEMM (Eq. 5)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.31, -0.17, 0.43), (0.5, 0.25, -0.4)])
def test_bloch_sum_dense_gemm_cfg1(cfg1, cfg1_oracle, kfrac):
    w = cfg1
    H, blocks = cfg1_oracle
    bi, bj, bR, off = blocks
    norb = norb_per_atom(w)
    first = np.concatenate([[0], np.cumsum(norb)])
    nb = int(first[-1])
    recip = 2 * np.pi * np.linalg.inv(w.lattice).T       # rows b_i, a_i . b_j = 2 pi delta_ij
    k = np.array(kfrac) @ recip
    Hk = np.zeros((nb, nb), dtype=complex)
    for b in range(len(bi)):
        I, J = int(bi[b]), int(bj[b])
        ph = np.exp(1j * (k @ (bR[b] @ w.lattice)))
        Hk[first[I]:first[I + 1], first[J]:first[J + 1]] += ph * H[off[b]:off[b + 1]].reshape(norb[I], norb[J])
    pts = mesh_points(w.lattice, w.ngrid)
    Phi = np.zeros((pts.shape[0], nb), dtype=complex)
    for a in range(-2, 3):
        for b_ in range(-2, 3):
            for c in range(-2, 3):
                Rv = np.array([a, b_, c]) @ w.lattice
                ph = np.exp(1j * (k @ Rv))
                for I in range(w.natom):
                    Phi[:, first[I]:first[I + 1]] += ph * oracle.phi(w.species, int(w.atom_species[I]),
                                                                     pts - w.atom_pos[I] - Rv)
    dV = abs(np.linalg.det(w.lattice)) / pts.shape[0]
    ref = Phi.conj().T @ (Phi * (w.V.reshape(-1, 1) * dV))
    assert np.abs(Hk - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(Hk - Hk.conj().T).max() <= 1e-13 * np.abs(ref).max()
    # the oracle's own k-folding (Eq. 5) is pinned by the same library GEMM
    Hk2 = oracle.fold_k(H, blocks, norb, kfrac)
    assert np.abs(Hk2 - ref).max() <= 1e-13 * np.abs(ref).max()


def test_gram_matrix_is_psd_and_negative_V_gives_nsd(cfg1):
    w = cfg1
    norb = norb_per_atom(w)
    first = np.concatenate([[0], np.cumsum(norb)])

    def gamma(H, blocks):
        bi, bj, bR, off = blocks
        M = np.zeros((first[-1], first[-1]))
        for b in range(len(bi)):
            I, J = int(bi[b]), int(bj[b])
            M[first[I]:first[I + 1], first[J]:first[J + 1]] += H[off[b]:off[b + 1]].reshape(norb[I], norb[J])
        return M
    S = gamma(*run_oracle(w, V=np.ones_like(w.V)))
    assert np.linalg.eigvalsh(S).min() > -1e-12
    Hn = gamma(*run_oracle(w, V=-np.abs(w.V) - 0.1))
    assert np.linalg.eigvalsh(Hn).max() < 1e-12
    # generated tables are normalised: on-site overlap ~ 1, different (l,m) ~ 0 (mesh-quadrature accuracy)
    on = S[:4, :4] - 0.0
    d = block_dict(*run_oracle(w, V=np.ones_like(w.V)), norb)
    blk = d[(0, 0, 0, 0, 0)]
    assert np.abs(blk - np.eye(4)).max() < 1e-4


# ---------------------------------------------------------------------------
# 10.-12. radial interpolation and Y_lm sum rules through orc_phi
# ---------------------------------------------------------------------------
def test_cubic_polynomial_reproduced_exactly():
    dr, rc = 0.05, 4.0
    ntab = int(round(rc / dr)) + 4
    r = np.arange(ntab) * dr
    poly = lambda x: 0.3 - 1.7 * x + 0.9 * x * x - 0.21 * x ** 3
    sp = wl.Species("cubic", rc, dr, np.array([0], dtype=np.int32), poly(r)[None, :].copy())
    rng = np.random.default_rng(3)
    rr = rng.uniform(0.0, rc * (1 - 1e-9), size=2000)
    dirs = rng.normal(size=(2000, 3))
    dirs /= np.linalg.norm(dirs, axis=1)[:, None]
    val = oracle.phi([sp], 0, dirs * rr[:, None])[:, 0] / (0.5 / math.sqrt(math.pi))
    rr_eff = np.linalg.norm(dirs * rr[:, None], axis=1)
    assert np.abs(val - poly(rr_eff)).max() < 5e-14
    # a quartic is NOT reproduced: the 4-point error term h^4 f''''/24 * t(t-1)(t-2)(t-3) shows up
    sp4 = wl.Species("quartic", rc, dr, np.array([0], dtype=np.int32), (r ** 4)[None, :].copy())
    v4 = oracle.phi([sp4], 0, np.array([[0.0, 0.0, 1.0 + 0.5 * dr]]))[0, 0] / (0.5 / math.sqrt(math.pi))
    t = 0.5
    assert v4 - (1.0 + 0.5 * dr) ** 4 == pytest.approx(-dr ** 4 * t * (t - 1) * (t - 2) * (t - 3), rel=1e-6)


def test_forward_stencil_nodes_and_cutoff():
    """Table = indicator of one node: the interpolant must be the Lagrange basis
    function of that node on the forward stencil k..k+3 (reading #4), and phi must
    vanish for r >= rc (reading #5)."""
    dr, rc = 0.1, 2.0
    ntab = int(round(rc / dr)) + 4
    T = np.zeros((1, ntab))
    T[0, 7] = 1.0
    sp = wl.Species("delta", rc, dr, np.array([0], dtype=np.int32), T)
    y00 = 0.5 / math.sqrt(math.pi)
    f = lambda r: oracle.phi([sp], 0, np.array([[r, 0.0, 0.0]]))[0, 0] / y00
    t = 0.25
    assert f((7 + t) * dr) == pytest.approx((1 - t) * (2 - t) * (3 - t) / 6, abs=1e-13)    # node is k
    assert f((6 + t) * dr) == pytest.approx(t * (2 - t) * (3 - t) / 2, abs=1e-13)          # node is k+1
    assert f((5 + t) * dr) == pytest.approx(-t * (1 - t) * (3 - t) / 2, abs=1e-13)         # k+2
    assert f((4 + t) * dr) == pytest.approx(t * (1 - t) * (2 - t) / 6, abs=1e-13)          # k+3
    assert f((8 + t) * dr) == 0.0 and f((3 + t) * dr) == 0.0
    T1 = np.ones((1, ntab))
    sp1 = wl.Species("one", rc, dr, np.array([0], dtype=np.int32), T1)
    assert oracle.phi([sp1], 0, np.array([[0.0, 0.0, rc]]))[0, 0] == 0.0
    assert oracle.phi([sp1], 0, np.array([[0.0, 0.0, np.nextafter(rc, 0)]]))[0, 0] == pytest.approx(y00, abs=1e-13)


def unit_table_species(ls, rc=2.0, dr=0.1):
    ntab = int(round(rc / dr)) + 4
    return wl.Species("unit", rc, dr, np.array(ls, dtype=np.int32), np.ones((len(ls), ntab)))


def test_unsold_and_orbital_order():
    sp = unit_table_species([0, 1, 2, 1])      # order of radial functions is kept as given (reading #8)
    rng = np.random.default_rng(2)
    d = rng.normal(size=(500, 3))
    d *= (rng.uniform(0.1, 1.9, size=500) / np.linalg.norm(d, axis=1))[:, None]
    Y = oracle.phi([sp], 0, d)
    assert Y.shape[1] == 1 + 3 + 5 + 3
    assert np.abs(Y[:, 0] ** 2 - 1 / (4 * math.pi)).max() < 1e-15
    assert np.abs((Y[:, 1:4] ** 2).sum(1) - 3 / (4 * math.pi)).max() < 1e-14
    assert np.abs((Y[:, 4:9] ** 2).sum(1) - 5 / (4 * math.pi)).max() < 1e-14
    assert np.abs(Y[:, 9:12] - Y[:, 1:4]).max() == 0.0


def test_ylm_orthonormal_under_spherical_quadrature():
    sp = unit_table_species([0, 1, 2])
    nth, nph = 12, 24
    x, wth = np.polynomial.legendre.leggauss(nth)
    ph = 2 * math.pi * np.arange(nph) / nph
    st = np.sqrt(1 - x * x)
    d = np.stack([np.outer(st, np.cos(ph)), np.outer(st, np.sin(ph)), np.outer(x, np.ones(nph))], axis=-1).reshape(-1, 3)
    wq = np.outer(wth, np.full(nph, 2 * math.pi / nph)).reshape(-1)
    Y = oracle.phi([sp], 0, d * 1.3)
    G = Y.T @ (Y * wq[:, None])
    assert np.abs(G - np.eye(9)).max() < 1e-13


def test_atom_on_mesh_point_r_zero():
    """Reading #6: at r = 0 the s orbital is f(0) Y00 and l > 0 orbitals vanish."""
    sp = unit_table_species([0, 1, 2])
    v = oracle.phi([sp], 0, np.zeros((1, 3)))[0]
    assert v[0] == pytest.approx(0.5 / math.sqrt(math.pi), abs=1e-15) and np.all(v[1:] == 0.0)
    w = wl.tiny(seed=3, natom=2)
    w.atom_pos[0] = (np.array([3, 4, 5]) / w.ngrid) @ w.lattice      # exactly on a mesh point
    H, blocks = run_oracle(w)
    assert np.all(np.isfinite(H))
    d = block_dict(H, blocks, norb_per_atom(w))
    ref = brute_force_block(w, 0, 1, (0, 0, 0))
    assert np.abs(d[(0, 1, 0, 0, 0)] - ref).max() <= 1e-13 * np.abs(H).max()


# ---------------------------------------------------------------------------
# 13. 90-degree rotation about z of atoms + V on a cubic mesh
# ---------------------------------------------------------------------------
def test_rotation_90_about_z():
    L, n = 9.0, 18
    lattice = np.diag([L, L, L])
    sp = wl.make_species("rot", 3.5, [(0, 0.6), (1, 0.5), (2, 0.7)])
    rng = np.random.default_rng(9)
    pos = rng.uniform(0, L, size=(3, 3))
    V = rng.normal(size=(n, n, n))
    H0, blocks0 = oracle.vlocal(lattice, [n] * 3, [sp], [0, 0, 0], pos, V)
    # rotate by +90 deg about z through the origin: (x,y,z) -> (-y,x,z); mesh index (i,j,k) -> (-j,i,k)
    pos_r = np.stack([-pos[:, 1], pos[:, 0], pos[:, 2]], axis=1)
    i, j, k = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    V_r = np.empty_like(V)
    V_r[(-j) % n, i, k] = V[i, j, k]
    H1, blocks1 = oracle.vlocal(lattice, [n] * 3, [sp], [0, 0, 0], pos_r, V_r)
    d0 = block_dict(H0, blocks0, [9] * 3)
    d1 = block_dict(H1, blocks1, [9] * 3)
    # orbital transformation phi'_m(Rr) = sum D phi(r): with x->-y', y->x' i.e. new (x',y') = (-y,x):
    # order: s | y z x | xy yz 3z2-1 xz x2-y2.  In rotated frame: y' = x, x' = -y
    #   p: y' <- x (idx 3), z' <- z, x' <- -y          d: x'y' = -xy; y'z' = xz; z2; x'z' = -yz; x'2-y'2 = -(x2-y2)
    D = np.zeros((9, 9))
    D[0, 0] = 1
    D[1, 3] = 1; D[2, 2] = 1; D[3, 1] = -1
    D[4, 4] = -1; D[5, 7] = 1; D[6, 6] = 1; D[7, 5] = -1; D[8, 8] = -1
    assert len(d0) == len(d1)
    scale = np.abs(H0).max()
    for (I, J, a, b, c), blk in d0.items():
        rot = d1[(I, J, -b, a, c)]
        assert np.abs(rot - D @ blk @ D.T).max() <= 1e-12 * scale


# ---------------------------------------------------------------------------
# 14. subset interface == full run; thread count independence
# ---------------------------------------------------------------------------
def test_block_subset_and_threads(cfg1, cfg1_oracle):
    w = cfg1
    H, (bi, bj, bR, off) = cfg1_oracle
    sel = np.sort(np.random.default_rng(0).choice(len(bi), 40, replace=False))
    Hs, (si, sj, sR, soff) = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V,
                                           blocks=(bi[sel], bj[sel], bR[sel]), nthreads=1)
    for n, b in enumerate(sel):
        assert np.array_equal(Hs[soff[n]:soff[n + 1]], H[off[b]:off[b + 1]])


def test_golden_regression_cfg1(cfg1, cfg1_oracle):
    """tests/golden/cfg1_oracle_sample.txt was written by tests/golden/make_golden.py (oracle only)."""
    import os
    H, blocks = cfg1_oracle
    d = block_dict(H, blocks, norb_per_atom(cfg1))
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle_sample.txt")
    lines = [l.split() for l in open(path) if not l.startswith("#")]
    header = [l for l in open(path) if l.startswith("# input sha256")][0].split()[-1]
    assert header == cfg1.sha256(), "seeded generator changed"
    assert len(lines) == 48
    for I, J, a, b, c, mu, nu, val in lines:
        got = d[(int(I), int(J), int(a), int(b), int(c))][int(mu), int(nu)]
        assert abs(float(val)) >= 1e-4 * np.abs(H).max()          # every stored value carries signal
        assert abs(got - float(val)) <= 1e-13 * abs(float(val))


# ---------------------------------------------------------------------------
# charge density (Eq. 44): pins of oracle.rho
# ---------------------------------------------------------------------------
def test_rho_adjoint_of_vlocal(cfg1, cfg1_oracle):
    """sum_g V(g) rho[D](g) dV = sum_blocks D : H[V] for ANY D (not symmetric) and ANY V: Eq. 44 is the adjoint of
    Eq. 45, and H comes from the already pinned orc_vlocal.  A dropped image, a transposed block or a wrong R sign in
    orc_rho breaks it (cfg1 has self-image blocks and several R per atom pair)."""
    w = cfg1
    H0, blocks = cfg1_oracle
    rng = np.random.default_rng(11)
    dV = abs(np.linalg.det(w.lattice)) / np.prod(w.ngrid)
    for trial in range(3):
        D = rng.normal(size=H0.shape)
        V = rng.normal(size=w.V.shape)
        HV, _ = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, V)
        r = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
        lhs, rhs = float((V * r).sum() * dV), float((D * HV).sum())
        assert abs(lhs - rhs) <= 1e-12 * np.abs(D).sum() * np.abs(HV).max()


def test_rho_brute_force_tiny():
    """Eq. 44 written out with explicit image sums R, R' in {-2..2}^3 on a tiny triclinic cell (numpy loops over the
    oracle's own phi only): rho(g) = sum_{I,J,R,R'} phi_I(r_g - tau_I - R')^T D(I,J,R) phi_J(r_g - tau_J - R - R')."""
    w = wl.tiny(seed=9, natom=2, ngrid=(6, 5, 7))
    H, blocks = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V)
    bi, bj, bR, off = blocks
    rng = np.random.default_rng(2)
    D = rng.normal(size=H.shape)
    got = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    pts = mesh_points(w.lattice, w.ngrid)
    norb = norb_per_atom(w)
    ref = np.zeros(len(pts))
    rng_img = range(-2, 3)
    phi_img = {}
    for I in range(w.natom):
        for a in rng_img:
            for b in rng_img:
                for c in rng_img:
                    Rv = np.array([a, b, c]) @ w.lattice
                    phi_img[(I, a, b, c)] = oracle.phi(w.species, int(w.atom_species[I]), pts - w.atom_pos[I] - Rv)
    for blk in range(len(bi)):
        I, J = int(bi[blk]), int(bj[blk])
        Dm = D[off[blk]:off[blk + 1]].reshape(norb[I], norb[J])
        for a in rng_img:
            for b in rng_img:
                for c in rng_img:
                    key = (J, a + int(bR[blk, 0]), b + int(bR[blk, 1]), c + int(bR[blk, 2]))
                    if key not in phi_img:
                        # image outside the explicit window: it must not reach any mesh point of the cell
                        Rv = np.array(key[1:]) @ w.lattice
                        assert not np.any(oracle.phi(w.species, int(w.atom_species[J]), pts - w.atom_pos[J] - Rv))
                        continue
                    ref += np.einsum("pm,mn,pn->p", phi_img[(I, a, b, c)], Dm, phi_img[key])
    assert np.abs(got.ravel() - ref).max() <= 1e-12 * np.abs(ref).max()


def test_rho_of_single_element_and_symmetry(cfg1, cfg1_oracle):
    """D with one non-zero element gives the product of two orbitals (sum over images); the partner block (J,I,-R)
    with the transposed matrix gives the same density."""
    w = cfg1
    H0, blocks = cfg1_oracle
    bi, bj, bR, off = blocks
    norb = norb_per_atom(w)
    b = int(np.nonzero((bi == 0) & (bj == 3))[0][0])
    D = np.zeros_like(H0)
    D[off[b] + 1 * norb[3] + 2] = 1.0            # mu = 1 of atom 0, nu = 2 of atom 3
    r1 = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    p = int(np.nonzero((bi == 3) & (bj == 0) & np.all(bR == -bR[b], axis=1))[0][0])
    D2 = np.zeros_like(H0)
    D2[off[p] + 2 * norb[0] + 1] = 1.0
    r2 = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D2, blocks)
    assert np.abs(r1).max() > 0 and np.abs(r1 - r2).max() <= 1e-14 * np.abs(r1).max()
    pts = mesh_points(w.lattice, w.ngrid)
    ref = np.zeros(len(pts))
    for a in range(-2, 3):
        for b_ in range(-2, 3):
            for c in range(-2, 3):
                Rp = np.array([a, b_, c]) @ w.lattice
                RJ = (np.array([a, b_, c]) + bR[b]) @ w.lattice
                ref += oracle.phi(w.species, int(w.atom_species[0]), pts - w.atom_pos[0] - Rp)[:, 1] * \
                    oracle.phi(w.species, int(w.atom_species[3]), pts - w.atom_pos[3] - RJ)[:, 2]
    assert np.abs(r1.ravel() - ref).max() <= 1e-13 * np.abs(ref).max()


# ---------------------------------------------------------------------------
# local Pulay force (Eq. 46): pins of oracle.phi_grad / oracle.fvl
# ---------------------------------------------------------------------------
def test_phi_grad_matches_finite_differences_of_phi():
    """grad phi (analytic angular part, derivative of the cubic interpolant for the radial part; readings #19, #20)
    against central differences of the pinned oracle.phi: a wrong Y_lm gradient, a dropped -l P rhat term or a wrong
    L_j' fails.  Points are kept away from table nodes, where the interpolant's derivative jumps by O(dr^3)."""
    sp = wl.make_species("x", 4.0, [(0, 0.6), (0, 1.1), (1, 0.5), (1, 0.9), (2, 0.7)], dr=0.01)
    rng = np.random.default_rng(5)
    u = rng.normal(size=(200, 3))
    u /= np.linalg.norm(u, axis=1)[:, None]
    r = (rng.integers(5, 380, size=200) + rng.uniform(0.3, 0.7, size=200)) * 0.01      # mid-interval radii
    d = u * r[:, None]
    ph, gr = oracle.phi_grad([sp], 0, d)
    assert np.abs(ph - oracle.phi([sp], 0, d)).max() <= 4e-16 * np.abs(ph).max()      # 3z^2-1 vs 2z^2-x^2-y^2
    h = 2e-5
    for c in range(3):
        e = np.zeros(3)
        e[c] = h
        fd = (oracle.phi([sp], 0, d + e) - oracle.phi([sp], 0, d - e)) / (2 * h)
        assert np.abs(gr[:, :, c] - fd).max() <= 2e-8 * max(1.0, np.abs(gr).max())
    # outside the cutoff the gradient is 0; at the nucleus only the p gradients survive (= c_1 f'(0) e_m, m = y, z, x)
    _, g_out = oracle.phi_grad([sp], 0, np.array([[4.0, 0.0, 0.0], [3.0, 3.0, 0.0]]))
    assert np.all(g_out == 0.0)
    _, g0 = oracle.phi_grad([sp], 0, np.zeros((1, 3)))
    _, g1 = oracle.phi_grad([sp], 0, np.array([[0.0, 0.0, 1e-9]]))       # just off the nucleus: same limit
    assert np.all(g0[0, :2] == 0.0) and np.all(g0[0, 8:] == 0.0)
    assert np.abs(g0[0, 2:8] - g1[0, 2:8]).max() <= 1e-6 * np.abs(g0).max()
    for blk in (g0[0, 2:5], g0[0, 5:8]):                                 # rows y, z, x -> e_y, e_z, e_x
        assert blk[0, 1] > 0 and blk[1, 2] == blk[0, 1] and blk[2, 0] == blk[0, 1]
        assert np.count_nonzero(blk) == 3


def _energy(w, D, blocks, pos):
    H, _ = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, pos, w.V, blocks=blocks[:3])
    return float(D @ H)


@pytest.mark.parametrize("on_mesh_point", [False, True])
def test_fvl_is_minus_dE_dtau_by_finite_differences(on_mesh_point):
    """F_K = -d/dtau_K [ sum_blocks D : H[V] ] at fixed V and D (reading #18), by central differences of the PINNED
    oracle.vlocal under a displaced atom, with a random NON-symmetric D (a transposed block index, a swapped
    derivative term or a wrong sign fails), on a triclinic cell with self-image blocks.  Second case: an atom exactly
    on a mesh point (reading #20)."""
    w = wl.tiny(seed=7, natom=3)
    if on_mesh_point:
        w.atom_pos[1] = (np.array([3, 4, 5]) / w.ngrid) @ w.lattice
    H, blocks = run_oracle(w)
    rng = np.random.default_rng(9)
    D = rng.normal(size=H.shape)
    F = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    scale = np.abs(F).max()
    assert scale > 1e-3
    for K in range(w.natom):
        for c in range(3):
            est = []
            for h in (4e-3, 2e-3):
                pp, pm = w.atom_pos.copy(), w.atom_pos.copy()
                pp[K, c] += h
                pm[K, c] -= h
                est.append(-(_energy(w, D, blocks, pp) - _energy(w, D, blocks, pm)) / (2 * h))
            rich = (4 * est[1] - est[0]) / 3                      # h^2 error removed
            assert abs(est[1] - F[K, c]) <= 4 * abs(est[1] - est[0]) + 1e-7 * scale       # consistent with O(h^2)
            assert abs(rich - F[K, c]) <= 2e-6 * scale, (K, c, rich, F[K, c])


def test_fvl_gaussian_closed_form():
    """Two Gaussian s orbitals, V = 1, D = one element: F_A = -dS/dA with S = N (pi/p)^{3/2} exp(-ab|A-B|^2/p)/(4 pi),
    i.e. F_A = +2ab/p (A - B) S, F_B = -F_A, as the mesh is refined (same quadrature behaviour as the overlap pin)."""
    alpha, beta = 0.7, 0.8
    for h, tol in ((0.5, 1e-6), (0.4, 1e-6)):
        lattice, ng, sp, asp, pos = two_gaussian_atoms(h, [(0, alpha)], [(0, beta)])
        bi, bj, bR, off = oracle.enumerate_blocks(lattice, sp, asp, pos)
        D = np.zeros(int(off[-1]))
        b = [k for k in range(len(bi)) if (bi[k], bj[k]) == (0, 1) and not bR[k].any()][0]
        D[off[b]] = 1.0
        F = oracle.fvl(lattice, ng, sp, asp, pos, np.ones(tuple(ng)), D, (bi, bj, bR, off))
        S = s0(alpha, beta, pos[0], pos[1]) / (4 * math.pi)
        exact = 2 * alpha * beta / (alpha + beta) * (pos[0] - pos[1]) * S
        assert np.abs(F[0] - exact).max() <= tol * np.abs(exact).max()
        assert np.abs(F[1] + exact).max() <= tol * np.abs(exact).max()


def test_fvl_shift_atoms_roll_V_and_linearity(cfg1, cfg1_oracle):
    """Shifting all atoms by one mesh vector and rolling V leaves F unchanged; F is linear in V and in D."""
    w = cfg1
    H, blocks = cfg1_oracle
    rng = np.random.default_rng(3)
    D = rng.normal(size=H.shape)
    F = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    shift = (np.array([1, 2, 3]) / w.ngrid) @ w.lattice
    F2 = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos + shift, np.roll(w.V, (1, 2, 3), (0, 1, 2)),
                    D, blocks)
    assert np.abs(F2 - F).max() <= 1e-11 * np.abs(F).max()
    V2 = rng.normal(size=w.V.shape)
    Fa = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, 2.0 * w.V - 0.5 * V2, D, blocks)
    Fb = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, V2, D, blocks)
    assert np.abs(Fa - (2.0 * F - 0.5 * Fb)).max() <= 1e-12 * np.abs(F).max()


# ---- l = 3 (f shells, reading #7 extended) --------------------------------------------------
def test_real_ylm_against_scipy_up_to_l3():
    """Every real Y_lm of the oracle, l = 0..3, against SciPy's complex harmonics (a library routine): with SciPy's
    Condon-Shortley Y_l^m, the real harmonic WITHOUT that phase is sqrt(2) (-1)^m Re Y_l^m (m > 0),
    sqrt(2) (-1)^m Im Y_l^|m| (m < 0), Y_l^0 (m = 0), in the order m = -l..l.  A wrong constant, sign, m-order or a
    swapped Cartesian factor in any of the 16 functions fails."""
    from scipy.special import sph_harm_y
    sp = unit_table_species([0, 1, 2, 3])
    rng = np.random.default_rng(41)
    d = rng.normal(size=(300, 3))
    d *= (rng.uniform(0.1, 1.9, size=300) / np.linalg.norm(d, axis=1))[:, None]
    Y = oracle.phi([sp], 0, d)
    assert Y.shape[1] == 16
    r = np.linalg.norm(d, axis=1)
    theta, phi = np.arccos(d[:, 2] / r), np.arctan2(d[:, 1], d[:, 0])
    col = 0
    for l in range(4):
        for m in range(-l, l + 1):
            y = sph_harm_y(l, abs(m), theta, phi)
            ref = y.real if m == 0 else math.sqrt(2) * (-1) ** m * (y.real if m > 0 else y.imag)
            assert np.abs(Y[:, col] - ref).max() < 1e-14, (l, m)
            col += 1


def test_f_shell_unsold_orthonormality_and_nucleus():
    sp = unit_table_species([3, 0, 3])
    rng = np.random.default_rng(42)
    d = rng.normal(size=(400, 3))
    d *= (rng.uniform(0.1, 1.9, size=400) / np.linalg.norm(d, axis=1))[:, None]
    Y = oracle.phi([sp], 0, d)
    assert Y.shape[1] == 7 + 1 + 7
    assert np.abs((Y[:, :7] ** 2).sum(1) - 7 / (4 * math.pi)).max() < 1e-14        # Unsold
    assert np.abs(Y[:, 8:] - Y[:, :7]).max() == 0.0
    sp = unit_table_species([0, 1, 2, 3])
    nth, nph = 12, 24
    x, wth = np.polynomial.legendre.leggauss(nth)
    ph = 2 * math.pi * np.arange(nph) / nph
    st = np.sqrt(1 - x * x)
    q = np.stack([np.outer(st, np.cos(ph)), np.outer(st, np.sin(ph)), np.outer(x, np.ones(nph))], axis=-1).reshape(-1, 3)
    wq = np.outer(wth, np.full(nph, 2 * math.pi / nph)).reshape(-1)
    Yq = oracle.phi([sp], 0, q * 1.3)
    assert np.abs(Yq.T @ (Yq * wq[:, None]) - np.eye(16)).max() < 1e-13
    v = oracle.phi([sp], 0, np.zeros((1, 3)))[0]
    assert v[0] != 0.0 and np.all(v[1:] == 0.0)                                   # reading #6


def test_f_shell_gradient_matches_finite_differences():
    """grad phi of an f shell (homogeneous cubic forms and their gradients, reading #19) against central differences
    of oracle.phi, whose l = 3 values are pinned against SciPy above."""
    sp = wl.make_species("f", 4.0, [(3, 0.6), (0, 0.8), (3, 1.0)], dr=0.01)
    rng = np.random.default_rng(43)
    u = rng.normal(size=(200, 3))
    u /= np.linalg.norm(u, axis=1)[:, None]
    r = (rng.integers(5, 380, size=200) + rng.uniform(0.3, 0.7, size=200)) * 0.01
    d = u * r[:, None]
    ph, gr = oracle.phi_grad([sp], 0, d)
    assert np.abs(ph - oracle.phi([sp], 0, d)).max() <= 1e-15 * np.abs(ph).max()
    h = 2e-5
    for c in range(3):
        e = np.zeros(3)
        e[c] = h
        fd = (oracle.phi([sp], 0, d + e) - oracle.phi([sp], 0, d - e)) / (2 * h)
        assert np.abs(gr[:, :, c] - fd).max() <= 2e-8 * max(1.0, np.abs(gr).max())
    _, g0 = oracle.phi_grad([sp], 0, np.zeros((1, 3)))
    assert np.all(g0[0, :7] == 0.0) and np.all(g0[0, 8:] == 0.0)                   # reading #20: only l = 1 survives


def test_f_shell_brute_force_and_force_fd():
    """Whole pipeline with an f shell on a triclinic cell: H blocks against the dense enlarged-window sum, and the
    force against Richardson-extrapolated central differences of the energy D : H[V] (as for l <= 2 above)."""
    w = wl.tiny(seed=13, natom=2, ngrid=(10, 9, 11), shells=((0, 0.7), (3, 0.6)), rcut=3.0)
    H, blocks = run_oracle(w)
    d = block_dict(H, blocks, norb_per_atom(w))
    scale = np.abs(H).max()
    keys = list(d.keys())
    for k in keys[::max(1, len(keys) // 10)]:
        ref = brute_force_block(w, k[0], k[1], k[2:])
        assert np.abs(d[k] - ref).max() <= 1e-13 * scale, k
    rng = np.random.default_rng(44)
    D = rng.normal(size=H.shape)
    F = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    fs = np.abs(F).max()
    for K in range(w.natom):
        for c in range(3):
            est = []
            for h in (4e-3, 2e-3):
                pp, pm = w.atom_pos.copy(), w.atom_pos.copy()
                pp[K, c] += h
                pm[K, c] -= h
                est.append(-(_energy(w, D, blocks, pp) - _energy(w, D, blocks, pm)) / (2 * h))
            rich = (4 * est[1] - est[0]) / 3
            assert abs(rich - F[K, c]) <= 2e-6 * fs, (K, c, rich, F[K, c])
