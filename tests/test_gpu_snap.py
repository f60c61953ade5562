"""Parity of gint_snap_psibeta (CUDA, through the C ABI) against oracle.snap_psibeta, element by element on the same
seeded inputs: S(I, J, R) = <phi| exp(-i A.r) |beta> by atom-centred quadrature (Eq. 47).
Bar: max|S_gpu - S_ref| <= 1e-10 * max|S_ref| (both sides are FP64 sums of the same 15 400 terms per element)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _quad():
    from paper_2603_21835_b200 import workloads as wl
    return wl.radial_quadrature(140) + wl.angular_quadrature(110)


def _context(w, proj, species=None, atom_species=None):
    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(w.lattice, w.ngrid, w.species if species is None else species,
                     w.atom_species if atom_species is None else atom_species, w.atom_pos, cuda_device=0)
    ctx.gint_snap_setup(proj, *_quad())
    return ctx


def _same_pairs(a, b):
    return all(np.array_equal(x, y) for x, y in zip(a, b))


def _compare(ctx, w, proj, A, species=None, atom_species=None, what=""):
    torch = _torch()
    import oracle
    sp = w.species if species is None else species
    asp = w.atom_species if atom_species is None else atom_species
    ref, pairs = oracle.snap_psibeta(w.lattice, sp, proj, asp, w.atom_pos, A, *_quad())
    assert _same_pairs(pairs, ctx.gint_snap_get_pairs()), what
    got = ctx.gint_snap_psibeta(A)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    scale = np.abs(ref).max()
    err = np.abs(got - ref).max()
    assert np.all(np.isfinite(got.real)) and np.all(np.isfinite(got.imag))
    assert err <= TOL * scale, "%s: max|dS| = %.3e, scale %.3e, rel %.3e" % (what, err, scale, err / scale)
    return got


@pytest.mark.parametrize("A", [(0.0, 0.0, 0.0), (0.1, -0.05, 0.2), (1.3, 0.4, -0.9)])
def test_cfg1_all_pairs(cfg1, A):
    """si8_sz: a small periodic cell, so most pairs are image pairs (R != 0); s and p orbitals against two s and two p
    projectors; A = 0 (real overlaps), a weak and a strong field."""
    from paper_2603_21835_b200 import workloads as wl
    proj = [wl.projector_species()]
    ctx = _context(cfg1, proj)
    got = _compare(ctx, cfg1, proj, A, what="si8_sz A=%s" % (A,))
    if A == (0.0, 0.0, 0.0):
        assert np.abs(got.imag).max() == 0.0


def test_triclinic_two_species_f_orbitals_d_projectors():
    """General lattice, one species with s..f orbitals and s, p, d projectors, one with a single s orbital and NO
    projectors (it hosts no pair but appears on the orbital side), an atom exactly on another's quadrature centre
    excluded by construction; ragged quadrature tail (15 400 points are not a multiple of 128)."""
    from paper_2603_21835_b200 import workloads as wl
    w = wl.tiny(seed=9, natom=5, ngrid=(12, 12, 12), rcut=3.0)
    big = wl.make_species("A", 3.0, [(0, 0.6), (1, 0.5), (2, 0.7), (3, 0.8)])
    small = wl.make_species("B", 2.4, [(0, 0.9)])
    none = wl.Species(name="none", rcut=0.0, dr=0.01, l=np.zeros(0, np.int32), table=np.zeros((0, 8)))
    proj = [wl.make_species("beta", 2.0, [(0, 1.5), (1, 1.8), (2, 2.2)]), none]
    asp = np.array([0, 1, 0, 1, 0], dtype=np.int32)
    ctx = _context(w, proj, species=[big, small], atom_species=asp)
    iat = ctx.gint_snap_get_pairs()[0]
    assert set(iat.tolist()) == {0, 2, 4}
    _compare(ctx, w, proj, (0.3, -0.2, 0.25), species=[big, small], atom_species=asp, what="triclinic")


@pytest.mark.parametrize("name", ["si64_dzp", "si64_tzdp"])
def test_cfg2_sizes_all_pairs(name):
    """64 atoms, 13 orbitals (2 x 2 accumulator fragments) and the paper's 22-orbital TZDP basis (4 x 4 fragments)."""
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make(name)
    proj = [wl.projector_species()]
    ctx = _context(w, proj)
    _compare(ctx, w, proj, (0.12, 0.07, -0.21), what=name)


def test_reproducible_and_tied_to_the_geometry(cfg1):
    """No atomics: two calls agree bit for bit.  Moving the atoms discards the pair list (the call then fails until
    gint_snap_setup is repeated), and the new result equals the oracle at the new positions."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    from paper_2603_21835_b200.binding import GintError
    proj = [wl.projector_species()]
    ctx = _context(cfg1, proj)
    A = (0.2, 0.1, -0.15)
    a = ctx.gint_snap_psibeta(A).clone()
    b = ctx.gint_snap_psibeta(A)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    rng = np.random.default_rng(5)
    pos2 = cfg1.atom_pos + rng.uniform(-0.2, 0.2, size=cfg1.atom_pos.shape)
    ctx.gint_update_positions(pos2)
    with pytest.raises(GintError):
        ctx.gint_snap_psibeta(A)
    ctx.gint_snap_setup(proj, *_quad())
    got = ctx.gint_snap_psibeta(A).cpu().numpy()
    ref, pairs = oracle.snap_psibeta(cfg1.lattice, cfg1.species, proj, cfg1.atom_species, pos2, A, *_quad())
    assert _same_pairs(pairs, ctx.gint_snap_get_pairs())
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_headline_size_sampled_pairs():
    """si512_dzp in the launch configuration bench.py times: the pair list against a count by k-d tree, and 150
    sampled pairs (on-site, neighbours, image pairs) against the oracle, each block element by element."""
    torch = _torch()
    import oracle
    from scipy.spatial import cKDTree
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make("si512_dzp")
    proj = [wl.projector_species()]
    ctx = _context(w, proj)
    iat, jat, R, off = ctx.gint_snap_get_pairs()
    cut = float(proj[0].rcut) + float(w.species[0].rcut)
    shifts = np.array([(i, j, k) for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1)])
    images = (w.atom_pos[None, :, :] + (shifts @ w.lattice)[:, None, :]).reshape(-1, 3)
    tree = cKDTree(images)
    count = sum(sum(1 for k in tree.query_ball_point(w.atom_pos[I], cut) if np.linalg.norm(images[k] - w.atom_pos[I]) < cut)
                for I in range(w.natom))
    assert count == len(iat)
    A = (0.08, -0.11, 0.05)
    got = ctx.gint_snap_psibeta(A)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    rng = np.random.default_rng(11)
    pick = np.unique(np.concatenate([rng.choice(len(iat), 120, replace=False),
                                     np.flatnonzero((iat == jat) & np.all(R == 0, axis=1))[:10],
                                     np.flatnonzero(np.any(R != 0, axis=1))[:20]]))
    n = off[1:] - off[:-1]
    sub_off = np.concatenate([[0], np.cumsum(n[pick])]).astype(np.int64)
    ref, _ = oracle.snap_psibeta(w.lattice, w.species, proj, w.atom_species, w.atom_pos, A, *_quad(),
                                 pairs=(iat[pick], jat[pick], R[pick], sub_off))
    scale = np.abs(got).max()
    for q, b in enumerate(pick):
        d = np.abs(got[off[b]:off[b + 1]] - ref[sub_off[q]:sub_off[q + 1]]).max()
        assert d <= TOL * scale, (int(b), d / scale)


def test_sharded_contexts_cover_all_pairs(cfg1):
    """nranks = 2 on one GPU: every rank computes the pairs of its projector atoms; together they reproduce the
    unsharded result block by block (no collective on this path)."""
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    proj = [wl.projector_species()]
    A = (0.1, -0.05, 0.2)
    full_ctx = _context(cfg1, proj)
    full = full_ctx.gint_snap_psibeta(A).cpu().numpy()
    fi, fj, fR, foff = full_ctx.gint_snap_get_pairs()
    index = {(int(fi[b]), int(fj[b])) + tuple(int(x) for x in fR[b]): b for b in range(len(fi))}
    seen = 0
    for rank in range(2):
        ctx = gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cuda_device=0,
                         rank=rank, nranks=2)
        ctx.gint_snap_setup(proj, *_quad())
        S = ctx.gint_snap_psibeta(A).cpu().numpy()
        iat, jat, R, off = ctx.gint_snap_get_pairs()
        assert np.all(iat % 2 == rank)
        for b in range(len(iat)):
            g = index[(int(iat[b]), int(jat[b])) + tuple(int(x) for x in R[b])]
            assert np.array_equal(S[off[b]:off[b + 1]], full[foff[g]:foff[g + 1]])   # same kernel, same order: bit-wise
        seen += len(iat)
    assert seen == len(fi)
