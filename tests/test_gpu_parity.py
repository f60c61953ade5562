"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by
element, on the same seeded inputs.  Bar (BASELINE.json north_star):
    max|H_gpu - H_ref| <= 1e-10 * max|H_ref|   in FP64.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def gpu_H(w, V=None, **kw):
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=0, **kw)
    Vd = torch.from_numpy(np.ascontiguousarray(w.V if V is None else V)).cuda()
    H = ctx.gint_vlocal(Vd)
    torch.cuda.synchronize()
    return H.cpu().numpy(), ctx


def oracle_H(w, V=None, blocks=None):
    import oracle
    return oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V if V is None else V,
                         blocks=blocks)


def assert_blocks_equal(ctx, blocks):
    bi, bj, bR, off = blocks
    i2, j2, R2, o2 = ctx.gint_get_blocks()
    assert np.array_equal(bi, i2) and np.array_equal(bj, j2) and np.array_equal(bR, R2) and np.array_equal(off, o2)


def assert_parity(Hg, Hr, what=""):
    scale = np.abs(Hr).max()
    err = np.abs(Hg - Hr).max()
    assert np.all(np.isfinite(Hg))
    assert err <= TOL * scale, "%s: max|dH| = %.3e, scale %.3e, rel %.3e" % (what, err, scale, err / scale)
    return err / scale


def test_cfg1_full(cfg1, cfg1_oracle):
    Hr, blocks = cfg1_oracle
    Hg, ctx = gpu_H(cfg1)
    assert_blocks_equal(ctx, blocks)
    assert_parity(Hg, Hr, "si8_sz")


@pytest.mark.parametrize("seed,ngrid", [(7, (12, 10, 14)), (11, (9, 13, 7)), (5, (16, 16, 16))])
def test_tiny_triclinic_ragged(seed, ngrid):
    """General lattice, mesh not divisible by the big-cell edge (ragged last cells),
    self-image blocks, s+p+d shells."""
    from paper_2603_21835_b200 import workloads as wl
    w = wl.tiny(seed=seed, ngrid=ngrid)
    Hr, blocks = oracle_H(w)
    Hg, ctx = gpu_H(w)
    assert_blocks_equal(ctx, blocks)
    assert_parity(Hg, Hr, "tiny seed %d" % seed)


@pytest.mark.parametrize("bcell", [(4, 4, 4), (2, 2, 2), (1, 1, 4), (3, 2, 4), (4, 4, 2), (2, 8, 4), (1, 1, 36), (1, 1, 300)])
def test_big_cell_shapes(cfg1, cfg1_oracle, bcell):
    Hr, _ = cfg1_oracle
    Hg, _ = gpu_H(cfg1, bcell=bcell)
    assert_parity(Hg, Hr, "bcell %s" % (bcell,))


def test_repeat_calls_overwrite_and_new_V(cfg1, cfg1_oracle):
    """gint_vlocal overwrites H and may be called repeatedly with different V (SCF loop)."""
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup
    w = cfg1
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    H = torch.full((ctx.h_len,), 7.0, dtype=torch.float64, device="cuda")
    V1 = torch.from_numpy(w.V).cuda()
    rng = np.random.default_rng(0)
    V2h = rng.normal(size=w.V.shape)
    ctx.gint_vlocal(V1, H)
    ctx.gint_vlocal(torch.from_numpy(V2h).cuda(), H)
    ctx.gint_vlocal(V1, H)
    torch.cuda.synchronize()
    assert_parity(H.cpu().numpy(), cfg1_oracle[0], "third call")
    ctx.gint_vlocal(torch.from_numpy(V2h).cuda(), H)
    Hr2, _ = oracle_H(w, V=V2h)
    assert_parity(H.cpu().numpy(), Hr2, "V2")
    # side stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        H3 = ctx.gint_vlocal(V1)
    s.synchronize()
    assert_parity(H3.cpu().numpy(), cfg1_oracle[0], "side stream")


def test_host_buffer_entry_point(cfg1, cfg1_oracle):
    _torch()
    from paper_2603_21835_b200 import gint_setup
    w = cfg1
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    Hh = ctx.gint_vlocal_host(w.V)
    assert_parity(Hh, cfg1_oracle[0], "gint_vlocal_host")


def test_gpu_symmetry_exact(cfg1):
    """The mirror kernel makes H(J,I,-R) the exact transpose of H(I,J,R)."""
    from helpers import block_dict, norb_per_atom
    Hg, ctx = gpu_H(cfg1)
    d = block_dict(Hg, ctx.gint_get_blocks(), norb_per_atom(cfg1))
    for (I, J, a, b, c), blk in d.items():
        assert np.array_equal(blk, d[(J, I, -a, -b, -c)].T)


def test_edge_cases():
    """Single atom (only self blocks); atom exactly on a mesh point; far-apart atoms
    (empty cells, zero cross blocks absent); mesh smaller than a big cell."""
    from paper_2603_21835_b200 import workloads as wl
    w = wl.tiny(seed=3, natom=1)
    assert_parity(gpu_H(w)[0], oracle_H(w)[0], "single atom")
    w = wl.tiny(seed=3, natom=2)
    w.atom_pos[0] = (np.array([3, 4, 5]) / w.ngrid) @ w.lattice
    assert_parity(gpu_H(w)[0], oracle_H(w)[0], "atom on mesh point")
    w = wl.tiny(seed=4, natom=2, ngrid=(40, 40, 40), lattice=np.eye(3) * 20.0, rcut=2.0)
    w.atom_pos[:] = [[3.0, 3.0, 3.0], [13.0, 13.0, 13.0]]
    Hg, ctx = gpu_H(w)
    assert ctx.nblocks == 2
    assert_parity(Hg, oracle_H(w)[0], "far apart")
    w = wl.tiny(seed=6, natom=2, ngrid=(3, 2, 3), rcut=2.0)
    assert_parity(gpu_H(w)[0], oracle_H(w)[0], "mesh smaller than a big cell")


def test_V_zero_and_constant(cfg1):
    Hg, _ = gpu_H(cfg1, V=np.zeros_like(cfg1.V))
    assert np.all(Hg == 0.0)
    S, _ = gpu_H(cfg1, V=np.ones_like(cfg1.V))
    Hc, _ = gpu_H(cfg1, V=np.full_like(cfg1.V, -0.37))
    assert np.abs(Hc + 0.37 * S).max() <= 1e-13 * np.abs(S).max()


def test_cluster60_full():
    """cfg5: two species (13 and 5 orbitals), empty big cells, dense core (cells split in K)."""
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make("cluster60")
    Hr, blocks = oracle_H(w)
    Hg, ctx = gpu_H(w)
    assert_blocks_equal(ctx, blocks)
    assert np.all(blocks[2] == 0)      # R = 0 only
    assert_parity(Hg, Hr, "cluster60")


def test_cfg2_full():
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make("si64_dzp")
    Hr, blocks = oracle_H(w)
    Hg, ctx = gpu_H(w)
    assert_blocks_equal(ctx, blocks)
    assert_parity(Hg, Hr, "si64_dzp")


@pytest.mark.parametrize("name", ["si216_dzp", "si512_dzp"])
def test_large_full_output(name):
    """Full-size configs in the launch configuration bench.py times (default big cells, whole work queue, the
    multi-GB psi scratch): EVERY element of H against the oracle at the 1e-10 bar, plus exact transpose symmetry."""
    from paper_2603_21835_b200 import workloads as wl
    from helpers import norb_per_atom
    w = wl.make(name)
    Hg, ctx = gpu_H(w)
    Hr, blocks = oracle_H(w)
    assert_blocks_equal(ctx, blocks)
    assert_parity(Hg, Hr, name)
    bi, bj, bR, off = blocks
    rng = np.random.default_rng(42)
    norb = norb_per_atom(w)
    key = {(int(bi[b]), int(bj[b]), int(bR[b, 0]), int(bR[b, 1]), int(bR[b, 2])): b for b in range(len(bi))}
    for b in rng.choice(len(bi), 2000, replace=False):
        p = key[(int(bj[b]), int(bi[b]), -int(bR[b, 0]), -int(bR[b, 1]), -int(bR[b, 2]))]
        A = Hg[off[b]:off[b + 1]].reshape(norb[bi[b]], norb[bj[b]])
        B = Hg[off[p]:off[p + 1]].reshape(norb[bj[b]], norb[bi[b]])
        assert np.array_equal(A, B.T)


def _sharded_cases():
    from paper_2603_21835_b200 import workloads as wl
    return [("si8_sz", lambda: wl.make("si8_sz")), ("tiny_ragged", lambda: wl.tiny(seed=7, ngrid=(12, 10, 14))),
            ("tiny_9_13_7", lambda: wl.tiny(seed=11, ngrid=(9, 13, 7))), ("si64_dzp", lambda: wl.make("si64_dzp"))]


@pytest.mark.parametrize("nranks", [2, 3])
@pytest.mark.parametrize("case", [0, 1, 2, 3])
def test_sharded_kernel_path_sums_to_oracle(case, nranks):
    """The multi-GPU path on the one GPU there is: one context per rank with
    gint_options.rank/nranks, every rank's gint_vlocal and gint_rho run on cuda:0, the partial H / rho buffers summed
    (what the all-reduce does) and compared with the oracle; gint_fold_k on the summed H.  The tiny cases have fewer
    cell layers along a1 than ranks, so some rank owns no work at all (its H must be all zeros)."""
    torch = _torch()
    import oracle
    from helpers import norb_per_atom
    from paper_2603_21835_b200 import gint_setup
    name, mk = _sharded_cases()[case]
    w = mk()
    Hr, blocks = oracle_H(w)
    rng = np.random.default_rng(100 + case)
    D = rng.normal(size=Hr.shape)
    rho_ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    Vd = torch.from_numpy(w.V).cuda()
    Dd = torch.from_numpy(D).cuda()
    Hsum = torch.zeros(Hr.shape[0], dtype=torch.float64, device="cuda")
    rsum = torch.zeros(tuple(int(x) for x in w.ngrid), dtype=torch.float64, device="cuda")
    fsum, empty_ranks, ctx = 0.0, 0, None
    for r in range(nranks):
        ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=0, rank=r, nranks=nranks)
        assert_blocks_equal(ctx, blocks)
        st = ctx.gint_get_stats()
        fsum += st["F_sym"]
        Hp = ctx.gint_vlocal(Vd)
        rp = ctx.gint_rho(Dd)
        if st["items"] == 0:
            empty_ranks += 1
            assert float(Hp.abs().max()) == 0.0 and float(rp.abs().max()) == 0.0
        Hsum += Hp
        rsum += rp
    torch.cuda.synchronize()
    full = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1).gint_get_stats()
    assert fsum == full["F_sym"]
    if name.startswith("tiny") and nranks == 3:
        assert empty_ranks >= 1
    assert_parity(Hsum.cpu().numpy(), Hr, "%s sharded x%d" % (name, nranks))
    assert np.abs(rsum.cpu().numpy() - rho_ref).max() <= TOL * np.abs(rho_ref).max()
    kf = (0.31, -0.17, 0.43)
    Hk = ctx.gint_fold_k(Hsum, kf).cpu().numpy()
    ref = oracle.fold_k(Hr, blocks, norb_per_atom(w), kf)
    assert np.abs(Hk - ref).max() <= 1e-10 * np.abs(ref).max()


def test_repeatability_stress():
    """The contraction kernel is a producer/consumer pipeline (bulk copies, mbarrier rings, dynamic queue) whose
    timing differs from call to call; 25 calls on the 64-atom workload must agree to rounding (the order of the
    atomic adds is the only freedom), which a stale or early read of a ring stage would break."""
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    w = wl.make("si64_dzp")
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    V = torch.from_numpy(w.V).cuda()
    H0 = ctx.gint_vlocal(V).clone()
    scale = float(H0.abs().max())
    H = torch.empty_like(H0)
    junk = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device="cuda")
    for i in range(25):
        if i % 3 == 0:
            junk.normal_()          # perturb cache state and timing
        ctx.gint_vlocal(V, H)
        assert float((H - H0).abs().max()) <= 1e-12 * scale, "call %d differs" % i


@pytest.mark.parametrize("kfrac", [(0.0, 0.0, 0.0), (0.31, -0.17, 0.43), (0.5, 0.25, -0.4)])
def test_fold_k_against_oracle(cfg1, kfrac):
    """H(k) = sum_R exp(i k.R) H(R) (Eq. 5) from the GPU blocks against the oracle's folding of the
    same blocks, element by element; self-image blocks (several R per atom pair) are what cfg1 is for."""
    torch = _torch()
    import oracle
    from helpers import norb_per_atom
    Hg, ctx = gpu_H(cfg1)
    Hk = ctx.gint_fold_k(torch.from_numpy(Hg).cuda(), kfrac)
    torch.cuda.synchronize()
    ref = oracle.fold_k(Hg, ctx.gint_get_blocks(), norb_per_atom(cfg1), kfrac)
    n, first = ctx.gint_num_orbitals()
    assert n == ref.shape[0] and np.array_equal(first, np.concatenate([[0], np.cumsum(norb_per_atom(cfg1))]))
    got = Hk.cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(got - got.conj().T).max() <= 1e-13 * np.abs(ref).max()      # Hermitian: H(R) = H(-R)^T


def test_fold_k_cluster_and_large():
    """Two species with different orbital counts (cluster60, R = 0 only: H(k) is real and k-independent), and the
    headline size: Gamma point of si512_dzp equals the plain block sum on sampled atom pairs."""
    torch = _torch()
    import oracle
    from helpers import norb_per_atom
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make("cluster60")
    Hg, ctx = gpu_H(w)
    Hd = torch.from_numpy(Hg).cuda()
    a = ctx.gint_fold_k(Hd, (0.0, 0.0, 0.0)).cpu().numpy()
    b = ctx.gint_fold_k(Hd, (0.37, 0.11, -0.29)).cpu().numpy()
    ref = oracle.fold_k(Hg, ctx.gint_get_blocks(), norb_per_atom(w), (0.0, 0.0, 0.0))
    assert np.abs(a - ref).max() <= 1e-13 * np.abs(ref).max() and np.array_equal(a, b) and np.all(a.imag == 0)
    w = wl.make("si512_dzp")
    Hg, ctx = gpu_H(w)
    Hk = ctx.gint_fold_k(torch.from_numpy(Hg).cuda(), (0.25, 0.5, -0.125)).cpu().numpy()
    bi, bj, bR, off = ctx.gint_get_blocks()
    norb = norb_per_atom(w)
    first = np.concatenate([[0], np.cumsum(norb)])
    rng = np.random.default_rng(3)
    scale = np.abs(Hg).max()
    for b in rng.choice(len(bi), 200, replace=False):
        I, J = int(bi[b]), int(bj[b])
        sel = np.nonzero((bi == I) & (bj == J))[0]
        ref = sum(np.exp(2j * np.pi * float(np.dot((0.25, 0.5, -0.125), bR[s]))) *
                  Hg[off[s]:off[s + 1]].reshape(norb[I], norb[J]) for s in sel)
        assert np.abs(Hk[first[I]:first[I + 1], first[J]:first[J + 1]] - ref).max() <= 1e-13 * scale
    # an atom pair without any block stays zero
    has = set(zip(bi.tolist(), bj.tolist()))
    I, J = next((i, j) for i in range(w.natom) for j in range(w.natom) if (i, j) not in has)
    assert np.all(Hk[first[I]:first[I + 1], first[J]:first[J + 1]] == 0)


def gpu_rho(w, D, **kw):
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=0, **kw)
    r = ctx.gint_rho(torch.from_numpy(np.ascontiguousarray(D)).cuda())
    torch.cuda.synchronize()
    return r.cpu().numpy(), ctx


def test_rho_cfg1_and_tiny(cfg1, cfg1_oracle):
    """Charge density (Eq. 44) against the oracle, element by element, with a random NON-symmetric
    D: cfg1 (self-image blocks), ragged triclinic meshes, then a gint_vlocal call on the same context (shared psi
    scratch) still matches."""
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    rng = np.random.default_rng(21)
    H0, blocks = cfg1_oracle
    D = rng.normal(size=H0.shape)
    ref = oracle.rho(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, D, blocks)
    got, ctx = gpu_rho(cfg1, D)
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
    torch = _torch()
    H = ctx.gint_vlocal(torch.from_numpy(cfg1.V).cuda())
    assert_parity(H.cpu().numpy(), H0, "vlocal after rho")
    for seed, ngrid in [(7, (12, 10, 14)), (11, (9, 13, 7))]:
        w = wl.tiny(seed=seed, ngrid=ngrid)
        Hr, blk = oracle_H(w)
        D = rng.normal(size=Hr.shape)
        ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blk)
        got, _ = gpu_rho(w, D)
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_rho_cfg2_and_cluster():
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    rng = np.random.default_rng(22)
    for name in ("si64_dzp", "cluster60"):
        w = wl.make(name)
        bi, bj, bR, off = oracle.enumerate_blocks(w.lattice, w.species, w.atom_species, w.atom_pos)
        D = rng.normal(size=int(off[-1]))
        ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, (bi, bj, bR, off))
        got, ctx = gpu_rho(w, D)
        assert np.array_equal(ctx.gint_get_blocks()[3], off)
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max(), name


def test_rho_large_full_mesh():
    """si512_dzp at full size: every mesh point of rho against the oracle at the 1e-10 bar (random NON-symmetric D),
    and the adjoint identity sum_g V rho dV = D : H[V] with H from gint_vlocal on the same context."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    w = wl.make("si512_dzp")
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    rng = np.random.default_rng(23)
    D = rng.normal(size=ctx.h_len)
    Dd = torch.from_numpy(D).cuda()
    rho = ctx.gint_rho(Dd)
    Vd = torch.from_numpy(w.V).cuda()
    H = ctx.gint_vlocal(Vd)
    dV = abs(np.linalg.det(w.lattice)) / np.prod(w.ngrid)
    lhs, rhs = float((Vd * rho).sum()) * dV, float((Dd * H).sum())
    # both sides are sums of ~1e7 terms of size <= max|H| max|D|: 1e-10 of the largest partial sum
    assert abs(lhs - rhs) <= 1e-10 * float((Dd * H).abs().sum())
    ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, ctx.gint_get_blocks())
    got = rho.cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


# ---- gint_fvl: local Pulay force (Eq. 46) ------------------------------------------------------
def gpu_fvl(w, D, **kw):
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, **kw)
    F = ctx.gint_fvl(torch.from_numpy(np.ascontiguousarray(w.V)).cuda(), torch.from_numpy(np.ascontiguousarray(D)).cuda())
    torch.cuda.synchronize()
    return F.cpu().numpy(), ctx


def assert_force_parity(got, ref, what):
    assert np.all(np.isfinite(got)), what
    err = np.abs(got - ref).max()
    assert err <= TOL * np.abs(ref).max(), "%s: max|dF| %.3e vs max|F| %.3e" % (what, err, np.abs(ref).max())


def test_fvl_cfg1_and_tiny(cfg1, cfg1_oracle):
    """Force of Eq. 46 against the oracle with a random NON-symmetric D: cfg1 (self-image blocks), ragged triclinic
    meshes (s, p, d shells), an atom on a mesh point (r = 0 rule), then gint_vlocal and gint_rho on the same context
    still match (shared scratch)."""
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    rng = np.random.default_rng(31)
    H0, blocks = cfg1_oracle
    D = rng.normal(size=H0.shape)
    ref = oracle.fvl(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cfg1.V, D, blocks)
    got, ctx = gpu_fvl(cfg1, D)
    assert_force_parity(got, ref, "cfg1")
    torch = _torch()
    H = ctx.gint_vlocal(torch.from_numpy(cfg1.V).cuda())
    assert_parity(H.cpu().numpy(), H0, "vlocal after fvl")
    rho_ref = oracle.rho(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, D, blocks)
    rho = ctx.gint_rho(torch.from_numpy(D).cuda()).cpu().numpy()
    assert np.abs(rho - rho_ref).max() <= TOL * np.abs(rho_ref).max()
    got2 = ctx.gint_fvl(torch.from_numpy(cfg1.V).cuda(), torch.from_numpy(D).cuda()).cpu().numpy()
    assert_force_parity(got2, ref, "cfg1, second call")
    for seed, ngrid in [(7, (12, 10, 14)), (11, (9, 13, 7))]:
        w = wl.tiny(seed=seed, ngrid=ngrid)
        Hr, blk = oracle_H(w)
        D = rng.normal(size=Hr.shape)
        ref = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blk)
        got, _ = gpu_fvl(w, D)
        assert_force_parity(got, ref, "tiny %d" % seed)
    # an atom exactly on a mesh point
    w = wl.tiny(seed=5, ngrid=(12, 12, 12))
    pos = np.array(w.atom_pos, dtype=np.float64)
    pos[0] = (np.array([3, 4, 5]) / 12.0) @ np.asarray(w.lattice)
    w.atom_pos = pos
    Hr, blk = oracle_H(w)
    D = rng.normal(size=Hr.shape)
    ref = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blk)
    got, _ = gpu_fvl(w, D)
    assert_force_parity(got, ref, "atom on a mesh point")


def test_fvl_cfg2_and_cluster():
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    rng = np.random.default_rng(32)
    for name in ("si64_dzp", "cluster60"):
        w = wl.make(name)
        blocks = oracle.enumerate_blocks(w.lattice, w.species, w.atom_species, w.atom_pos)
        D = rng.normal(size=int(blocks[3][-1]))
        ref = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
        got, _ = gpu_fvl(w, D)
        assert_force_parity(got, ref, name)


def test_fvl_sharded_sums_to_oracle(cfg1, cfg1_oracle):
    """nranks = 2, 3 on one GPU: the partial forces of the ranks sum to the oracle's."""
    import oracle
    rng = np.random.default_rng(33)
    H0, blocks = cfg1_oracle
    D = rng.normal(size=H0.shape)
    ref = oracle.fvl(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cfg1.V, D, blocks)
    for nranks in (2, 3):
        tot = np.zeros_like(ref)
        for rank in range(nranks):
            got, _ = gpu_fvl(cfg1, D, rank=rank, nranks=nranks)
            tot += got
        assert_force_parity(tot, ref, "nranks %d" % nranks)


def test_fvl_large_full():
    """si512_dzp at full size: all 512 x 3 force components against the oracle at the 1e-10 bar."""
    import oracle
    from paper_2603_21835_b200 import workloads as wl
    w = wl.make("si512_dzp")
    rng = np.random.default_rng(34)
    blocks = oracle.enumerate_blocks(w.lattice, w.species, w.atom_species, w.atom_pos)
    D = rng.normal(size=int(blocks[3][-1]))
    got, ctx = gpu_fvl(w, D)
    assert np.array_equal(ctx.gint_get_blocks()[3], blocks[3])
    ref = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    assert_force_parity(got, ref, "si512_dzp")


# ---- second workloads: f shell, the paper's TZDP basis, rc = 10 ------------------------------
@pytest.mark.parametrize("name", ["si8_dzpf", "si64_tzdp", "si64_dzp_rc10"])
def test_second_workloads_all_three_calls(name):
    """gint_vlocal, gint_rho and gint_fvl element by element against the oracle on: an f shell (l = 3, 20 orbitals),
    TZDP 3s3p2d = 22 orbitals per atom (the basis of the paper's performance runs) and rc = 10 a.u.
    (its validation cutoff)."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    w = wl.make(name)
    Hr, blocks = oracle_H(w)
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    assert np.array_equal(ctx.gint_get_blocks()[3], blocks[3])
    Vd = torch.from_numpy(w.V).cuda()
    assert_parity(ctx.gint_vlocal(Vd).cpu().numpy(), Hr, name)
    rng = np.random.default_rng(51)
    D = rng.normal(size=Hr.shape)
    Dd = torch.from_numpy(D).cuda()
    ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    got = ctx.gint_rho(Dd).cpu().numpy()
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max(), name + " rho"
    Fr = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    assert_force_parity(ctx.gint_fvl(Vd, Dd).cpu().numpy(), Fr, name + " fvl")


def test_update_positions_on_device(cfg1):
    """Moving the atoms (velocity-Verlet step of Ehrenfest dynamics): after gint_update_positions all
    three calls match the oracle at the new geometry, and moving back reproduces the first H (to the rounding of the
    atomics' order)."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import gint_setup
    w = cfg1
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    Vd = torch.from_numpy(w.V).cuda()
    H0 = ctx.gint_vlocal(Vd).cpu().numpy()
    rng = np.random.default_rng(62)
    pos2 = w.atom_pos + rng.uniform(-0.5, 0.5, size=w.atom_pos.shape)
    ctx.gint_update_positions(pos2)
    Hr, blocks = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, pos2, w.V)
    assert np.array_equal(ctx.gint_get_blocks()[3], blocks[3])
    assert_parity(ctx.gint_vlocal(Vd).cpu().numpy(), Hr, "moved atoms")
    D = rng.normal(size=Hr.shape)
    Dd = torch.from_numpy(D).cuda()
    ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, pos2, D, blocks)
    assert np.abs(ctx.gint_rho(Dd).cpu().numpy() - ref).max() <= TOL * np.abs(ref).max()
    Fr = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, pos2, w.V, D, blocks)
    assert_force_parity(ctx.gint_fvl(Vd, Dd).cpu().numpy(), Fr, "moved atoms")
    ctx.gint_update_positions(w.atom_pos)
    assert np.abs(ctx.gint_vlocal(Vd).cpu().numpy() - H0).max() <= 1e-13 * np.abs(H0).max()


@pytest.mark.parametrize("name,limit", [("si8_sz", 1 << 16), ("si64_dzp", 48 << 20), ("cluster60", 8 << 20)])
def test_scratch_limit_batches(name, limit):
    """gint_options.scratch_max_bytes: when the psi scratch may not hold all regions, consecutive batches of regions
    reuse it (the psi kernel then zero-fills what it skips).  All three calls against the oracle with many batches,
    and the context really uses the small buffer."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    w = wl.make(name)
    Hr, blocks = oracle_H(w)
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, scratch_max_bytes=limit)
    st = ctx.gint_get_stats()
    full = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1).gint_get_stats()
    assert st["batches"] >= 4 and st["psi_scratch_bytes"] < full["psi_scratch_bytes"] / 3
    assert st["F_sym"] == full["F_sym"] and st["executed_flops"] == full["executed_flops"]
    Vd = torch.from_numpy(w.V).cuda()
    rng = np.random.default_rng(71)
    D = rng.normal(size=Hr.shape)
    Dd = torch.from_numpy(D).cuda()
    rho_ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    F_ref = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    for rep in range(2):   # second round: the scratch holds the last batch's values of the previous call
        assert_parity(ctx.gint_vlocal(Vd).cpu().numpy(), Hr, "%s batched, round %d" % (name, rep))
        got = ctx.gint_rho(Dd).cpu().numpy()
        assert np.abs(got - rho_ref).max() <= TOL * np.abs(rho_ref).max()
        assert_force_parity(ctx.gint_fvl(Vd, Dd).cpu().numpy(), F_ref, "%s batched" % name)


def test_large_tables_stay_in_global_memory():
    """Radial tables too large for shared memory (fine dr: 2 species x 4 padded functions x 3004 nodes = 192 KB > 56 KB)
    take the kernels' global-memory table path (psi and force kernels instantiated with TAB_SMEM = false): all three
    calls against the oracle on a triclinic cell with two species."""
    torch = _torch()
    import oracle
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    w = wl.tiny(seed=17, natom=4, ngrid=(11, 10, 12))
    fine = [wl.make_species("fine-a", 3.0, [(0, 0.6), (1, 0.5), (2, 0.7)], dr=0.001),
            wl.make_species("fine-b", 3.0, [(0, 0.9), (1, 0.8), (3, 0.6)], dr=0.001)]
    w.species = fine
    w.atom_species = np.array([0, 1, 0, 1], dtype=np.int32)
    Hr, blocks = oracle_H(w)
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos)
    Vd = torch.from_numpy(w.V).cuda()
    assert_parity(ctx.gint_vlocal(Vd).cpu().numpy(), Hr, "tables in global memory")
    rng = np.random.default_rng(81)
    D = rng.normal(size=Hr.shape)
    Dd = torch.from_numpy(D).cuda()
    ref = oracle.rho(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, D, blocks)
    assert np.abs(ctx.gint_rho(Dd).cpu().numpy() - ref).max() <= TOL * np.abs(ref).max()
    Fr = oracle.fvl(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V, D, blocks)
    assert_force_parity(ctx.gint_fvl(Vd, Dd).cpu().numpy(), Fr, "tables in global memory")
