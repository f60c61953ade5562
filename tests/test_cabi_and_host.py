"""CPU-side tests: the C-ABI library loads and exports every symbol of include/gint.h;
host logic of gint_setup (block table, big-cell lists, error codes) checked without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2603_21835_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_2603_21835_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "gint.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(gint_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTED), declared ^ set(binding.EXPORTED)
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in declared:
        assert getattr(lib, name) is not None


def test_product_does_not_import_oracle():
    """The product path shares no code with the oracle and never calls it."""
    pkg = os.path.join(ROOT, "paper_2603_21835_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".hpp", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "gint_oracle" not in txt and "libgint_oracle" not in txt and "oracle/" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2603_21835_b200 import" not in txt and "libgint_b200" not in txt, f


@pytest.fixture(scope="module")
def host_ctx_cfg1(cfg1):
    from paper_2603_21835_b200 import gint_setup
    w = cfg1
    return gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1)


def test_block_table_matches_oracle_enumeration(cfg1, host_ctx_cfg1):
    import oracle
    bi, bj, bR, off = oracle.enumerate_blocks(cfg1.lattice, cfg1.species, cfg1.atom_species, cfg1.atom_pos)
    i2, j2, R2, o2 = host_ctx_cfg1.gint_get_blocks()
    assert np.array_equal(bi, i2) and np.array_equal(bj, j2) and np.array_equal(bR, R2) and np.array_equal(off, o2)
    assert host_ctx_cfg1.nblocks == 376 and host_ctx_cfg1.h_len == 6016


def test_host_only_context_refuses_device_calls(cfg1, host_ctx_cfg1):
    from paper_2603_21835_b200 import binding
    with pytest.raises(binding.GintError) as e:
        host_ctx_cfg1.gint_vlocal_host(cfg1.V)
    assert e.value.code == binding.GINT_ENODEVICE


def brute_cell_lists(w, bcell):
    """Independent (numpy) construction of the per-cell (atom, image) lists: an image is
    listed iff one of the cell's mesh points lies strictly inside its cutoff sphere."""
    n = np.array(w.ngrid)
    nc = -(-n // np.array(bcell))
    idx = np.stack(np.meshgrid(*[np.arange(x) for x in n], indexing="ij"), axis=-1).reshape(-1, 3)
    pts = (idx / n) @ w.lattice
    cell = ((idx[:, 0] // bcell[0]) * nc[1] + idx[:, 1] // bcell[1]) * nc[2] + idx[:, 2] // bcell[2]
    out = set()
    counts = np.zeros(len(idx), dtype=np.int64)
    for I in range(w.natom):
        sp = w.species[w.atom_species[I]]
        for a in range(-3, 4):
            for b in range(-3, 4):
                for c in range(-3, 4):
                    d = pts - w.atom_pos[I] - np.array([a, b, c]) @ w.lattice
                    inside = np.einsum("ij,ij->i", d, d) < sp.rcut ** 2
                    counts += inside * sp.norb
                    for cc in np.unique(cell[inside]):
                        out.add((int(cc), I, a, b, c))
    return out, counts


@pytest.mark.parametrize("bcell", [(4, 4, 4), (3, 2, 4)])
def test_cell_lists_exact_and_sorted(bcell):
    from paper_2603_21835_b200 import gint_setup
    w = wl.tiny(seed=7)
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1, bcell=bcell)
    start, atom, R = ctx.gint_get_cell_lists()
    got = set()
    for c in range(len(start) - 1):
        keys = [(int(atom[i]), int(R[i, 0]), int(R[i, 1]), int(R[i, 2])) for i in range(start[c], start[c + 1])]
        assert keys == sorted(keys)             # canonical order inside a cell
        got |= {(c,) + k for k in keys}
    want, counts = brute_cell_lists(w, bcell)
    assert got == want
    st = ctx.gint_get_stats()
    assert st["F_pt"] == pytest.approx(float(np.sum(2.0 * counts * counts)), rel=1e-14)
    assert st["F_sym"] == pytest.approx(float(np.sum(counts * (counts + 1.0))), rel=1e-14)
    assert st["entries"] == len(want)


def test_survey_sizes_cfg1_cfg2(cfg1, host_ctx_cfg1):
    """cfg1 F_pt = 6.95e7, F_sym = 3.60e7, in-sphere pairs 3.12e5."""
    st = host_ctx_cfg1.gint_get_stats()
    assert st["F_pt"] == pytest.approx(6.95e7, rel=5e-3)
    assert st["F_sym"] == pytest.approx(3.60e7, rel=5e-3)
    assert st["insphere_pairs"] == pytest.approx(3.12e5, rel=5e-3)


def test_rank_sharding_partitions_the_cells():
    from paper_2603_21835_b200 import gint_setup
    w = wl.tiny(seed=7)
    full = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1)
    sf, af, Rf = full.gint_get_cell_lists()
    tot = 0
    seen = np.zeros(len(sf) - 1, dtype=int)
    for r in range(3):
        part = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1, rank=r, nranks=3)
        s, a, R = part.gint_get_cell_lists()
        tot += len(a)
        seen += (np.diff(s) > 0)
        assert part.nblocks == full.nblocks      # same H layout on every rank
    assert tot == len(af) and np.all(seen == (np.diff(sf) > 0))
    assert full.gint_get_stats()["F_pt"] == pytest.approx(sum(
        gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1, rank=r, nranks=3)
        .gint_get_stats()["F_pt"] for r in range(3)))


def test_error_codes():
    from paper_2603_21835_b200 import binding, gint_setup
    w = wl.tiny(seed=7)

    def setup(**kw):
        a = dict(lattice=w.lattice, ngrid=w.ngrid, species=w.species, atom_species=w.atom_species,
                 atom_pos=w.atom_pos, cuda_device=-1)
        a.update(kw)
        return gint_setup(**a)
    with pytest.raises(binding.GintError) as e:
        setup(lattice=np.array([[1.0, 0, 0], [2.0, 0, 0], [0, 0, 1.0]]))
    assert e.value.code == binding.GINT_EINVAL
    with pytest.raises(binding.GintError) as e:
        setup(ngrid=[4, 0, 4])
    assert e.value.code == binding.GINT_EINVAL
    with pytest.raises(binding.GintError) as e:
        setup(atom_species=np.array([0, 5, 0]))
    assert e.value.code == binding.GINT_EINVAL
    sp = w.species[0]
    short = wl.Species("short", sp.rcut, sp.dr, sp.l, sp.table[:, : int(sp.rcut / sp.dr) + 1].copy())
    with pytest.raises(binding.GintError) as e:
        setup(species=[short])
    assert e.value.code == binding.GINT_EINVAL
    g_shell = wl.Species("g", sp.rcut, sp.dr, np.array([4], dtype=np.int32), sp.table[:1].copy())
    with pytest.raises(binding.GintError) as e:
        setup(species=[g_shell])
    assert e.value.code == binding.GINT_EUNSUPPORTED
    with pytest.raises(binding.GintError) as e:
        setup(bcell=(16, 8, 8))
    assert e.value.code == binding.GINT_EUNSUPPORTED
    pos = w.atom_pos.copy()
    pos[0, 0] = np.nan
    with pytest.raises(binding.GintError) as e:
        setup(atom_pos=pos)
    assert e.value.code == binding.GINT_EINVAL
    assert binding._strerror(binding.GINT_ECUDA) == "CUDA error"


def test_bench_flop_count_matches_the_plan(cfg1):
    """bench.py counts the useful flops itself (k-d tree over atom images) so that its oracle arm needs no product
    library; the count equals the plan's own statistics on a cubic cell with self-images, a triclinic cell and the
    two-species cluster."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    from paper_2603_21835_b200 import gint_setup
    for w in (cfg1, wl.tiny(seed=7), wl.tiny(seed=11, ngrid=(9, 13, 7)), wl.make("cluster60")):
        st = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1).gint_get_stats()
        fpt, fsym = bench.useful_flops(w)
        assert fpt == st["F_pt"] and fsym == st["F_sym"], w.name


def test_reference_arm_runs_without_the_product_library(tmp_path):
    """`bench.py --impl reference` must load oracle/ only: run it with the product .so masked (an import hook that
    fails on the binding) and check the JSON line."""
    import json
    import subprocess
    import sys
    hook = tmp_path / "sitecustomize.py"
    hook.write_text(
        "import sys, importlib.abc\n"
        "class _Block(importlib.abc.MetaPathFinder):\n"
        "    def find_spec(self, name, path, target=None):\n"
        "        if name == 'paper_2603_21835_b200.binding':\n"
        "            raise ImportError('product library masked for this test')\n"
        "sys.meta_path.insert(0, _Block())\n")
    env = dict(os.environ, PYTHONPATH=str(tmp_path) + os.pathsep + os.environ.get("PYTHONPATH", ""))
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "si8_sz",
                          "--steps", "1", "--warmup", "0", "--ref-atoms", "2"], env=env, capture_output=True, text=True,
                         timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0


def test_update_positions_equals_fresh_setup(cfg1):
    """gint_update_positions (moving nuclei): a host-only context moved to new
    positions holds the same block table, cell lists and plan statistics as a context set up there, whatever the
    number of setup threads; a bad position leaves the context unchanged."""
    import os
    from paper_2603_21835_b200 import gint_setup
    rng = np.random.default_rng(61)
    pos2 = cfg1.atom_pos + rng.uniform(-0.6, 0.6, size=cfg1.atom_pos.shape)
    ctx = gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cuda_device=-1)
    nb0 = ctx.nblocks
    ctx.gint_update_positions(pos2)
    os.environ["GINT_SETUP_THREADS"] = "1"
    try:
        ref = gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, pos2, cuda_device=-1)
    finally:
        del os.environ["GINT_SETUP_THREADS"]
    assert ctx.nblocks == ref.nblocks and ctx.h_len == ref.h_len and ctx.nblocks != nb0
    for a, b in zip(ctx.gint_get_blocks(), ref.gint_get_blocks()):
        assert np.array_equal(a, b)
    for a, b in zip(ctx.gint_get_cell_lists(), ref.gint_get_cell_lists()):
        assert np.array_equal(a, b)
    assert ctx.gint_get_stats() == ref.gint_get_stats()
    bad = pos2.copy()
    bad[0, 0] = np.nan
    with pytest.raises(Exception):
        ctx.gint_update_positions(bad)
    assert ctx.gint_get_stats() == ref.gint_get_stats()


def test_scratch_limit_makes_batches(cfg1):
    """scratch_max_bytes (host logic): the plan cuts the regions into batches that fit, keeps work and block table, and
    never goes below what the largest region needs."""
    from paper_2603_21835_b200 import gint_setup
    full = gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cuda_device=-1)
    s0 = full.gint_get_stats()
    assert s0["batches"] == 1
    for limit in (1, 1 << 16, 1 << 18):
        ctx = gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cuda_device=-1,
                         scratch_max_bytes=limit)
        s = ctx.gint_get_stats()
        assert s["batches"] > 1 and s["psi_scratch_bytes"] < s0["psi_scratch_bytes"]
        assert s["psi_scratch_bytes"] <= max(limit, 8192 * 40 * 16)       # one region at most: 40 groups x 16 stages
        assert s["F_sym"] == s0["F_sym"] and s["executed_flops"] == s0["executed_flops"] and ctx.nblocks == full.nblocks
    with pytest.raises(Exception):
        gint_setup(cfg1.lattice, cfg1.ngrid, cfg1.species, cfg1.atom_species, cfg1.atom_pos, cuda_device=-1, scratch_max_bytes=-5)


def test_bench_helpers_run_without_a_gpu():
    """bench.py's host-side helpers: the peaks file (or its fallback) and the ncu traffic record under profiles/."""
    import importlib.util
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    peaks, src = bench.measured_peaks()
    assert peaks["hbm_gbs"] > 1000 and peaks["bf16_tflops"] > 100 and src in ("measured", "fallback")
    t = bench.ncu_traffic("si512_dzp")
    assert t is not None and 1e9 < t < 1e11
    assert bench.ncu_traffic("no_such_workload") is None


def test_snap_pair_list_equals_the_oracles_enumeration():
    """gint_snap_setup on host-only contexts: the (I, J, R) list and the block offsets of Eq. 47
    against oracle.enumerate_snap_pairs -- cubic cfg1 with image pairs, a triclinic cell with a species that has no
    projectors, and a self image exactly at the cutoff (strict inequality)."""
    import oracle
    from paper_2603_21835_b200 import gint_setup
    from paper_2603_21835_b200.binding import GintError
    rx, rw = wl.radial_quadrature(8)
    an, aw = wl.angular_quadrature(6)
    none = wl.Species(name="none", rcut=0.0, dr=0.01, l=np.zeros(0, np.int32), table=np.zeros((0, 8)))
    w1 = wl.make("si8_sz")
    w2 = wl.tiny(seed=9, natom=5, ngrid=(12, 12, 12), rcut=3.0)
    sp2 = [wl.make_species("A", 3.0, [(0, 0.6), (1, 0.5)]), wl.make_species("B", 2.4, [(0, 0.9)])]
    asp2 = np.array([0, 1, 0, 1, 0], dtype=np.int32)
    cases = [(w1.lattice, w1.ngrid, w1.species, w1.atom_species, w1.atom_pos, [wl.projector_species()]),
             (w2.lattice, w2.ngrid, sp2, asp2, w2.atom_pos, [wl.make_species("beta", 2.0, [(0, 1.5), (1, 1.8)]), none]),
             (np.diag([5.0, 9.0, 9.0]), (10, 18, 18), [wl.make_species("A", 3.0, [(0, 0.6)])], np.zeros(1, np.int32),
              np.array([[0.123456789, 1.1, 2.2]]), [wl.make_species("beta", 2.0, [(0, 1.5)])])]
    for lat, ng, species, asp, pos, proj in cases:
        ctx = gint_setup(lat, ng, species, asp, pos, cuda_device=-1)
        with pytest.raises(GintError):
            ctx.gint_snap_get_pairs()                       # not set up yet
        ctx.gint_snap_setup(proj, rx, rw, an, aw)
        got = ctx.gint_snap_get_pairs()
        ref = oracle.enumerate_snap_pairs(lat, species, proj, asp, pos)
        assert all(np.array_equal(a, b) for a, b in zip(got, ref))
        assert len(got[0]) > 0
    assert [tuple(r) for r in got[2].tolist()] == [(0, 0, 0)]   # the tie case: no (+-1, 0, 0) self image


def test_snap_pairs_are_dealt_out_by_projector_atom():
    """nranks = 3: the ranks' pair lists are disjoint, cover the full list, and rank r holds exactly the pairs of the
    atoms I with I % 3 == r (host-only contexts)."""
    from paper_2603_21835_b200 import gint_setup
    w = wl.make("si8_sz")
    proj = [wl.projector_species()]
    rx, rw = wl.radial_quadrature(8)
    an, aw = wl.angular_quadrature(6)
    def pairs(rank, nranks):
        ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1, rank=rank, nranks=nranks)
        ctx.gint_snap_setup(proj, rx, rw, an, aw)
        iat, jat, R, off = ctx.gint_snap_get_pairs()
        assert off[0] == 0 and np.all(np.diff(off) > 0)
        return [tuple(x) for x in np.column_stack([iat, jat, R]).tolist()]
    full = pairs(0, 1)
    parts = [pairs(r, 3) for r in range(3)]
    for r, p in enumerate(parts):
        assert p and all(k[0] % 3 == r for k in p)
    assert sorted(sum(parts, [])) == full
