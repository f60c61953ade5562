"""N > 1 path on CPU: two processes, `gloo` backend, rendezvous on 127.0.0.1.

bench.py shards the big cells over ranks (`gint_setup(..., rank, nranks)`), lets every rank integrate
its share into a partial H and sums the partial buffers with ONE all-reduce -- the path's only exchange
step.  Without a GPU the integration itself cannot run (there is no CPU fallback), so
this test covers everything around it: the shards partition the cell lists and the useful flops, every
rank holds the same H layout, and the float64 all-reduce over an h_len buffer sums the shards' partial
contributions exactly as the single-rank buffer would hold them.
"""
import os
import socket
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.make("si8_sz")
        full = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1)
        part = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1,
                          rank=rank, nranks=world)
        # same H layout on every rank
        bi, bj, bR, off = part.gint_get_blocks()
        layout = torch.from_numpy(np.concatenate([bi, bj, bR.ravel(), off]).astype(np.int64))
        ref = layout.clone()
        dist.broadcast(ref, src=0)
        assert torch.equal(layout, ref) and part.h_len == full.h_len
        # the shards partition the useful work
        st, sf = part.gint_get_stats(), full.gint_get_stats()
        t = torch.tensor([st["F_pt"], st["F_sym"], st["insphere_pairs"], st["entries"]], dtype=torch.float64)
        dist.all_reduce(t)
        assert t[0].item() == sf["F_pt"] and t[1].item() == sf["F_sym"]
        assert t[2].item() == sf["insphere_pairs"] and t[3].item() == sf["entries"]
        # every non-empty cell belongs to exactly one rank
        s_part = part.gint_get_cell_lists()[0]
        owned = torch.from_numpy((np.diff(s_part) > 0).astype(np.int64))
        dist.all_reduce(owned)
        assert np.array_equal(owned.numpy(), (np.diff(full.gint_get_cell_lists()[0]) > 0).astype(np.int64))
        # the exchange step: partial H buffers (here: each cell's contribution tagged by its owner) sum to the whole
        rng = np.random.default_rng(5)
        contrib = rng.normal(size=(len(owned), 8))                 # per cell, a fixed pseudo-contribution
        idx = rng.integers(0, part.h_len, size=(len(owned), 8))    # ... to fixed H elements
        mine = np.diff(s_part) > 0
        H = np.zeros(part.h_len)
        np.add.at(H, idx[mine].ravel(), contrib[mine].ravel())
        Ht = torch.from_numpy(H)
        dist.all_reduce(Ht)
        Hall = np.zeros(part.h_len)
        allc = np.diff(full.gint_get_cell_lists()[0]) > 0
        np.add.at(Hall, idx[allc].ravel(), contrib[allc].ravel())
        assert np.allclose(Ht.numpy(), Hall, rtol=0, atol=1e-12)
        open(os.path.join(out_dir, "ok%d" % rank), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert all(os.path.exists(os.path.join(str(tmp_path), "ok%d" % r)) for r in range(2))
