"""gint_fold_k_static: the entry point that allocates nothing (include/gint.h).  Its phase scratch is a fixed
`static __device__` array inside the library instead of memory the context allocated; everything else is gint_fold_k
(H(k) = sum_R exp(i k.R) H(R), Eq. 5).  Checked here against the existing path and the oracle, on
calls in a row that share the array.  This file is named to be collected last.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-13   # the fold tests' tolerance (tests/test_gpu_parity.py::test_fold_k_against_oracle)


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _context_with_H(w):
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=0)
    H = ctx.gint_vlocal(torch.from_numpy(np.ascontiguousarray(w.V)).cuda())
    torch.cuda.synchronize()
    return ctx, H


def test_fold_k_static_matches_existing_path_on_calls_in_a_row(cfg1):
    """Two contexts (cfg1 with its self-image blocks, and a smaller triclinic one whose blocks cover only the head of
    the shared array) called one after the other with different k: every call equals gint_fold_k and the oracle, so
    nothing survives from the call before; the output buffer starts as NaN, so every element is written."""
    torch = _torch()
    import oracle
    from helpers import norb_per_atom
    from paper_2603_21835_b200 import workloads as wl
    small = wl.tiny(seed=11, natom=4, ngrid=(9, 13, 7))
    cases = [(cfg1,) + _context_with_H(cfg1), (small,) + _context_with_H(small)]
    assert len(cases[1][1].gint_get_blocks()[0]) < len(cases[0][1].gint_get_blocks()[0])
    ks = [(0.31, -0.17, 0.43), (0.5, 0.25, -0.4), (0.0, 0.0, 0.0), (-0.23, 0.41, 0.09)]
    for rep, k in enumerate(ks):
        for w, ctx, H in (cases if rep % 2 == 0 else cases[::-1]):
            n = ctx.gint_num_orbitals()[0]
            out = torch.full((n, n), float("nan"), dtype=torch.complex128, device="cuda")
            ctx.gint_fold_k_static(H, k, out)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
            old = ctx.gint_fold_k(H, k).cpu().numpy()
            ref = oracle.fold_k(H.cpu().numpy(), ctx.gint_get_blocks(), norb_per_atom(w), k)
            scale = np.abs(ref).max()
            assert np.all(np.isfinite(got.real)) and np.all(np.isfinite(got.imag))
            assert np.abs(got - old).max() <= TOL * scale, "%s k=%s: differs from gint_fold_k" % (w.name, k)
            assert np.abs(got - ref).max() <= TOL * scale, "%s k=%s: differs from the oracle" % (w.name, k)


def test_fold_k_static_back_to_back_without_sync_and_without_allocation(cfg1):
    """Calls queued back to back on one stream (the second one's phase kernel overwrites the array only after the
    first one's fold kernel has read it: stream order), device memory in use unchanged by the calls."""
    torch = _torch()
    ctx, H = _context_with_H(cfg1)
    n = ctx.gint_num_orbitals()[0]
    ks = [(0.31, -0.17, 0.43), (0.5, 0.25, -0.4), (0.11, 0.0, -0.37)]
    want = [ctx.gint_fold_k(H, k).clone() for k in ks]
    outs = [torch.empty((n, n), dtype=torch.complex128, device="cuda") for _ in ks]
    ctx.gint_fold_k_static(H, ks[0], outs[0])          # kernels loaded before the memory reading below
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        for k, o in zip(ks, outs):
            ctx.gint_fold_k_static(H, k, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    for k, o, w_ in zip(ks, outs, want):
        assert float((o - w_).abs().max()) <= TOL * float(w_.abs().max()), "k=%s" % (k,)


def test_fold_k_static_rejects_more_blocks_than_the_array_holds():
    """A lattice gas of 4096 one-orbital atoms with 81 neighbours each: 331 776 blocks > the 262 144 the fixed array
    holds.  The static entry point refuses with GINT_EUNSUPPORTED and launches nothing; gint_fold_k still works."""
    torch = _torch()
    from paper_2603_21835_b200 import gint_setup, workloads as wl
    from paper_2603_21835_b200.binding import GintError, gint_fold_k_static_max_blocks
    nmax = gint_fold_k_static_max_blocks()
    assert nmax == 1 << 18
    n, a = 16, 4.0
    sp = wl.make_species("gas", 5.0, [(0, 0.8)])
    g = np.arange(n) * a
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) + 0.37
    ctx = gint_setup(np.eye(3) * n * a, (64, 64, 64), [sp], np.zeros(len(pos), np.int32), pos, cuda_device=0)
    nblk = len(ctx.gint_get_blocks()[0])
    assert nblk > nmax
    H = torch.ones(ctx.h_len, dtype=torch.float64, device="cuda")
    out = torch.full((len(pos), len(pos)), 7.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(GintError) as ei:
        ctx.gint_fold_k_static(H, (0.1, 0.2, 0.3), out)
    assert ei.value.code == -2 and str(nmax) in str(ei.value) and str(nblk) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                     # untouched
    Hk = ctx.gint_fold_k(H, (0.0, 0.0, 0.0))            # the allocating path takes any size
    torch.cuda.synchronize()
    assert abs(float(Hk.real.sum()) - nblk) <= 1e-9 * nblk
