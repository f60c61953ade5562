"""ctypes binding of libgint_b200.so -- argument marshalling only.

Function names follow include/gint.h.  Every step of the hot path runs inside the
library's CUDA kernels; PyTorch is used for device buffers and the stream handle.
There is no CPU fallback: if the shared library is missing, importing this module
raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgint_b200.so")

GINT_OK, GINT_EINVAL, GINT_EUNSUPPORTED, GINT_ENOMEM, GINT_ECUDA, GINT_ENODEVICE = 0, -1, -2, -3, -4, -5

EXPORTED = ("gint_setup", "gint_update_positions", "gint_num_blocks", "gint_get_blocks", "gint_vlocal", "gint_vlocal_host", "gint_get_stats",
            "gint_set_profiling", "gint_get_kernel_ms", "gint_num_orbitals", "gint_fold_k", "gint_fold_k_static", "gint_fold_k_static_max_blocks", "gint_snap_setup", "gint_snap_num_pairs", "gint_snap_get_pairs", "gint_snap_psibeta", "gint_rho", "gint_fvl", "gint_get_cell_lists", "gint_measure_fp64_peak", "gint_destroy", "gint_strerror", "gint_last_error")

STAT_NAMES = ("cells", "items", "entries", "max_rows", "executed_flops", "flush_elems", "smem_bytes", "kernels_per_call",
              "F_pt", "F_sym", "insphere_pairs", "evaluated_pairs", "psi_scratch_bytes", "psi_load_bytes", "ring_stages",
              "regions", "ksteps_full", "ksteps_partial", "dmma_in_partial_ksteps", "stage_visits", "dmma_max_sched_item", "dmma_max_sched_stage", "dmma_max_warp_stage", "bcell1", "bcell2", "bcell3",
              "dmma_diag_runs", "dmma_rect_runs", "dmma_other_runs", "runs", "batches", "s31")


class GintError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str):
        super().__init__("%s failed: %s (%d) %s" % (where, _strerror(code), code, detail))
        self.code = code


class _Species(ctypes.Structure):
    _fields_ = [("rcut", ctypes.c_double), ("dr", ctypes.c_double), ("ntab", ctypes.c_int32), ("nrad", ctypes.c_int32),
                ("l", ctypes.POINTER(ctypes.c_int32)), ("table", ctypes.POINTER(ctypes.c_double))]


class _Options(ctypes.Structure):
    _fields_ = [("bcell", ctypes.c_int32 * 3), ("rank", ctypes.c_int32), ("nranks", ctypes.c_int32),
                ("pad", ctypes.c_int32), ("scratch_max_bytes", ctypes.c_int64)]


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError("libgint_b200.so not built: run `python -m paper_2603_21835_b200.build` "
                          "(there is no CPU fallback for the gint_vlocal hot path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    P = ctypes.POINTER
    lib.gint_setup.restype = ctypes.c_int
    lib.gint_setup.argtypes = [P(vp), P(dbl), P(i32), i32, P(_Species), i32, P(i32), P(dbl), i32, P(_Options)]
    lib.gint_update_positions.restype = ctypes.c_int
    lib.gint_update_positions.argtypes = [vp, P(dbl)]
    lib.gint_num_blocks.restype = ctypes.c_int
    lib.gint_num_blocks.argtypes = [vp, P(i64), P(i64)]
    lib.gint_get_blocks.restype = ctypes.c_int
    lib.gint_get_blocks.argtypes = [vp, P(i32), P(i32), P(i32), P(i64)]
    lib.gint_vlocal.restype = ctypes.c_int
    lib.gint_vlocal.argtypes = [vp, vp, vp, vp]
    lib.gint_vlocal_host.restype = ctypes.c_int
    lib.gint_vlocal_host.argtypes = [vp, P(dbl), P(dbl)]
    lib.gint_num_orbitals.restype = ctypes.c_int
    lib.gint_num_orbitals.argtypes = [vp, P(i64), P(i64)]
    lib.gint_fold_k.restype = ctypes.c_int
    lib.gint_fold_k.argtypes = [vp, vp, P(dbl), vp, vp]
    lib.gint_fold_k_static.restype = ctypes.c_int
    lib.gint_fold_k_static.argtypes = [vp, vp, P(dbl), vp, vp]
    lib.gint_fold_k_static_max_blocks.restype = ctypes.c_int64
    lib.gint_fold_k_static_max_blocks.argtypes = []
    lib.gint_snap_setup.restype = ctypes.c_int
    lib.gint_snap_setup.argtypes = [vp, P(_Species), i32, P(dbl), P(dbl), i32, P(dbl), P(dbl)]
    lib.gint_snap_num_pairs.restype = ctypes.c_int
    lib.gint_snap_num_pairs.argtypes = [vp, P(i64), P(i64)]
    lib.gint_snap_get_pairs.restype = ctypes.c_int
    lib.gint_snap_get_pairs.argtypes = [vp, P(i32), P(i32), P(i32), P(i64)]
    lib.gint_snap_psibeta.restype = ctypes.c_int
    lib.gint_snap_psibeta.argtypes = [vp, P(dbl), vp, vp]
    lib.gint_rho.restype = ctypes.c_int
    lib.gint_rho.argtypes = [vp, vp, vp, vp]
    lib.gint_fvl.restype = ctypes.c_int
    lib.gint_fvl.argtypes = [vp, vp, vp, vp, vp]
    lib.gint_get_stats.restype = ctypes.c_int
    lib.gint_get_stats.argtypes = [vp, P(dbl), i32]
    lib.gint_set_profiling.restype = ctypes.c_int
    lib.gint_set_profiling.argtypes = [vp, i32]
    lib.gint_get_kernel_ms.restype = ctypes.c_int
    lib.gint_get_kernel_ms.argtypes = [vp, P(dbl)]
    lib.gint_get_cell_lists.restype = ctypes.c_int
    lib.gint_get_cell_lists.argtypes = [vp, P(i64), P(i64), P(i64), P(i32), P(i32)]
    lib.gint_measure_fp64_peak.restype = ctypes.c_int
    lib.gint_measure_fp64_peak.argtypes = [i32, dbl, P(dbl)]
    lib.gint_destroy.restype = ctypes.c_int
    lib.gint_destroy.argtypes = [vp]
    lib.gint_strerror.restype = ctypes.c_char_p
    lib.gint_strerror.argtypes = [ctypes.c_int]
    lib.gint_last_error.restype = ctypes.c_char_p
    lib.gint_last_error.argtypes = []
    return lib


_lib = _load()


def _strerror(code: int) -> str:
    return _lib.gint_strerror(code).decode()


def _check(code: int, where: str):
    if code < 0:
        raise GintError(code, where, _lib.gint_last_error().decode())
    return code


def _ptr(a: np.ndarray, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


class GintContext:
    """Owner of a gint_ctx*.  Methods are the C calls of include/gint.h, same names."""

    def __init__(self, handle: int, ngrid, natom: int):
        self._h = ctypes.c_void_p(handle)
        self.natom = int(natom)
        self.ngrid = tuple(int(x) for x in ngrid)
        nb, hl = ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.gint_num_blocks(self._h, ctypes.byref(nb), ctypes.byref(hl)), "gint_num_blocks")
        self.nblocks, self.h_len = int(nb.value), int(hl.value)

    def gint_update_positions(self, atom_pos):
        """Rebuild the context for new atom positions [natom][3]; nblocks / h_len are refreshed (the block table may change)."""
        pos = np.ascontiguousarray(atom_pos, dtype=np.float64).reshape(-1, 3)
        if pos.shape[0] != self.natom:
            raise ValueError("atom_pos must be [natom][3]")
        _check(_lib.gint_update_positions(self._h, _ptr(pos, ctypes.c_double)), "gint_update_positions")
        nb, hl = ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.gint_num_blocks(self._h, ctypes.byref(nb), ctypes.byref(hl)), "gint_num_blocks")
        self.nblocks, self.h_len = int(nb.value), int(hl.value)

    # -- queries -----------------------------------------------------------------
    def gint_get_blocks(self):
        n = self.nblocks
        iat = np.empty(max(n, 1), dtype=np.int32)
        jat = np.empty(max(n, 1), dtype=np.int32)
        R = np.empty((max(n, 1), 3), dtype=np.int32)
        off = np.empty(n + 1, dtype=np.int64)
        _check(_lib.gint_get_blocks(self._h, _ptr(iat, ctypes.c_int32), _ptr(jat, ctypes.c_int32),
                                    _ptr(R, ctypes.c_int32), _ptr(off, ctypes.c_int64)), "gint_get_blocks")
        return iat[:n], jat[:n], R[:n], off

    def gint_get_stats(self) -> dict:
        s = np.zeros(32, dtype=np.float64)
        n = _check(_lib.gint_get_stats(self._h, _ptr(s, ctypes.c_double), 32), "gint_get_stats")
        return {STAT_NAMES[i]: float(s[i]) for i in range(n)}

    def gint_set_profiling(self, on: bool = True):
        _check(_lib.gint_set_profiling(self._h, 1 if on else 0), "gint_set_profiling")

    def gint_get_kernel_ms(self):
        """(contraction kernel ms, mirror kernel ms, whole call ms, psi kernel ms) of the last gint_vlocal call."""
        ms = np.zeros(4, dtype=np.float64)
        _check(_lib.gint_get_kernel_ms(self._h, _ptr(ms, ctypes.c_double)), "gint_get_kernel_ms")
        return float(ms[0]), float(ms[1]), float(ms[2]), float(ms[3])

    def gint_get_cell_lists(self):
        nc, ne = ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.gint_get_cell_lists(self._h, ctypes.byref(nc), ctypes.byref(ne), None, None, None),
               "gint_get_cell_lists")
        start = np.empty(nc.value + 1, dtype=np.int64)
        atom = np.empty(max(ne.value, 1), dtype=np.int32)
        R = np.empty((max(ne.value, 1), 3), dtype=np.int32)
        _check(_lib.gint_get_cell_lists(self._h, None, None, _ptr(start, ctypes.c_int64), _ptr(atom, ctypes.c_int32),
                                        _ptr(R, ctypes.c_int32)), "gint_get_cell_lists")
        return start, atom[:ne.value], R[:ne.value]

    # -- the hot path ----------------------------------------------------------------
    def gint_vlocal(self, V_dev, H_dev=None, stream=None):
        """V_dev: CUDA float64 tensor [N1][N2][N3]; H_dev: CUDA float64 tensor [h_len] (allocated if None).
        Asynchronous on `stream` (default: torch's current stream)."""
        import torch
        if not (V_dev.is_cuda and V_dev.dtype == torch.float64 and V_dev.is_contiguous()):
            raise ValueError("V_dev must be a contiguous CUDA float64 tensor")
        if tuple(V_dev.shape) != self.ngrid:
            raise ValueError("V_dev shape %s != mesh %s" % (tuple(V_dev.shape), self.ngrid))
        if H_dev is None:
            H_dev = torch.empty(self.h_len, dtype=torch.float64, device=V_dev.device)
        if not (H_dev.is_cuda and H_dev.dtype == torch.float64 and H_dev.is_contiguous() and H_dev.numel() == self.h_len):
            raise ValueError("H_dev must be a contiguous CUDA float64 tensor of h_len elements")
        s = torch.cuda.current_stream(V_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_vlocal(self._h, ctypes.c_void_p(V_dev.data_ptr()), ctypes.c_void_p(H_dev.data_ptr()),
                                ctypes.c_void_p(s)), "gint_vlocal")
        return H_dev

    def gint_rho(self, D_dev, rho_dev=None, stream=None):
        """rho(r_g) of Eq. 44 from density-matrix blocks D_dev (H layout); returns a CUDA float64 tensor [N1][N2][N3]."""
        import torch
        if not (D_dev.is_cuda and D_dev.dtype == torch.float64 and D_dev.is_contiguous() and D_dev.numel() == self.h_len):
            raise ValueError("D_dev must be a contiguous CUDA float64 tensor of h_len elements")
        if rho_dev is None:
            rho_dev = torch.empty(self.ngrid, dtype=torch.float64, device=D_dev.device)
        if not (rho_dev.is_cuda and rho_dev.dtype == torch.float64 and rho_dev.is_contiguous() and tuple(rho_dev.shape) == self.ngrid):
            raise ValueError("rho_dev must be a contiguous CUDA float64 tensor [N1][N2][N3]")
        s = torch.cuda.current_stream(D_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_rho(self._h, ctypes.c_void_p(D_dev.data_ptr()), ctypes.c_void_p(rho_dev.data_ptr()),
                             ctypes.c_void_p(s)), "gint_rho")
        return rho_dev

    def gint_fvl(self, V_dev, D_dev, F_dev=None, stream=None):
        """Local Pulay force of Eq. 46 from V and density-matrix blocks D_dev (H layout); returns a CUDA float64 tensor [natom][3]."""
        import torch
        if not (V_dev.is_cuda and V_dev.dtype == torch.float64 and V_dev.is_contiguous() and tuple(V_dev.shape) == self.ngrid):
            raise ValueError("V_dev must be a contiguous CUDA float64 tensor [N1][N2][N3]")
        if not (D_dev.is_cuda and D_dev.dtype == torch.float64 and D_dev.is_contiguous() and D_dev.numel() == self.h_len):
            raise ValueError("D_dev must be a contiguous CUDA float64 tensor of h_len elements")
        if F_dev is None:
            F_dev = torch.empty((self.natom, 3), dtype=torch.float64, device=V_dev.device)
        if not (F_dev.is_cuda and F_dev.dtype == torch.float64 and F_dev.is_contiguous() and tuple(F_dev.shape) == (self.natom, 3)):
            raise ValueError("F_dev must be a contiguous CUDA float64 tensor [natom][3]")
        s = torch.cuda.current_stream(V_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_fvl(self._h, ctypes.c_void_p(V_dev.data_ptr()), ctypes.c_void_p(D_dev.data_ptr()),
                             ctypes.c_void_p(F_dev.data_ptr()), ctypes.c_void_p(s)), "gint_fvl")
        return F_dev

    def gint_num_orbitals(self):
        """(norb_tot, first[natom+1]) of the dense k-space matrix."""
        n = ctypes.c_int64()
        first = np.zeros(self.natom + 1, dtype=np.int64)
        _check(_lib.gint_num_orbitals(self._h, ctypes.byref(n), _ptr(first, ctypes.c_int64)), "gint_num_orbitals")
        return int(n.value), first

    def gint_fold_k(self, H_dev, kfrac, Hk_dev=None, stream=None):
        """H(k) = sum_R exp(i k.R) H(R) (Eq. 5); returns a CUDA complex128 tensor [norb_tot][norb_tot]."""
        import torch
        n = self.gint_num_orbitals()[0]
        if not (H_dev.is_cuda and H_dev.dtype == torch.float64 and H_dev.is_contiguous() and H_dev.numel() == self.h_len):
            raise ValueError("H_dev must be a contiguous CUDA float64 tensor of h_len elements")
        if Hk_dev is None:
            Hk_dev = torch.empty((n, n), dtype=torch.complex128, device=H_dev.device)
        if not (Hk_dev.is_cuda and Hk_dev.dtype == torch.complex128 and Hk_dev.is_contiguous() and tuple(Hk_dev.shape) == (n, n)):
            raise ValueError("Hk_dev must be a contiguous CUDA complex128 tensor [norb_tot][norb_tot]")
        k = np.ascontiguousarray(kfrac, dtype=np.float64).reshape(3)
        s = torch.cuda.current_stream(H_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_fold_k(self._h, ctypes.c_void_p(H_dev.data_ptr()), _ptr(k, ctypes.c_double),
                                ctypes.c_void_p(Hk_dev.data_ptr()), ctypes.c_void_p(s)), "gint_fold_k")
        return Hk_dev

    def gint_fold_k_static(self, H_dev, kfrac, Hk_dev, stream=None):
        """gint_fold_k with the phase scratch in the library's fixed device array (no allocation: the caller passes
        Hk_dev); GintError(GINT_EUNSUPPORTED) beyond gint_fold_k_static_max_blocks() blocks."""
        import torch
        n = self.gint_num_orbitals()[0]
        if not (H_dev.is_cuda and H_dev.dtype == torch.float64 and H_dev.is_contiguous() and H_dev.numel() == self.h_len):
            raise ValueError("H_dev must be a contiguous CUDA float64 tensor of h_len elements")
        if not (Hk_dev.is_cuda and Hk_dev.dtype == torch.complex128 and Hk_dev.is_contiguous() and tuple(Hk_dev.shape) == (n, n)):
            raise ValueError("Hk_dev must be a contiguous CUDA complex128 tensor [norb_tot][norb_tot]")
        k = np.ascontiguousarray(kfrac, dtype=np.float64).reshape(3)
        s = torch.cuda.current_stream(H_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_fold_k_static(self._h, ctypes.c_void_p(H_dev.data_ptr()), _ptr(k, ctypes.c_double),
                                       ctypes.c_void_p(Hk_dev.data_ptr()), ctypes.c_void_p(s)), "gint_fold_k_static")
        return Hk_dev

    def gint_snap_setup(self, proj: Sequence, rad_x, rad_w, ang_xyz, ang_w):
        """Projector tables (objects like the species; nrad = 0 allowed) and the quadrature tables of gint_snap_psibeta."""
        arr, keep = _species_array(proj)
        rx = np.ascontiguousarray(rad_x, dtype=np.float64).reshape(-1)
        rw = np.ascontiguousarray(rad_w, dtype=np.float64).reshape(-1)
        an = np.ascontiguousarray(ang_xyz, dtype=np.float64).reshape(-1, 3)
        aw = np.ascontiguousarray(ang_w, dtype=np.float64).reshape(-1)
        if rx.shape != rw.shape or an.shape[0] != aw.shape[0]:
            raise ValueError("quadrature nodes and weights disagree in length")
        _check(_lib.gint_snap_setup(self._h, arr, int(rx.shape[0]), _ptr(rx, ctypes.c_double), _ptr(rw, ctypes.c_double),
                                    int(aw.shape[0]), _ptr(an, ctypes.c_double), _ptr(aw, ctypes.c_double)), "gint_snap_setup")
        del keep

    def gint_snap_get_pairs(self):
        """(iat[n], jat[n], R[n][3], offset[n+1]) of the (I, J, R) pairs; offsets in complex elements."""
        n, slen = ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.gint_snap_num_pairs(self._h, ctypes.byref(n), ctypes.byref(slen)), "gint_snap_num_pairs")
        n = int(n.value)
        iat = np.zeros(n, dtype=np.int32); jat = np.zeros(n, dtype=np.int32)
        R = np.zeros((n, 3), dtype=np.int32); off = np.zeros(n + 1, dtype=np.int64)
        _check(_lib.gint_snap_get_pairs(self._h, _ptr(iat, ctypes.c_int32), _ptr(jat, ctypes.c_int32), _ptr(R, ctypes.c_int32),
                                        _ptr(off, ctypes.c_int64)), "gint_snap_get_pairs")
        return iat, jat, R, off

    def gint_snap_psibeta(self, A, S_dev=None, stream=None):
        """S = <phi| exp(-i A.r) |beta> of every pair (Eq. 47); returns a CUDA complex128 tensor of s_len elements."""
        import torch
        slen = ctypes.c_int64()
        _check(_lib.gint_snap_num_pairs(self._h, None, ctypes.byref(slen)), "gint_snap_num_pairs")
        if S_dev is None:
            S_dev = torch.empty(int(slen.value), dtype=torch.complex128, device="cuda")
        if not (S_dev.is_cuda and S_dev.dtype == torch.complex128 and S_dev.is_contiguous() and S_dev.numel() == int(slen.value)):
            raise ValueError("S_dev must be a contiguous CUDA complex128 tensor of s_len elements")
        a = np.ascontiguousarray(A, dtype=np.float64).reshape(3)
        s = torch.cuda.current_stream(S_dev.device).cuda_stream if stream is None else int(stream)
        _check(_lib.gint_snap_psibeta(self._h, _ptr(a, ctypes.c_double), ctypes.c_void_p(S_dev.data_ptr()), ctypes.c_void_p(s)),
               "gint_snap_psibeta")
        return S_dev

    def gint_vlocal_host(self, V_host: np.ndarray, H_host: Optional[np.ndarray] = None) -> np.ndarray:
        """End-to-end call with HOST buffers (H2D of V, kernels, D2H of H, synchronise)."""
        V_host = np.ascontiguousarray(V_host, dtype=np.float64)
        if tuple(V_host.shape) != self.ngrid:
            raise ValueError("V_host shape mismatch")
        if H_host is None:
            H_host = np.empty(self.h_len, dtype=np.float64)
        _check(_lib.gint_vlocal_host(self._h, _ptr(V_host, ctypes.c_double), _ptr(H_host, ctypes.c_double)),
               "gint_vlocal_host")
        return H_host

    def gint_destroy(self):
        if self._h is not None and self._h.value:
            _lib.gint_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.gint_destroy()
        except Exception:
            pass


def _species_array(species: Sequence):
    """ctypes array of gint_species for objects with .rcut .dr .l[nrad] .table[nrad][ntab] (+ the arrays to keep alive)."""
    keep = []
    arr = (_Species * len(species))()
    for i, s in enumerate(species):
        l = np.ascontiguousarray(s.l, dtype=np.int32)
        tab = np.ascontiguousarray(s.table, dtype=np.float64)
        if tab.ndim != 2 or tab.shape[0] != l.shape[0]:
            raise ValueError("species table must be [nrad][ntab]")
        keep += [l, tab]
        arr[i].rcut, arr[i].dr = float(s.rcut), float(s.dr)
        arr[i].ntab, arr[i].nrad = int(tab.shape[1]), int(l.shape[0])
        arr[i].l, arr[i].table = _ptr(l, ctypes.c_int32), _ptr(tab, ctypes.c_double)
    return arr, keep


def gint_setup(lattice, ngrid, species: Sequence, atom_species, atom_pos, cuda_device: int = 0,
               bcell=(0, 0, 0), rank: int = 0, nranks: int = 1, scratch_max_bytes: int = 0) -> GintContext:
    """species: objects with .rcut .dr .l[nrad] .table[nrad][ntab].  cuda_device < 0: host-only context."""
    lattice = np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
    ng = np.ascontiguousarray(ngrid, dtype=np.int32).reshape(3)
    pos = np.ascontiguousarray(atom_pos, dtype=np.float64).reshape(-1, 3)
    asp = np.ascontiguousarray(atom_species, dtype=np.int32).reshape(-1)
    if asp.shape[0] != pos.shape[0]:
        raise ValueError("atom_species and atom_pos disagree on natom")
    arr, keep = _species_array(species)
    opt = _Options()
    for d in range(3):
        opt.bcell[d] = int(bcell[d])
    opt.rank, opt.nranks = int(rank), int(nranks)
    opt.scratch_max_bytes = int(scratch_max_bytes)
    h = ctypes.c_void_p()
    _check(_lib.gint_setup(ctypes.byref(h), _ptr(lattice, ctypes.c_double), _ptr(ng, ctypes.c_int32), len(species),
                           arr, int(pos.shape[0]), _ptr(asp, ctypes.c_int32), _ptr(pos, ctypes.c_double),
                           int(cuda_device), ctypes.byref(opt)), "gint_setup")
    return GintContext(h.value, ng, pos.shape[0])


def gint_fold_k_static_max_blocks() -> int:
    return int(_lib.gint_fold_k_static_max_blocks())


def gint_measure_fp64_peak(cuda_device: int = 0, seconds: float = 0.5) -> float:
    out = ctypes.c_double()
    _check(_lib.gint_measure_fp64_peak(int(cuda_device), float(seconds), ctypes.byref(out)), "gint_measure_fp64_peak")
    return float(out.value)
