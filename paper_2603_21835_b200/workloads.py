"""Seeded synthetic workloads for gint_vlocal (BASELINE.json `configs`).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It
produces inputs -- cell, atoms, tabulated radial functions, mesh, V_eff -- and
contains none of the method's arithmetic (no orbital evaluation, no real
spherical harmonics, no interpolation, no H).  The paper's own performance
inputs (bulk-Si supercells, DZP/TZDP SIAB orbitals, 8 a.u. cutoff;
PAPER.md:583-613, Table 1) are not available offline; these Si-like / cluster
recipes stand in for them.  Every constant the BASELINE.json text leaves open
is fixed here and listed in DESIGN.md ("Input recipe").

Layouts (all C-contiguous, float64 / int32):
  lattice[3][3]      rows a1,a2,a3 (bohr)
  ngrid[3]           mesh points along a1,a2,a3; point (i,j,k) sits at
                     (i/N1) a1 + (j/N2) a2 + (k/N3) a3
  V[N1][N2][N3]      local potential on the mesh (Hartree), k fastest
  species[s]         Species(rcut, dr, l[nrad], table[nrad][ntab]); table node
                     k is f(k*dr); f == 0 for r >= rcut; ntab covers rcut+3dr
  atom_species[natom], atom_pos[natom][3]   Cartesian bohr, never wrapped
"""
from __future__ import annotations

import dataclasses
import hashlib
import math
from typing import List, Sequence

import numpy as np

DR = 0.01  # radial table step (bohr), BASELINE.json


@dataclasses.dataclass
class Species:
    name: str
    rcut: float
    dr: float
    l: np.ndarray        # [nrad] int32, l ascending then zeta ascending
    table: np.ndarray    # [nrad][ntab] float64

    @property
    def nrad(self) -> int:
        return int(self.l.shape[0])

    @property
    def ntab(self) -> int:
        return int(self.table.shape[1])

    @property
    def norb(self) -> int:
        return int(np.sum(2 * self.l + 1))


@dataclasses.dataclass
class Workload:
    name: str
    lattice: np.ndarray
    ngrid: np.ndarray
    species: List[Species]
    atom_species: np.ndarray
    atom_pos: np.ndarray
    V: np.ndarray
    seed: int

    @property
    def natom(self) -> int:
        return int(self.atom_pos.shape[0])

    @property
    def norb_total(self) -> int:
        return int(sum(self.species[s].norb for s in self.atom_species))

    def sha256(self) -> str:
        h = hashlib.sha256()
        for a in (self.lattice, self.ngrid, self.atom_species, self.atom_pos, self.V):
            h.update(np.ascontiguousarray(a).tobytes())
        for sp in self.species:
            h.update(np.float64([sp.rcut, sp.dr]).tobytes())
            h.update(np.ascontiguousarray(sp.l).tobytes())
            h.update(np.ascontiguousarray(sp.table).tobytes())
        return h.hexdigest()


# ----------------------------------------------------------------------------
# radial tables
# ----------------------------------------------------------------------------
def radial_table(l: int, alpha: float, rcut: float, dr: float = DR) -> np.ndarray:
    """f(r) = N r^l exp(-alpha r^2) (1-(r/rc)^2)^3 for r<rc, else 0, tabulated at
    k*dr, k = 0 .. round(rc/dr)+3, normalised so that int_0^rc f^2 r^2 dr = 1 by
    composite Simpson on the table nodes 0..rc (BASELINE.json configs[0])."""
    nrc = int(round(rcut / dr))
    assert abs(nrc * dr - rcut) < 1e-9 and nrc % 2 == 0
    ntab = nrc + 4
    r = np.arange(ntab, dtype=np.float64) * dr
    f = np.zeros(ntab, dtype=np.float64)
    inside = np.arange(ntab) < nrc
    ri = r[inside]
    f[inside] = ri ** l * np.exp(-alpha * ri * ri) * (1.0 - (ri / rcut) ** 2) ** 3
    g = (f * f * r * r)[: nrc + 1]
    w = np.ones(nrc + 1)
    w[1:-1:2] = 4.0
    w[2:-1:2] = 2.0
    integral = dr / 3.0 * float(np.sum(w * g))
    return f / math.sqrt(integral)


def gaussian_table(alpha: float, rcut: float, dr: float = DR, l: int = 0) -> np.ndarray:
    """Pure r^l exp(-alpha r^2) table (no cutoff polynomial, no normalisation)
    used by the analytic-overlap pins; zero from rcut on."""
    nrc = int(round(rcut / dr))
    ntab = nrc + 4
    r = np.arange(ntab, dtype=np.float64) * dr
    f = r ** l * np.exp(-alpha * r * r)
    f[nrc:] = 0.0
    return f


def make_species(name: str, rcut: float, shells: Sequence[tuple], dr: float = DR) -> Species:
    """shells: sequence of (l, alpha), already ordered l ascending, zeta ascending."""
    ls = np.array([s[0] for s in shells], dtype=np.int32)
    tab = np.stack([radial_table(int(l), float(a), rcut, dr) for l, a in shells])
    return Species(name=name, rcut=float(rcut), dr=float(dr), l=ls, table=np.ascontiguousarray(tab))


def species_sz(rcut: float = 6.0) -> Species:
    """cfg1: 1s + 1p, alpha = 0.5 (exp(-0.5 r^2)), 4 orbitals."""
    return make_species("Si-SZ", rcut, [(0, 0.5), (1, 0.5)])


def species_dzp(name: str, rcut: float, a1: float, a2: float) -> Species:
    """2s 2p 1d = 13 orbitals; the single d shell uses zeta-1's alpha."""
    return make_species(name, rcut, [(0, a1), (0, a2), (1, a1), (1, a2), (2, a1)])


def species_tzdp(name: str, rcut: float, a1: float, a2: float, a3: float) -> Species:
    """3s 3p 2d = 22 orbitals, the basis of the paper's performance runs."""
    return make_species(name, rcut, [(0, a1), (0, a2), (0, a3), (1, a1), (1, a2), (1, a3), (2, a1), (2, a2)])


def species_dzpf(name: str, rcut: float, a1: float, a2: float) -> Species:
    """2s 2p 1d 1f = 20 orbitals: exercises l = 3 (the paper's larger basis sets carry f shells)."""
    return make_species(name, rcut, [(0, a1), (0, a2), (1, a1), (1, a2), (2, a1), (3, a1)])


def species_2s1p(name: str, rcut: float, a1: float, a2: float) -> Species:
    """H-like 2s 1p = 5 orbitals; the single p shell uses zeta-1's alpha."""
    return make_species(name, rcut, [(0, a1), (0, a2), (1, a1)])


# ----------------------------------------------------------------------------
# nonlocal projectors and atom-centred quadrature tables (gint_snap_psibeta)
# ----------------------------------------------------------------------------
def projector_species(name: str = "Si-beta", rcut: float = 3.0) -> Species:
    """Projector functions beta_{l zeta} of a norm-conserving pseudopotential, tabulated like the orbitals: two s and
    two p projectors (8 components), localised within `rcut` of the nucleus (the paper's projectors are "extremely
    localised around atomic cores").  No real pseudopotential file is available offline; the shapes stand in."""
    return make_species(name, rcut, [(0, 1.2), (0, 2.5), (1, 1.0), (1, 2.0)])


def radial_quadrature(n: int = 140):
    """n-point Gauss-Legendre rule mapped to the unit interval: nodes x in (0, 1) and weights with sum 1 (the paper's
    140-point radial grid; the caller scales by the projector cutoff).  Library routine, no arithmetic
    of the method."""
    x, w = np.polynomial.legendre.leggauss(int(n))
    return np.ascontiguousarray(0.5 * (x + 1.0)), np.ascontiguousarray(0.5 * w)


def angular_quadrature(npts: int = 110):
    """Lebedev-Laikov rule on the unit sphere: unit vectors [npts][3] and weights with sum 4 pi (110 points = order 17,
    PAPER.md:424).  Taken from scipy's table."""
    from scipy.integrate import lebedev_rule
    order = {6: 3, 14: 5, 26: 7, 38: 9, 50: 11, 74: 13, 86: 15, 110: 17, 146: 19, 170: 21, 194: 23, 230: 25, 266: 27,
             302: 29, 350: 31, 434: 35, 590: 41}[int(npts)]
    x, w = lebedev_rule(order)
    return np.ascontiguousarray(x.T), np.ascontiguousarray(w)


# ----------------------------------------------------------------------------
# potentials (orthorhombic cells only -- all BASELINE configs are cubic)
# ----------------------------------------------------------------------------
def _periodic_gauss_1d(n: int, length: float, centre: np.ndarray, sigma2: float, reach: float) -> np.ndarray:
    """g[a, i] = sum over images m with |x_i - c_a - m L| < reach of
    exp(-(x_i - c_a - m L)^2 / sigma2); x_i = i L / n."""
    x = np.arange(n, dtype=np.float64) * (length / n)
    g = np.zeros((centre.shape[0], n))
    mmax = int(math.ceil((reach + np.max(np.abs(centre)) + length) / length)) + 1
    for m in range(-mmax, mmax + 1):
        d = x[None, :] - centre[:, None] - m * length
        g += np.where(np.abs(d) < reach, np.exp(-d * d / sigma2), 0.0)
    return g


def gaussian_wells(lattice, ngrid, pos, depth, sigma2=1.5, reach=8.0) -> np.ndarray:
    """V(r) = sum_{atoms, images} depth_a exp(-|r - tau_a - R|^2 / sigma2); the
    Gaussian factorises along the three orthogonal axes, images are summed per
    axis while |d| < reach (tail < 1e-18)."""
    L = np.diag(lattice)
    assert np.allclose(lattice, np.diag(L)), "generator potentials need an orthorhombic cell"
    gx = _periodic_gauss_1d(int(ngrid[0]), L[0], pos[:, 0], sigma2, reach)
    gy = _periodic_gauss_1d(int(ngrid[1]), L[1], pos[:, 1], sigma2, reach)
    gz = _periodic_gauss_1d(int(ngrid[2]), L[2], pos[:, 2], sigma2, reach)
    depth = np.asarray(depth, dtype=np.float64)
    yz = (gy[:, :, None] * gz[:, None, :]).reshape(pos.shape[0], -1)
    V = (gx * depth[:, None]).T @ yz
    return V.reshape(int(ngrid[0]), int(ngrid[1]), int(ngrid[2]))


def fourier_noise(lattice, ngrid, rng: np.random.Generator, gmax: int = 3, sigma: float = 0.05) -> np.ndarray:
    """sum_G a_G cos(G.r) + b_G sin(G.r) over integer triples 0 < |(h,k,l)| <= gmax,
    one of each +-G pair (first non-zero component positive), lexicographic
    order, a_G then b_G drawn from N(0, sigma^2).  G = 2 pi (h/L1, k/L2, l/L3)."""
    n1, n2, n3 = (int(x) for x in ngrid)
    t1 = 2 * np.pi * np.arange(n1) / n1
    t2 = 2 * np.pi * np.arange(n2) / n2
    t3 = 2 * np.pi * np.arange(n3) / n3
    V = np.zeros((n1, n2, n3))
    for h in range(-gmax, gmax + 1):
        for k in range(-gmax, gmax + 1):
            for l in range(-gmax, gmax + 1):
                n2_ = h * h + k * k + l * l
                if n2_ == 0 or n2_ > gmax * gmax:
                    continue
                first = h if h != 0 else (k if k != 0 else l)
                if first < 0:
                    continue
                a = rng.normal(0.0, sigma)
                b = rng.normal(0.0, sigma)
                ph = h * t1[:, None, None] + k * t2[None, :, None] + l * t3[None, None, :]
                V += a * np.cos(ph) + b * np.sin(ph)
    return V


# ----------------------------------------------------------------------------
# structures
# ----------------------------------------------------------------------------
_DIAMOND = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                     [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
A0 = 10.26  # bohr


def diamond_supercell(nrep: int) -> np.ndarray:
    """Ideal sites of an nrep^3 supercell of the 8-atom cubic diamond cell,
    cell-major (ix, iy, iz) then the 8 basis sites."""
    out = []
    for ix in range(nrep):
        for iy in range(nrep):
            for iz in range(nrep):
                out.append((_DIAMOND + np.array([ix, iy, iz])) * A0)
    return np.concatenate(out, axis=0)


def si_like(nrep: int, seed: int, basis: str, disp: float, ngrid: int, name: str) -> Workload:
    rng = np.random.default_rng(seed)
    a = A0 * nrep
    lattice = np.eye(3) * a
    ideal = diamond_supercell(nrep)
    pos = ideal + rng.uniform(-disp, disp, size=ideal.shape)   # draw 1: displacements [natom][3]
    sp = {"SZ": lambda: species_sz(6.0),
          "DZP": lambda: species_dzp("Si-DZP", 8.0, 0.3, 0.9),
          "TZDP": lambda: species_tzdp("Si-TZDP", 8.0, 0.3, 0.6, 1.2),
          "DZP10": lambda: species_dzp("Si-DZP-rc10", 10.0, 0.3, 0.9),
          "DZPF": lambda: species_dzpf("Si-DZPF", 6.0, 0.5, 1.0)}[basis]()
    ng = np.array([ngrid] * 3, dtype=np.int32)
    V = gaussian_wells(lattice, ng, pos, np.full(pos.shape[0], -2.0))
    V = V + fourier_noise(lattice, ng, rng)                     # draw 2: Fourier coefficients
    return Workload(name=name, lattice=lattice, ngrid=ng, species=[sp],
                    atom_species=np.zeros(pos.shape[0], dtype=np.int32),
                    atom_pos=np.ascontiguousarray(pos), V=np.ascontiguousarray(V), seed=seed)


def cluster60(seed: int = 4, ngrid: int = 160, box: float = 40.0) -> Workload:
    """cfg5: 30 C-like + 30 H-like atoms, uniform in a radius-8 sphere at the box
    centre, min separation 2.0 bohr by seeded rejection (candidates uniform in
    the cube [-8,8]^3 about the centre; first 30 accepted are C-like)."""
    rng = np.random.default_rng(seed)
    pts: list = []
    while len(pts) < 60:
        c = rng.uniform(-8.0, 8.0, size=3)
        if np.dot(c, c) >= 64.0:
            continue
        if any(np.linalg.norm(c - p) < 2.0 for p in pts):
            continue
        pts.append(c)
    pos = np.array(pts) + box / 2.0
    lattice = np.eye(3) * box
    sp_c = species_dzp("C-DZP", 7.0, 0.4, 1.2)
    sp_h = species_2s1p("H-2s1p", 6.0, 0.5, 1.5)
    atom_species = np.array([0] * 30 + [1] * 30, dtype=np.int32)
    ng = np.array([ngrid] * 3, dtype=np.int32)
    depth = np.where(atom_species == 0, -2.0, -1.0)
    V = gaussian_wells(lattice, ng, pos, depth)
    return Workload(name="cluster60", lattice=lattice, ngrid=ng, species=[sp_c, sp_h],
                    atom_species=atom_species, atom_pos=np.ascontiguousarray(pos),
                    V=np.ascontiguousarray(V), seed=seed)


CONFIGS = ("si8_sz", "si64_dzp", "si216_dzp", "si512_dzp", "cluster60")
# second workloads: the paper's own basis (TZDP 3s3p2d = 22 orbitals, rc = 8 a.u.),
# its validation cutoff (rc = 10 a.u.) and an f shell; same cells, meshes, seeds and V recipe
EXTRA_CONFIGS = ("si8_dzpf", "si64_tzdp", "si64_dzp_rc10", "si512_tzdp", "si512_dzp_rc10")


def make(name: str) -> Workload:
    """The five BASELINE.json configs (CONFIGS) and the second workloads (EXTRA_CONFIGS), by name."""
    if name == "si8_sz":
        return si_like(1, 0, "SZ", 0.05, 36, name)
    if name == "si64_dzp":
        return si_like(2, 1, "DZP", 0.1, 72, name)
    if name == "si216_dzp":
        return si_like(3, 2, "DZP", 0.1, 108, name)
    if name == "si512_dzp":
        return si_like(4, 3, "DZP", 0.1, 144, name)
    if name == "cluster60":
        return cluster60()
    if name == "si8_dzpf":
        return si_like(1, 0, "DZPF", 0.05, 36, name)
    if name == "si64_tzdp":
        return si_like(2, 1, "TZDP", 0.1, 72, name)
    if name == "si64_dzp_rc10":
        return si_like(2, 1, "DZP10", 0.1, 72, name)
    if name == "si512_tzdp":
        return si_like(4, 3, "TZDP", 0.1, 144, name)
    if name == "si512_dzp_rc10":
        return si_like(4, 3, "DZP10", 0.1, 144, name)
    raise KeyError(name)


def tiny(seed: int = 7, natom: int = 3, ngrid=(12, 10, 14), lattice=None, shells=((0, 0.6), (1, 0.5), (2, 0.7)),
         rcut: float = 3.0, noise: float = 0.3) -> Workload:
    """Small random workload for brute-force pins and edge cases: general
    (possibly triclinic) lattice, random atoms, random smooth-ish V."""
    rng = np.random.default_rng(seed)
    if lattice is None:
        lattice = np.array([[5.0, 0.0, 0.0], [0.7, 4.6, 0.0], [-0.4, 0.5, 5.4]])
    lattice = np.asarray(lattice, dtype=np.float64)
    frac = rng.uniform(0.0, 1.0, size=(natom, 3))
    pos = frac @ lattice
    sp = make_species("tiny", rcut, list(shells))
    ng = np.array(ngrid, dtype=np.int32)
    V = rng.normal(0.0, noise, size=tuple(int(x) for x in ng)) - 0.5
    return Workload(name="tiny", lattice=lattice, ngrid=ng, species=[sp],
                    atom_species=np.zeros(natom, dtype=np.int32), atom_pos=np.ascontiguousarray(pos),
                    V=np.ascontiguousarray(V), seed=seed)
