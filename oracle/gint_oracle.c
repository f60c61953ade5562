/*
 * gint_oracle.c -- CPU ORACLE for gint_vlocal.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product path
 * (paper_2603_21835_b200/) never does; the two share no code.
 *
 * What it computes (the plain definition, written out; fp64 arithmetic, long
 * double accumulators):
 *
 *   H_mu,nu(R) = dV * sum_{n in Z^3} phi_mu(r_n - tau_I) * V[n mod N]
 *                                  * phi_nu(r_n - tau_J - R)
 *       -- PAPER.md:393-398 (Sec. 3.3.1, Eq. 45); dV defined at PAPER.md:398
 *   phi_mu(r) = f_{I l zeta}(|r|) * Y_lm(r/|r|)
 *       -- PAPER.md:66-70 (Sec. 2.1, Eq. 1)
 *   R = lattice vector from the cell of mu (atom I) to the cell of nu (atom J)
 *       -- PAPER.md:104-106 (text after Eq. 6)
 *   r_n = (n1/N1) a1 + (n2/N2) a2 + (n3/N3) a3,  dV = |det(a1,a2,a3)|/(N1 N2 N3)
 *
 * Readings of the paper where it is silent (numbering
 * of SURVEY.md Sec. 8(c)):
 *   #1 the sum runs over ALL space with V periodic on the mesh;
 *   #2 mesh point (i,j,k) sits at fractional (i/N1, j/N2, k/N3);
 *   #3 V is C-ordered [N1][N2][N3];
 *   #4 radial part: cubic Lagrange on the forward stencil k..k+3, k=floor(r/dr);
 *   #5 phi = 0 iff r >= rcut;
 *   #6 at r < 1e-12 the direction is taken as (0,0,0): Y_00 constant, l>0 -> 0;
 *   #7 real Y_lm in fixed Cartesian form, no Condon-Shortley phase, m-order
 *      l=1: y,z,x; l=2: xy, yz, 3z^2-1, xz, x^2-y^2;
 *   #8 orbitals of an atom: radial functions in the given order, each with its
 *      2l+1 m-components;
 *   #9 block set: every (I,J,R) with |tau_J + R - tau_I| < rc_I + rc_J (strict),
 *      sorted by (I, J, R1, R2, R3); block row-major n_I x n_J.
 *
 * Structure (deliberately unlike the CUDA path: atom-pair-major, no big
 * cells, no cell lists): for every atom I list the unwrapped mesh points inside
 * its sphere with phi_I there; for every block of I walk that list, evaluate
 * phi_J on the points also inside J's sphere, accumulate.
 *
 * Pins: tests/test_oracle_pins.py (brute force, H(R)=H(-R)^T, V=c, Gaussian
 * closed forms, plane-wave V, unit impulse, shift/roll, Bloch-sum dense GEMM,
 * cubic reproduction, Unsold, quadrature orthonormality, 90-degree rotation).
 * Conventions #4, #7, #8 cannot be pinned against ABACUS output (none is
 * printed in the paper); they are pinned by the closed forms above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_ORB 64

typedef struct {
    double rcut, dr;
    int ntab, nrad;
    const int *l;        /* [nrad] */
    const double *table; /* [nrad][ntab] */
    int norb;
} orc_species;

/* ---- real spherical harmonics, l <= 2 (reading #7) ---------------------- */
static int ylm_real(int l, double x, double y, double z, double *out)
{
    const double pi = 3.14159265358979323846;
    if (l == 0) {
        out[0] = 0.5 * sqrt(1.0 / pi);
        return 1;
    }
    if (l == 1) {
        double c = sqrt(3.0 / (4.0 * pi));
        out[0] = c * y;
        out[1] = c * z;
        out[2] = c * x;
        return 3;
    }
    if (l == 2) {
        double c1 = 0.5 * sqrt(15.0 / pi);
        double c2 = 0.25 * sqrt(5.0 / pi);
        double c3 = 0.25 * sqrt(15.0 / pi);
        out[0] = c1 * x * y;
        out[1] = c1 * y * z;
        out[2] = c2 * (3.0 * z * z - 1.0);
        out[3] = c1 * x * z;
        out[4] = c3 * (x * x - y * y);
        return 5;
    }
    if (l == 3) { /* reading #7 extended: real f harmonics, m = -3..3, Cartesian forms on the unit sphere */
        double a = 0.25 * sqrt(35.0 / (2.0 * pi)); /* m = -3, +3 */
        double b = 0.5 * sqrt(105.0 / pi);         /* m = -2 */
        double c = 0.25 * sqrt(21.0 / (2.0 * pi)); /* m = -1, +1 */
        double d = 0.25 * sqrt(7.0 / pi);          /* m = 0 */
        double e = 0.25 * sqrt(105.0 / pi);        /* m = +2 */
        out[0] = a * y * (3.0 * x * x - y * y);
        out[1] = b * x * y * z;
        out[2] = c * y * (5.0 * z * z - 1.0);
        out[3] = d * z * (5.0 * z * z - 3.0);
        out[4] = c * x * (5.0 * z * z - 1.0);
        out[5] = e * z * (x * x - y * y);
        out[6] = a * x * (x * x - 3.0 * y * y);
        return 7;
    }
    return -1;
}

/* ---- radial part: 4-point Lagrange, forward stencil (reading #4) -------- */
static double radial_interp(const double *T, double r, double dr)
{
    double s = r / dr;
    int k = (int)floor(s);
    double t = s - (double)k;
    double L0 = (1.0 - t) * (2.0 - t) * (3.0 - t) / 6.0;
    double L1 = t * (2.0 - t) * (3.0 - t) / 2.0;
    double L2 = -t * (1.0 - t) * (3.0 - t) / 2.0;
    double L3 = t * (1.0 - t) * (2.0 - t) / 6.0;
    return T[k] * L0 + T[k + 1] * L1 + T[k + 2] * L2 + T[k + 3] * L3;
}

/* phi_mu(d) for all orbitals of one species; returns 0 if outside the cutoff
 * (out is zero-filled), 1 otherwise.  Eq. 1. */
static int phi_eval(const orc_species *sp, const double d[3], double *out)
{
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    int o = 0;
    if (!(r < sp->rcut)) {
        for (int i = 0; i < sp->norb; i++) out[i] = 0.0;
        return 0;
    }
    double x = 0.0, y = 0.0, z = 0.0;
    if (r >= 1e-12) {
        x = d[0] / r;
        y = d[1] / r;
        z = d[2] / r;
    }
    for (int k = 0; k < sp->nrad; k++) {
        double f = radial_interp(sp->table + (size_t)k * sp->ntab, r, sp->dr);
        double Y[7];
        int nm = ylm_real(sp->l[k], x, y, z, Y);
        if (sp->l[k] > 0 && r < 1e-12) /* reading #6: l>0 -> 0 at the nucleus */
            for (int m = 0; m < nm; m++) Y[m] = 0.0;
        for (int m = 0; m < nm; m++) out[o++] = f * Y[m];
    }
    return 1;
}

/* ---- small geometry helpers --------------------------------------------- */
static double det3(const double *A)
{
    return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
           A[2] * (A[3] * A[7] - A[4] * A[6]);
}

/* inv = A^{-1} (A rows are lattice vectors; frac = cart * inv) */
static void inv3(const double *A, double *inv)
{
    double d = det3(A);
    inv[0] = (A[4] * A[8] - A[5] * A[7]) / d;
    inv[1] = (A[2] * A[7] - A[1] * A[8]) / d;
    inv[2] = (A[1] * A[5] - A[2] * A[4]) / d;
    inv[3] = (A[5] * A[6] - A[3] * A[8]) / d;
    inv[4] = (A[0] * A[8] - A[2] * A[6]) / d;
    inv[5] = (A[2] * A[3] - A[0] * A[5]) / d;
    inv[6] = (A[3] * A[7] - A[4] * A[6]) / d;
    inv[7] = (A[1] * A[6] - A[0] * A[7]) / d;
    inv[8] = (A[0] * A[4] - A[1] * A[3]) / d;
}

static void unpack_species(int nspecies, const double *sp_rcut, const double *sp_dr, const int *sp_ntab,
                           const int *sp_nrad, const int *sp_l, const double *sp_table, orc_species *sp)
{
    size_t lo = 0, to = 0;
    for (int s = 0; s < nspecies; s++) {
        sp[s].rcut = sp_rcut[s];
        sp[s].dr = sp_dr[s];
        sp[s].ntab = sp_ntab[s];
        sp[s].nrad = sp_nrad[s];
        sp[s].l = sp_l + lo;
        sp[s].table = sp_table + to;
        sp[s].norb = 0;
        for (int k = 0; k < sp_nrad[s]; k++) sp[s].norb += 2 * sp_l[lo + k] + 1;
        lo += (size_t)sp_nrad[s];
        to += (size_t)sp_nrad[s] * (size_t)sp_ntab[s];
    }
}

/* ---- public: orbital values at one displacement (used by the pins) ------ */
int orc_phi(int nspecies, const double *sp_rcut, const double *sp_dr, const int *sp_ntab, const int *sp_nrad,
            const int *sp_l, const double *sp_table, int species, int npts, const double *d /* [npts][3] */,
            double *out /* [npts][norb] */)
{
    orc_species sp[16];
    if (nspecies > 16 || species < 0 || species >= nspecies) return -1;
    unpack_species(nspecies, sp_rcut, sp_dr, sp_ntab, sp_nrad, sp_l, sp_table, sp);
    for (int p = 0; p < npts; p++) phi_eval(&sp[species], d + 3 * (size_t)p, out + (size_t)p * sp[species].norb);
    return sp[species].norb;
}

/* ---- public: block enumeration (reading #9) ------------------------------
 * Pass cap = 0 to count only.  Returns the number of blocks, or -1.          */
int64_t orc_enumerate_blocks(const double *lattice, int natom, const double *pos, const double *rc_atom,
                             int64_t cap, int32_t *bi, int32_t *bj, int32_t *bR /* [cap][3] */)
{
    double inv[9];
    if (fabs(det3(lattice)) < 1e-300) return -1;
    inv3(lattice, inv);
    /* |b_i| = length of column i of A^{-1}: the fractional coordinate i changes by at
     * most rho*|b_i| inside a ball of radius rho */
    double blen[3];
    for (int i = 0; i < 3; i++) blen[i] = sqrt(inv[i] * inv[i] + inv[3 + i] * inv[3 + i] + inv[6 + i] * inv[6 + i]);
    int64_t nb = 0;
    for (int I = 0; I < natom; I++)
        for (int J = 0; J < natom; J++) {
            double dc[3] = {pos[3 * I] - pos[3 * J], pos[3 * I + 1] - pos[3 * J + 1], pos[3 * I + 2] - pos[3 * J + 2]};
            double reach = rc_atom[I] + rc_atom[J];
            int lo[3], hi[3];
            for (int i = 0; i < 3; i++) {
                double f = dc[0] * inv[i] + dc[1] * inv[3 + i] + dc[2] * inv[6 + i]; /* frac of tau_I - tau_J */
                lo[i] = (int)floor(f - reach * blen[i]) - 1;
                hi[i] = (int)ceil(f + reach * blen[i]) + 1;
            }
            for (int r1 = lo[0]; r1 <= hi[0]; r1++)
                for (int r2 = lo[1]; r2 <= hi[1]; r2++)
                    for (int r3 = lo[2]; r3 <= hi[2]; r3++) {
                        double v[3];
                        for (int c = 0; c < 3; c++)
                            v[c] = r1 * lattice[c] + r2 * lattice[3 + c] + r3 * lattice[6 + c] - dc[c];
                        double dist = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
                        if (dist < reach) {
                            if (nb < cap) {
                                bi[nb] = I;
                                bj[nb] = J;
                                bR[3 * nb] = r1;
                                bR[3 * nb + 1] = r2;
                                bR[3 * nb + 2] = r3;
                            }
                            nb++;
                        }
                    }
        }
    return nb;
}

static inline int64_t pmod(int64_t a, int64_t n)
{
    int64_t m = a % n;
    return m < 0 ? m + n : m;
}

/* ---- public: H for a list of blocks --------------------------------------
 * blocks (bi,bj,bR) may be any subset, but must be grouped by bi (all blocks of
 * one row atom contiguous) -- the sorted full list is.  out_off[b] = first
 * double of block b in out; block is row-major n_I x n_J.
 * nthreads <= 0: OpenMP default.  Returns threads used, or <0 on error.      */
int orc_vlocal(const double *lattice, const int *ngrid, int nspecies, const double *sp_rcut, const double *sp_dr,
               const int *sp_ntab, const int *sp_nrad, const int *sp_l, const double *sp_table, int natom_unused,
               const int *atom_species, const double *pos, const double *V, int64_t nblk, const int32_t *bi,
               const int32_t *bj, const int32_t *bR, const int64_t *out_off, double *out, int nthreads)
{
    orc_species sp[16];
    (void)natom_unused;
    if (nspecies > 16) return -1;
    unpack_species(nspecies, sp_rcut, sp_dr, sp_ntab, sp_nrad, sp_l, sp_table, sp);
    for (int s = 0; s < nspecies; s++)
        if (sp[s].norb > ORC_MAX_ORB) return -2;
    double inv[9];
    double vol = fabs(det3(lattice));
    if (vol < 1e-300) return -3;
    inv3(lattice, inv);
    double blen[3];
    for (int i = 0; i < 3; i++) blen[i] = sqrt(inv[i] * inv[i] + inv[3 + i] * inv[3 + i] + inv[6 + i] * inv[6 + i]);
    const int64_t N1 = ngrid[0], N2 = ngrid[1], N3 = ngrid[2];
    const double dV = vol / ((double)N1 * (double)N2 * (double)N3);

    /* groups of consecutive blocks with the same row atom */
    int64_t ngroup = 0;
    int64_t *gstart = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nblk + 1));
    if (!gstart) return -4;
    for (int64_t b = 0; b < nblk; b++)
        if (b == 0 || bi[b] != bi[b - 1]) gstart[ngroup++] = b;
    gstart[ngroup] = nblk;

    int used = 1;
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t g = 0; g < ngroup; g++) {
        const int I = bi[gstart[g]];
        const orc_species *sI = &sp[atom_species[I]];
        const double *tI = pos + 3 * (size_t)I;
        /* step 1: unwrapped mesh points inside the sphere of I, with phi_I */
        int lo[3], hi[3];
        for (int i = 0; i < 3; i++) {
            double f = tI[0] * inv[i] + tI[1] * inv[3 + i] + tI[2] * inv[6 + i];
            lo[i] = (int)floor((f - sI->rcut * blen[i]) * (double)ngrid[i]) - 1;
            hi[i] = (int)ceil((f + sI->rcut * blen[i]) * (double)ngrid[i]) + 1;
        }
        size_t cap = (size_t)(hi[0] - lo[0] + 1) * (size_t)(hi[1] - lo[1] + 1) * (size_t)(hi[2] - lo[2] + 1);
        int32_t *pn = (int32_t *)malloc(sizeof(int32_t) * 3 * cap);
        double *pphi = (double *)malloc(sizeof(double) * (size_t)sI->norb * cap);
        if (!pn || !pphi) {
            err = 1;
            free(pn);
            free(pphi);
            continue;
        }
        size_t np = 0;
        for (int n1 = lo[0]; n1 <= hi[0]; n1++)
            for (int n2 = lo[1]; n2 <= hi[1]; n2++)
                for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                    double f1 = (double)n1 / (double)N1, f2 = (double)n2 / (double)N2, f3 = (double)n3 / (double)N3;
                    double d[3];
                    for (int c = 0; c < 3; c++)
                        d[c] = f1 * lattice[c] + f2 * lattice[3 + c] + f3 * lattice[6 + c] - tI[c];
                    if (phi_eval(sI, d, pphi + np * (size_t)sI->norb)) {
                        pn[3 * np] = n1;
                        pn[3 * np + 1] = n2;
                        pn[3 * np + 2] = n3;
                        np++;
                    }
                }
        /* steps 2-3: every block of this row atom */
        for (int64_t b = gstart[g]; b < gstart[g + 1]; b++) {
            const int J = bj[b];
            const orc_species *sJ = &sp[atom_species[J]];
            const int nI = sI->norb, nJ = sJ->norb;
            double cJ[3]; /* tau_J + R */
            for (int c = 0; c < 3; c++)
                cJ[c] = pos[3 * (size_t)J + c] + bR[3 * b] * lattice[c] + bR[3 * b + 1] * lattice[3 + c] +
                        bR[3 * b + 2] * lattice[6 + c];
            long double acc[ORC_MAX_ORB * ORC_MAX_ORB];
            for (int i = 0; i < nI * nJ; i++) acc[i] = 0.0L;
            double phiJ[ORC_MAX_ORB];
            for (size_t p = 0; p < np; p++) {
                int n1 = pn[3 * p], n2 = pn[3 * p + 1], n3 = pn[3 * p + 2];
                double f1 = (double)n1 / (double)N1, f2 = (double)n2 / (double)N2, f3 = (double)n3 / (double)N3;
                double d[3];
                for (int c = 0; c < 3; c++)
                    d[c] = f1 * lattice[c] + f2 * lattice[3 + c] + f3 * lattice[6 + c] - cJ[c];
                if (!phi_eval(sJ, d, phiJ)) continue;
                double v = V[(pmod(n1, N1) * N2 + pmod(n2, N2)) * N3 + pmod(n3, N3)];
                const double *phiI = pphi + p * (size_t)nI;
                for (int mu = 0; mu < nI; mu++) {
                    double a = phiI[mu] * v;
                    for (int nu = 0; nu < nJ; nu++) acc[mu * nJ + nu] += (long double)(a * phiJ[nu]);
                }
            }
            double *o = out + out_off[b];
            for (int i = 0; i < nI * nJ; i++) o[i] = (double)(acc[i] * (long double)dV);
        }
        free(pn);
        free(pphi);
    }
    free(gstart);
    return err ? -5 : used;
}

/* ---- public: charge density on the mesh -----------------------------------
 *   rho(r_g) = sum_{R,R'} sum_{mu,nu} rho_mu,nu(R) phi_mu(r_g - tau_I - R')
 *                                     phi_nu(r_g - tau_J - R - R')
 *       -- PAPER.md:384-391 (Sec. 3.3.1, Eq. 44)
 * written out: for every block (I,J,R) and every UNWRAPPED mesh point n (the
 * sum over R' is the sum over the unwrapped points that fold onto g = n mod N)
 * inside both spheres, add D_mu,nu phi_mu(r_n - tau_I) phi_nu(r_n - tau_J - R)
 * to rho[n mod N].  D holds the listed blocks back to back (same layout as H).
 * blocks must be grouped by bi.  rho[N1][N2][N3] is overwritten.
 * Pinned in tests/test_oracle_pins.py by the adjoint identity
 *   sum_g V(g) rho(g) dV = sum_blocks D : H[V]   (H from orc_vlocal)
 * and by a brute-force sum on a tiny cell.  Returns threads used or <0.      */
int orc_rho(const double *lattice, const int *ngrid, int nspecies, const double *sp_rcut, const double *sp_dr,
            const int *sp_ntab, const int *sp_nrad, const int *sp_l, const double *sp_table, int natom_unused,
            const int *atom_species, const double *pos, int64_t nblk, const int32_t *bi, const int32_t *bj,
            const int32_t *bR, const int64_t *d_off, const double *D, double *rho, int nthreads)
{
    orc_species sp[16];
    (void)natom_unused;
    if (nspecies > 16) return -1;
    unpack_species(nspecies, sp_rcut, sp_dr, sp_ntab, sp_nrad, sp_l, sp_table, sp);
    for (int s = 0; s < nspecies; s++)
        if (sp[s].norb > ORC_MAX_ORB) return -2;
    double inv[9];
    double vol = fabs(det3(lattice));
    if (vol < 1e-300) return -3;
    inv3(lattice, inv);
    double blen[3];
    for (int i = 0; i < 3; i++) blen[i] = sqrt(inv[i] * inv[i] + inv[3 + i] * inv[3 + i] + inv[6 + i] * inv[6 + i]);
    const int64_t N1 = ngrid[0], N2 = ngrid[1], N3 = ngrid[2];
    for (int64_t i = 0; i < N1 * N2 * N3; i++) rho[i] = 0.0;

    int64_t ngroup = 0;
    int64_t *gstart = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nblk + 1));
    if (!gstart) return -4;
    for (int64_t b = 0; b < nblk; b++)
        if (b == 0 || bi[b] != bi[b - 1]) gstart[ngroup++] = b;
    gstart[ngroup] = nblk;

    int used = 1;
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t g = 0; g < ngroup; g++) {
        const int I = bi[gstart[g]];
        const orc_species *sI = &sp[atom_species[I]];
        const double *tI = pos + 3 * (size_t)I;
        int lo[3], hi[3];
        for (int i = 0; i < 3; i++) {
            double f = tI[0] * inv[i] + tI[1] * inv[3 + i] + tI[2] * inv[6 + i];
            lo[i] = (int)floor((f - sI->rcut * blen[i]) * (double)ngrid[i]) - 1;
            hi[i] = (int)ceil((f + sI->rcut * blen[i]) * (double)ngrid[i]) + 1;
        }
        double phiI[ORC_MAX_ORB], phiJ[ORC_MAX_ORB];
        for (int n1 = lo[0]; n1 <= hi[0]; n1++)
            for (int n2 = lo[1]; n2 <= hi[1]; n2++)
                for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                    double f1 = (double)n1 / (double)N1, f2 = (double)n2 / (double)N2, f3 = (double)n3 / (double)N3;
                    double r[3], d[3];
                    for (int c = 0; c < 3; c++) {
                        r[c] = f1 * lattice[c] + f2 * lattice[3 + c] + f3 * lattice[6 + c];
                        d[c] = r[c] - tI[c];
                    }
                    if (!phi_eval(sI, d, phiI)) continue;
                    long double acc = 0.0L;
                    for (int64_t b = gstart[g]; b < gstart[g + 1]; b++) {
                        const int J = bj[b];
                        const orc_species *sJ = &sp[atom_species[J]];
                        for (int c = 0; c < 3; c++)
                            d[c] = r[c] - (pos[3 * (size_t)J + c] + bR[3 * b] * lattice[c] + bR[3 * b + 1] * lattice[3 + c] +
                                           bR[3 * b + 2] * lattice[6 + c]);
                        if (!phi_eval(sJ, d, phiJ)) continue;
                        const double *Db = D + d_off[b];
                        for (int mu = 0; mu < sI->norb; mu++) {
                            double t = 0.0;
                            for (int nu = 0; nu < sJ->norb; nu++) t += Db[mu * sJ->norb + nu] * phiJ[nu];
                            acc += (long double)(phiI[mu] * t);
                        }
                    }
                    double *o = rho + (pmod(n1, N1) * N2 + pmod(n2, N2)) * N3 + pmod(n3, N3);
                    double add = (double)acc;
#ifdef _OPENMP
#pragma omp atomic
#endif
                    *o += add;
                }
    }
    free(gstart);
    return err ? -5 : used;
}

/* ==== local Pulay force (the paper's cal_gint_fvl) ===========================================
 *
 *   F_I = - sum_R sum_{mu,nu} rho_{nu mu}(R) sum_g [ d phi_mu(r_g - tau_I)/d tau_I  V(r_g) phi_nu(r_g - tau_J - R)
 *                                                   + phi_mu(r_g - tau_I) V(r_g) d phi_nu(r_g - tau_J - R)/d tau_I ] dV
 *       -- PAPER.md:400-411 (Sec. 3.3.1, Eq. 46); general form PAPER.md:262-266 (Eq. 30): "The derivatives of the
 *          NAOs are computed analytically for the angular part (real spherical harmonics) and numerically for the
 *          radial part."
 *
 * Readings:
 *   #18 The density-matrix coefficient of the orbital pair (mu on atom I in cell 0, nu on atom J in cell R) is the
 *       block element D(I,J,R)[mu][nu] -- the same coefficient that Eq. 44 calls rho_{mu nu}(R) and Eq. 46 calls
 *       rho_{nu mu}(R) (with Eq. 29, E = sum_R sum_{mu nu} rho_{nu mu}(R) H_{mu nu}(R)).  Hence
 *           F_K = - sum_blocks sum_{mu nu} D(I,J,R)[mu][nu] * d H(I,J,R)[mu][nu] / d tau_K   at fixed V and D,
 *       the derivative acting on phi_mu when K = I and on phi_nu when K = J (both when I = J).  With
 *       d phi(r - tau)/d tau = -grad phi(r - tau):
 *           F_I += dV sum_n V[n mod N] sum_{mu nu} D[mu][nu] grad phi_mu(r_n - tau_I) phi_nu(r_n - tau_J - R)
 *           F_J += dV sum_n V[n mod N] sum_{mu nu} D[mu][nu] phi_mu(r_n - tau_I) grad phi_nu(r_n - tau_J - R)
 *       (all-space sum over unwrapped mesh points n, reading #1).
 *   #19 Radial derivative: the derivative of the SAME cubic Lagrange interpolant that defines f (reading #4),
 *       f'(r) = (1/dr) sum_j T[k+j] L_j'(t); angular part analytic.  With phi = f(r) P(d/r), P the homogeneous
 *       polynomial of degree l behind Y_lm:  grad phi = f' rhat P + (f / r) (gradP(rhat) - l P rhat).
 *   #20 At r < 1e-12 (reading #6) the limit for f ~ r^l is used: grad phi = c_1 f'(0) e_m for l = 1, 0 otherwise.
 *       Outside the cutoff (r >= rcut) grad phi = 0.
 */

/* derivative of the interpolant with respect to r */
static double radial_interp_deriv(const double *T, double r, double dr)
{
    double s = r / dr;
    int k = (int)floor(s);
    double t = s - (double)k;
    /* d/dt of L0..L3 of radial_interp */
    double D0 = -((2.0 - t) * (3.0 - t) + (1.0 - t) * (3.0 - t) + (1.0 - t) * (2.0 - t)) / 6.0;
    double D1 = ((2.0 - t) * (3.0 - t) - t * (3.0 - t) - t * (2.0 - t)) / 2.0;
    double D2 = -((1.0 - t) * (3.0 - t) - t * (3.0 - t) - t * (1.0 - t)) / 2.0;
    double D3 = ((1.0 - t) * (2.0 - t) - t * (2.0 - t) - t * (1.0 - t)) / 6.0;
    return (T[k] * D0 + T[k + 1] * D1 + T[k + 2] * D2 + T[k + 3] * D3) / dr;
}

/* homogeneous polynomials P_lm(x,y,z) with Y_lm(rhat) = P_lm(rhat), and their Cartesian gradients (reading #7) */
static int ylm_poly_grad(int l, double x, double y, double z, double *P, double (*G)[3])
{
    const double pi = 3.14159265358979323846;
    if (l == 0) {
        P[0] = 0.5 * sqrt(1.0 / pi);
        G[0][0] = G[0][1] = G[0][2] = 0.0;
        return 1;
    }
    if (l == 1) {
        double c = sqrt(3.0 / (4.0 * pi));
        P[0] = c * y; G[0][0] = 0.0; G[0][1] = c;   G[0][2] = 0.0;
        P[1] = c * z; G[1][0] = 0.0; G[1][1] = 0.0; G[1][2] = c;
        P[2] = c * x; G[2][0] = c;   G[2][1] = 0.0; G[2][2] = 0.0;
        return 3;
    }
    if (l == 2) {
        double c1 = 0.5 * sqrt(15.0 / pi), c2 = 0.25 * sqrt(5.0 / pi), c3 = 0.25 * sqrt(15.0 / pi);
        P[0] = c1 * x * y;                         G[0][0] = c1 * y;        G[0][1] = c1 * x;        G[0][2] = 0.0;
        P[1] = c1 * y * z;                         G[1][0] = 0.0;           G[1][1] = c1 * z;        G[1][2] = c1 * y;
        P[2] = c2 * (2.0 * z * z - x * x - y * y); G[2][0] = -2.0 * c2 * x; G[2][1] = -2.0 * c2 * y; G[2][2] = 4.0 * c2 * z;
        P[3] = c1 * x * z;                         G[3][0] = c1 * z;        G[3][1] = 0.0;           G[3][2] = c1 * x;
        P[4] = c3 * (x * x - y * y);               G[4][0] = 2.0 * c3 * x;  G[4][1] = -2.0 * c3 * y; G[4][2] = 0.0;
        return 5;
    }
    if (l == 3) { /* homogeneous cubic forms of the f harmonics (r^2 = x^2 + y^2 + z^2 put back) and their gradients */
        double a = 0.25 * sqrt(35.0 / (2.0 * pi)), b = 0.5 * sqrt(105.0 / pi), c = 0.25 * sqrt(21.0 / (2.0 * pi));
        double d = 0.25 * sqrt(7.0 / pi), e = 0.25 * sqrt(105.0 / pi);
        double q = 4.0 * z * z - x * x - y * y; /* 5 z^2 - r^2 */
        P[0] = a * y * (3.0 * x * x - y * y);
        G[0][0] = a * 6.0 * x * y; G[0][1] = a * (3.0 * x * x - 3.0 * y * y); G[0][2] = 0.0;
        P[1] = b * x * y * z;
        G[1][0] = b * y * z; G[1][1] = b * x * z; G[1][2] = b * x * y;
        P[2] = c * y * q;
        G[2][0] = c * (-2.0 * x * y); G[2][1] = c * (q - 2.0 * y * y); G[2][2] = c * 8.0 * y * z;
        P[3] = d * z * (2.0 * z * z - 3.0 * x * x - 3.0 * y * y); /* z (5 z^2 - 3 r^2) */
        G[3][0] = d * (-6.0 * x * z); G[3][1] = d * (-6.0 * y * z); G[3][2] = d * (6.0 * z * z - 3.0 * x * x - 3.0 * y * y);
        P[4] = c * x * q;
        G[4][0] = c * (q - 2.0 * x * x); G[4][1] = c * (-2.0 * x * y); G[4][2] = c * 8.0 * x * z;
        P[5] = e * z * (x * x - y * y);
        G[5][0] = e * 2.0 * x * z; G[5][1] = -e * 2.0 * y * z; G[5][2] = e * (x * x - y * y);
        P[6] = a * x * (x * x - 3.0 * y * y);
        G[6][0] = a * (3.0 * x * x - 3.0 * y * y); G[6][1] = -a * 6.0 * x * y; G[6][2] = 0.0;
        return 7;
    }
    return -1;
}

/* phi and grad phi for all orbitals of one species at displacement d; returns 0 outside the cutoff */
static int phi_grad_eval(const orc_species *sp, const double d[3], double *phi, double (*grad)[3])
{
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    int o = 0;
    if (!(r < sp->rcut)) {
        for (int i = 0; i < sp->norb; i++) phi[i] = grad[i][0] = grad[i][1] = grad[i][2] = 0.0;
        return 0;
    }
    double u[3] = {0.0, 0.0, 0.0};
    if (r >= 1e-12) {
        u[0] = d[0] / r;
        u[1] = d[1] / r;
        u[2] = d[2] / r;
    }
    for (int k = 0; k < sp->nrad; k++) {
        const double *T = sp->table + (size_t)k * sp->ntab;
        const int l = sp->l[k];
        double f = radial_interp(T, r, sp->dr), fp = radial_interp_deriv(T, r, sp->dr);
        double P[7], G[7][3];
        int nm = ylm_poly_grad(l, u[0], u[1], u[2], P, G);
        for (int m = 0; m < nm; m++, o++) {
            if (r < 1e-12) { /* reading #20 */
                phi[o] = (l == 0) ? f * P[m] : 0.0;
                for (int c = 0; c < 3; c++) grad[o][c] = (l == 1) ? fp * G[m][c] : 0.0;
            } else {
                phi[o] = f * P[m];
                for (int c = 0; c < 3; c++)
                    grad[o][c] = fp * u[c] * P[m] + (f / r) * (G[m][c] - (double)l * P[m] * u[c]);
            }
        }
    }
    return 1;
}

/* public: orbital gradients at given displacements (used by the pins) */
int orc_phi_grad(int nspecies, const double *sp_rcut, const double *sp_dr, const int *sp_ntab, const int *sp_nrad,
                 const int *sp_l, const double *sp_table, int species, int npts, const double *d /* [npts][3] */,
                 double *phi /* [npts][norb] */, double *grad /* [npts][norb][3] */)
{
    orc_species sp[16];
    if (nspecies > 16 || species < 0 || species >= nspecies) return -1;
    unpack_species(nspecies, sp_rcut, sp_dr, sp_ntab, sp_nrad, sp_l, sp_table, sp);
    if (sp[species].norb > ORC_MAX_ORB) return -2;
    for (int p = 0; p < npts; p++)
        phi_grad_eval(&sp[species], d + 3 * (size_t)p, phi + (size_t)p * sp[species].norb,
                      (double(*)[3])(grad + (size_t)p * sp[species].norb * 3));
    return sp[species].norb;
}

/* public: forces F[natom][3] (overwritten) from density-matrix blocks D (H layout), Eq. 46 as read above.
 * blocks grouped by bi.  Returns threads used or <0. */
int orc_fvl(const double *lattice, const int *ngrid, int nspecies, const double *sp_rcut, const double *sp_dr,
            const int *sp_ntab, const int *sp_nrad, const int *sp_l, const double *sp_table, int natom,
            const int *atom_species, const double *pos, const double *V, int64_t nblk, const int32_t *bi,
            const int32_t *bj, const int32_t *bR, const int64_t *d_off, const double *D, double *F, int nthreads)
{
    orc_species sp[16];
    if (nspecies > 16) return -1;
    unpack_species(nspecies, sp_rcut, sp_dr, sp_ntab, sp_nrad, sp_l, sp_table, sp);
    for (int s = 0; s < nspecies; s++)
        if (sp[s].norb > ORC_MAX_ORB) return -2;
    double inv[9];
    double vol = fabs(det3(lattice));
    if (vol < 1e-300) return -3;
    inv3(lattice, inv);
    double blen[3];
    for (int i = 0; i < 3; i++) blen[i] = sqrt(inv[i] * inv[i] + inv[3 + i] * inv[3 + i] + inv[6 + i] * inv[6 + i]);
    const int64_t N1 = ngrid[0], N2 = ngrid[1], N3 = ngrid[2];
    const double dV = vol / ((double)N1 * (double)N2 * (double)N3);
    long double *Facc = (long double *)calloc((size_t)natom * 3, sizeof(long double));
    int64_t *gstart = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nblk + 1));
    if (!Facc || !gstart) {
        free(Facc);
        free(gstart);
        return -4;
    }
    int64_t ngroup = 0;
    for (int64_t b = 0; b < nblk; b++)
        if (b == 0 || bi[b] != bi[b - 1]) gstart[ngroup++] = b;
    gstart[ngroup] = nblk;

    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#endif
    /* one private accumulator array per thread, summed at the end: the terms and their long double accumulation are
     * unchanged; only the contended atomic updates of long doubles (lock-based, 6 per (point, block)) are gone */
    long double *Fthr = (long double *)calloc((size_t)used * (size_t)natom * 3, sizeof(long double));
    if (!Fthr) {
        free(Facc);
        free(gstart);
        return -4;
    }
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t g = 0; g < ngroup; g++) {
        int me = 0;
#ifdef _OPENMP
        me = omp_get_thread_num();
#endif
        long double *Fme = Fthr + (size_t)me * (size_t)natom * 3;
        const int I = bi[gstart[g]];
        const orc_species *sI = &sp[atom_species[I]];
        const double *tI = pos + 3 * (size_t)I;
        int lo[3], hi[3];
        for (int i = 0; i < 3; i++) {
            double f = tI[0] * inv[i] + tI[1] * inv[3 + i] + tI[2] * inv[6 + i];
            lo[i] = (int)floor((f - sI->rcut * blen[i]) * (double)ngrid[i]) - 1;
            hi[i] = (int)ceil((f + sI->rcut * blen[i]) * (double)ngrid[i]) + 1;
        }
        double phiI[ORC_MAX_ORB], gI[ORC_MAX_ORB][3], phiJ[ORC_MAX_ORB], gJ[ORC_MAX_ORB][3];
        for (int n1 = lo[0]; n1 <= hi[0]; n1++)
            for (int n2 = lo[1]; n2 <= hi[1]; n2++)
                for (int n3 = lo[2]; n3 <= hi[2]; n3++) {
                    double f1 = (double)n1 / (double)N1, f2 = (double)n2 / (double)N2, f3 = (double)n3 / (double)N3;
                    double r[3], d[3];
                    for (int c = 0; c < 3; c++) {
                        r[c] = f1 * lattice[c] + f2 * lattice[3 + c] + f3 * lattice[6 + c];
                        d[c] = r[c] - tI[c];
                    }
                    if (!phi_grad_eval(sI, d, phiI, gI)) continue;
                    const double v = V[(pmod(n1, N1) * N2 + pmod(n2, N2)) * N3 + pmod(n3, N3)];
                    for (int64_t b = gstart[g]; b < gstart[g + 1]; b++) {
                        const int J = bj[b];
                        const orc_species *sJ = &sp[atom_species[J]];
                        for (int c = 0; c < 3; c++)
                            d[c] = r[c] - (pos[3 * (size_t)J + c] + bR[3 * b] * lattice[c] + bR[3 * b + 1] * lattice[3 + c] +
                                           bR[3 * b + 2] * lattice[6 + c]);
                        if (!phi_grad_eval(sJ, d, phiJ, gJ)) continue;
                        const double *Db = D + d_off[b];
                        double fI[3] = {0.0, 0.0, 0.0}, fJ[3] = {0.0, 0.0, 0.0};
                        for (int mu = 0; mu < sI->norb; mu++)
                            for (int nu = 0; nu < sJ->norb; nu++) {
                                const double dmn = Db[mu * sJ->norb + nu];
                                for (int c = 0; c < 3; c++) {
                                    fI[c] += dmn * gI[mu][c] * phiJ[nu];
                                    fJ[c] += dmn * phiI[mu] * gJ[nu][c];
                                }
                            }
                        for (int c = 0; c < 3; c++) {
                            Fme[3 * (size_t)I + c] += (long double)(v * fI[c]);
                            Fme[3 * (size_t)J + c] += (long double)(v * fJ[c]);
                        }
                    }
                }
    }
    for (int t = 0; t < used; t++)
        for (int i = 0; i < 3 * natom; i++) Facc[i] += Fthr[(size_t)t * (size_t)natom * 3 + i];
    for (int i = 0; i < 3 * natom; i++) F[i] = (double)(Facc[i] * (long double)dV);
    free(Fthr);
    free(Facc);
    free(gstart);
    return used;
}
