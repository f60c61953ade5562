/*
 * gint.h -- C ABI of the B200-native gint_vlocal library (libgint_b200.so).
 *
 * The library builds the local-potential Hamiltonian of NAO-based (RT-TD)DFT on
 * a uniform real-space mesh,
 *
 *   H_mu,nu(R) = sum_g phi_mu(r_g - tau_I) V(r_g) phi_nu(r_g - tau_J - R) dV
 *                                   -- PAPER.md:393-398 (Sec. 3.3.1, Eq. 45)
 *   phi_mu(r)  = f_{I,l,zeta}(|r|) Y_lm(r/|r|)
 *                                   -- PAPER.md:66-70 (Sec. 2.1, Eq. 1)
 *
 * with R the lattice vector from the cell of mu (atom I) to the cell of nu
 * (atom J) -- PAPER.md:104-106 -- and the result stored as dense blocks per
 * (I, J, R).  gint_setup plays the role of the paper's GintInfo initialisation
 * (mesh -> BigGrid partition -> per-BigGrid atom lists; Fig. 2 at
 * PAPER.md:368); gint_vlocal is the paper's cal_gint_vl.
 *
 * Conventions:
 *   - Units bohr / Hartree, FP64 only, real V, one spin channel.
 *   - Mesh point (i,j,k) sits at (i/N1) a1 + (j/N2) a2 + (k/N3) a3; dV = |det A|/(N1 N2 N3).
 *   - The sum over g runs over all space with V periodic on the mesh.
 *   - Radial part: 4-point (cubic) Lagrange interpolation of the table on the
 *     forward stencil k..k+3, k = floor(r/dr); phi = 0 iff r >= rcut.
 *   - Real Y_lm, l <= 3, no Condon-Shortley phase, with (x,y,z) = r/|r|:
 *       l=0: 1/(2 sqrt(pi));   l=1: sqrt(3/4pi) * {y, z, x};
 *       l=2: {1/2 sqrt(15/pi) xy, 1/2 sqrt(15/pi) yz, 1/4 sqrt(5/pi) (3z^2-1),
 *             1/2 sqrt(15/pi) xz, 1/4 sqrt(15/pi) (x^2-y^2)};
 *       l=3: {1/4 sqrt(35/2pi) y(3x^2-y^2), 1/2 sqrt(105/pi) xyz, 1/4 sqrt(21/2pi) y(5z^2-1), 1/4 sqrt(7/pi) z(5z^2-3),
 *             1/4 sqrt(21/2pi) x(5z^2-1), 1/4 sqrt(105/pi) z(x^2-y^2), 1/4 sqrt(35/2pi) x(x^2-3y^2)}.
 *     For |r| < 1e-12 bohr the l>0 components are 0.
 *   - Orbital order inside an atom: radial functions in the order given, each
 *     followed by its 2l+1 m-components in the order above.
 *   - Block set: every (I,J,R) with |tau_J + R - tau_I| < rcut_I + rcut_J
 *     (strict), both (I,J,R) and (J,I,-R) stored, sorted lexicographically by
 *     (I, J, R1, R2, R3); block = row-major n_I x n_J (rows: orbitals of I);
 *     blocks are packed back to back (offset = prefix sum of n_I*n_J).
 *   - Atom positions are used as given (never wrapped into the cell); R labels are
 *     relative to them.
 *
 * Pointers are HOST pointers unless the name ends in _dev.  All calls return 0
 * (GINT_OK) or a negative error code; nothing throws or aborts across this
 * boundary.  A gint_ctx may be used from one thread at a time.
 */
#ifndef GINT_B200_H
#define GINT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GINT_OK 0
#define GINT_EINVAL (-1)       /* null pointer, bad shape, non-positive size, table too short, singular lattice */
#define GINT_EUNSUPPORTED (-2) /* l > 3, too many orbitals per atom, H too large for 32-bit block offsets */
#define GINT_ENOMEM (-3)       /* host or device allocation failed */
#define GINT_ECUDA (-4)        /* CUDA runtime error; text via gint_last_error() */
#define GINT_ENODEVICE (-5)    /* call needs a device but the context was created host-only (cuda_device < 0) */

typedef struct gint_ctx gint_ctx; /* opaque; owns all host and device metadata */

/* One atomic species: nrad tabulated radial functions f(r), node k at r = k*dr.
 * Requirements: dr > 0, rcut > 0, ntab*dr >= rcut + 3*dr (the forward stencil may
 * read three nodes past floor(rcut/dr)); 0 <= l[k] <= 3; nrad <= 8; sum(2l+1) <= 64.
 * The arrays are copied during gint_setup and not retained. */
typedef struct {
    double rcut;         /* phi == 0 for r >= rcut (bohr)                          */
    double dr;           /* radial table step (bohr)                               */
    int32_t ntab;        /* nodes per table                                        */
    int32_t nrad;        /* number of radial functions                             */
    const int32_t *l;    /* [nrad] angular momentum of each radial function        */
    const double *table; /* [nrad][ntab], row-major                                */
} gint_species;

/* Tuning / sharding options; pass NULL for the defaults. */
typedef struct {
    int32_t bcell[3]; /* big-cell edge in mesh points ("BigGrid"); 0 -> the largest of 8, 6, 4 that
                         divides N (8 otherwise).  Need not divide N; clamped to N; product <= 512, edge <= 255. */
    int32_t rank;     /* this process' share of the big cells: cells with                                   */
    int32_t nranks;   /*   (cell index along a1) % nranks == rank are integrated; 0/1 -> all (single GPU)  */
    int64_t scratch_max_bytes; /* upper bound for the psi scratch buffer (0 -> 16 GiB).  When all regions do not fit,
                         consecutive batches of regions reuse the buffer (each call then runs its psi and contraction
                         kernels once per batch; results are the same); never smaller than one region needs.      */
} gint_options;

/* Build the context: validate, enumerate (I,J,R) blocks, partition the mesh into
 * big cells, build the per-cell (atom, image) lists and the work queue, upload.
 *   lattice[9]        rows a1, a2, a3 (Cartesian, bohr); any non-singular cell
 *   ngrid[3]          N1, N2, N3 > 0
 *   atom_species[natom], atom_pos[natom][3] (Cartesian)
 *   cuda_device       >= 0: device ordinal; < 0: host-only context (no CUDA call is
 *                     made; block table and statistics can be queried, gint_vlocal
 *                     returns GINT_ENODEVICE)
 * The host plan is built with std::thread workers (hardware_concurrency, at most 32; the environment variable
 * GINT_SETUP_THREADS overrides the count; the result does not depend on it).
 * On failure *out is NULL. */
int gint_setup(gint_ctx **out, const double *lattice, const int32_t *ngrid, int32_t nspecies,
               const gint_species *species, int32_t natom, const int32_t *atom_species, const double *atom_pos,
               int32_t cuda_device, const gint_options *opt);

/* New atom positions for an existing context (Ehrenfest dynamics moves the nuclei every step, PAPER.md:220-222,
 * Eq. 42 at PAPER.md:326): rebuilds the big-cell lists, the block table and the work items for atom_pos
 * ([natom][3] Cartesian, bohr, host pointer; species, lattice, mesh, big-cell size and rank stay as given to
 * gint_setup) and replaces the context's device tables and scratch buffers.  The BLOCK TABLE MAY CHANGE (pairs move
 * in and out of range): query gint_num_blocks / gint_get_blocks again and size H, D accordingly.  Synchronises the
 * device first (calls in flight read the old tables).  On a plan error (GINT_EINVAL / GINT_EUNSUPPORTED) the context
 * is unchanged; on a CUDA error afterwards it is only good for gint_destroy. */
int gint_update_positions(gint_ctx *ctx, const double *atom_pos);

/* Number of H blocks and length of the H buffer in doubles. */
int gint_num_blocks(const gint_ctx *ctx, int64_t *nblocks, int64_t *h_len);

/* Block table: iat[nblocks], jat[nblocks], R[nblocks][3], offset[nblocks+1] (in
 * doubles).  Any output pointer may be NULL. */
int gint_get_blocks(const gint_ctx *ctx, int32_t *iat, int32_t *jat, int32_t *R, int64_t *offset);

/* H <- Eq. 45 for the potential V.
 *   V_dev   device pointer, [N1][N2][N3] doubles, third index fastest; read only
 *   H_dev   device pointer, h_len doubles; OVERWRITTEN (not accumulated into)
 *   stream  cudaStream_t (as void*), NULL = legacy default stream
 * Asynchronous: enqueues two memsets, the psi kernel, the contraction kernel and the
 * mirror kernel on `stream`; no host synchronisation, no allocation, no host<->device
 * copy.  The context owns a device scratch buffer for psi (stats[12] bytes; 8.5 GB for
 * the 512-atom Si-like workload; bounded by gint_options.scratch_max_bytes, stats[30] batches).
 * With nranks > 1 H holds this rank's partial sum (sum over ranks = full H).
 * Kernel faults surface at the caller's next synchronisation. */
int gint_vlocal(gint_ctx *ctx, const double *V_dev, double *H_dev, void *stream);

/* Convenience end-to-end call with HOST buffers: copies V to the device, runs
 * gint_vlocal, copies H back, synchronises.  V_host [N1][N2][N3], H_host [h_len]. */
int gint_vlocal_host(gint_ctx *ctx, const double *V_host, double *H_host);

/* Charge density on the mesh from density-matrix blocks (the paper's cal_gint_rho):
 *
 *   rho(r_g) = sum_{R,R'} sum_{mu,nu} rho_mu,nu(R) phi_mu(r_g - tau_I - R') phi_nu(r_g - tau_J - R - R')
 *                                                          -- PAPER.md:384-391 (Sec. 3.3.1, Eq. 44)
 *   D_dev    device pointer, h_len doubles: the blocks rho_mu,nu(I,J,R) in exactly the layout of H (every block of
 *            the table is used as given; no symmetry of D is assumed); read only
 *   rho_dev  device pointer, [N1][N2][N3] doubles; OVERWRITTEN
 * Asynchronous on `stream` (two memsets, the psi kernel with unit weights and the contraction kernel in its density
 * mode, FP64 tensor pipe).  All calls on one context share its scratch buffers and work queue: they must be
 * stream-ordered with each other (same stream, or ordered by events).
 * With nranks > 1 rho holds this rank's partial sum. */
int gint_rho(gint_ctx *ctx, const double *D_dev, double *rho_dev, void *stream);

/* Local Pulay force (the paper's cal_gint_fvl):
 *
 *   F_I = - sum_R sum_{mu,nu} rho_nu,mu(R) sum_g [ d phi_mu(r_g - tau_I)/d tau_I  V(r_g) phi_nu(r_g - tau_J - R)
 *                                                + phi_mu(r_g - tau_I) V(r_g) d phi_nu(r_g - tau_J - R)/d tau_I ] dV
 *                                                          -- PAPER.md:400-411 (Sec. 3.3.1, Eq. 46)
 * read as F_K = - sum_blocks sum_{mu,nu} D(I,J,R)[mu][nu] dH(I,J,R)[mu][nu]/d tau_K at fixed V and D (the derivative
 * acts on phi_mu for K = I and on phi_nu for K = J), all-space mesh sum as for gint_vlocal.  Radial derivative: the
 * derivative of the same cubic Lagrange interpolant that defines the radial function ("numerically for the radial
 * part"), angular part analytic.  At r < 1e-12: grad phi = f'(0) c_1 e_m for l = 1, 0 otherwise.
 *   V_dev   device pointer, [N1][N2][N3] doubles; read only
 *   D_dev   device pointer, h_len doubles: density-matrix blocks in the layout of H (no symmetry assumed); read only
 *   F_dev   device pointer, [natom][3] doubles (Hartree / bohr, Cartesian); OVERWRITTEN
 * Asynchronous on `stream`: psi kernel (unit weights), E = D + D^T gather, T = E Phi on the FP64 tensor pipe, force
 * kernel.  The first call allocates two more scratch buffers (8 (32 ngroup)^2 bytes per region and one as large as
 * the psi scratch) and may return GINT_ENOMEM; later calls allocate nothing.  Same stream-ordering rule as gint_rho.
 * With nranks > 1 F holds this rank's partial sum. */
int gint_fvl(gint_ctx *ctx, const double *V_dev, const double *D_dev, double *F_dev, void *stream);

/* k-space assembly of the real-space blocks (the next step of the paper's workflow after cal_gint_vl):
 *
 *   H_mu,nu(k) = sum_R exp(i k.R) H_mu,nu(R)              -- PAPER.md:92-95 (Sec. 2.1, Eq. 5)
 *
 * with k = kfrac[0] b1 + kfrac[1] b2 + kfrac[2] b3, a_i . b_j = 2 pi delta_ij (so k.R = 2 pi kfrac . (R1,R2,R3)).
 *   H_dev    device pointer, h_len doubles as written by gint_vlocal; read only
 *   kfrac    HOST pointer, 3 doubles
 *   Hk_dev   device pointer, [norb_tot][norb_tot] complex numbers as interleaved (re, im) doubles, row-major;
 *            rows: orbitals of atom I (atoms in input order), columns: orbitals of atom J; OVERWRITTEN
 * Asynchronous on `stream` (two kernels: the phases exp(i k.R) of all blocks into a scratch array the context
 * owns, then one pass that writes every element of H(k) once).  gint_num_orbitals returns norb_tot and, if `first`
 * is not NULL, first[natom+1] = the first row/column of every atom (first[natom] = norb_tot). */
int gint_num_orbitals(const gint_ctx *ctx, int64_t *norb_tot, int64_t *first);
int gint_fold_k(gint_ctx *ctx, const double *H_dev, const double *kfrac, double *Hk_dev, void *stream);

/* gint_fold_k for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same result (Eq. 5), same two kernels, but the phase scratch is
 * a fixed array inside the library -- a file-scope `static __device__` array of gint_fold_k_static_max_blocks() =
 * 262144 entries x 16 bytes = 4 MiB that every GPU loading the library holds until the process exits -- instead of
 * memory the context allocated.  Its device address is resolved once per device at gint_setup
 * (cudaGetSymbolAddress); the call itself runs no cudaMalloc, cudaFree or allocating library routine.
 *   - a context with more blocks than the maximum: GINT_EUNSUPPORTED, nothing launched (use gint_fold_k);
 *   - nothing in the array has to start at zero: the first kernel rewrites entries 0 .. nblk-1, the second reads only
 *     those, on the same stream;
 *   - ALL contexts of a device share the array and it keeps the last call's contents: calls that can overlap on the
 *     GPU (different streams, or different contexts on one device) race on it -- keep them on one stream or order
 *     them with events.  gint_fold_k has no such restriction between contexts. */
int64_t gint_fold_k_static_max_blocks(void);
int gint_fold_k_static(gint_ctx *ctx, const double *H_dev, const double *kfrac, double *Hk_dev, void *stream);

/* Spherical-grid integration of the velocity-gauge nonlocal overlaps (the paper's snap_psibeta, independent of the
 * uniform mesh) -- PAPER.md:415-426 (Sec. 3.3.2, Eq. 47):
 *
 *   S(I, J, R)[mu][b] = < phi_mu(r - tau_J - R) | exp(-i A.r) | beta_b(r - tau_I) >
 *     = sum_i sum_a  rad_w[i] rb r_i^2  ang_w[a]  phi_mu(tau_I + r_i n_a - tau_J - R)
 *                    exp(-i A.(tau_I + r_i n_a))  beta_b(r_i n_a),       r_i = rad_x[i] rb,  n_a = ang_xyz[a]
 *
 * for every atom I whose species has projectors and every orbital-carrying image (J, R) with
 * |tau_J + R - tau_I| < rb_I + rc_J (strict).  Readings of the paper: r is the absolute Cartesian position with the
 * atoms where the caller put them (never wrapped); phi is real, so the bra needs no conjugate; a projector
 * beta_{l m zeta}(r) = b_{l zeta}(|r|) Y_lm(r/|r|) is tabulated and interpolated exactly like an orbital (same
 * stencil, cutoff rule, r -> 0 rule and real Y_lm as above); the quadrature is centred on atom I, radial nodes from a
 * rule on (0, 1) scaled by the projector cutoff rb of I's species (the paper: 140-point Gauss-Legendre), angular
 * nodes on the unit sphere with weights summing to 4 pi (the paper: 110-point Lebedev-Laikov).  The tables are the
 * caller's: the library does not generate quadrature rules.
 *
 * gint_snap_setup   proj[nspecies]: the projectors of each species in the gint_species layout (nrad = 0: the species
 *                   hosts none; nrad <= 8, l <= 3, at most 16 components per species; at most 32 orbitals per atom on
 *                   the orbital side: GINT_EUNSUPPORTED beyond); rad_x[nrad_pts], rad_w[nrad_pts], ang_xyz[nang][3],
 *                   ang_w[nang]: HOST arrays, copied.  Builds the pair list for the context's current positions and
 *                   uploads the tables; may be called again (new projectors or rules).  gint_update_positions
 *                   discards the pair list: call gint_snap_setup again afterwards.  Works on a host-only context
 *                   too (pair list only; gint_snap_psibeta then returns GINT_ENODEVICE).
 * gint_snap_num_pairs / gint_snap_get_pairs   the pairs sorted by (I, J, R1, R2, R3): iat[n], jat[n], R[n][3],
 *                   offset[n+1] in COMPLEX elements; block b is [n_J][m_I] row-major (rows: orbitals of J in block
 *                   order, columns: projector components of I, radial functions in the order given, m = -l..l).
 * gint_snap_psibeta A: HOST pointer, 3 doubles (bohr^-1); S_dev: device pointer, 2 s_len doubles, interleaved
 *                   (re, im); OVERWRITTEN, every element written once.  Asynchronous on `stream`, one kernel (one
 *                   CTA per two pairs of an atom I, the sum over points on the FP64 tensor pipe), no atomics: results
 *                   are bit-wise reproducible.  Allocates nothing.
 * With gint_options.nranks > 1 the pairs are independent problems dealt out by projector atom: a context keeps the
 * pairs of the atoms I with I % nranks == rank (its pair list and S cover those only; no collective is involved, the
 * caller gathers the blocks if it needs them in one place). */
int gint_snap_setup(gint_ctx *ctx, const gint_species *proj, int32_t nrad_pts, const double *rad_x, const double *rad_w,
                    int32_t nang, const double *ang_xyz, const double *ang_w);
int gint_snap_num_pairs(const gint_ctx *ctx, int64_t *npair, int64_t *s_len);
int gint_snap_get_pairs(const gint_ctx *ctx, int32_t *iat, int32_t *jat, int32_t *R, int64_t *offset);
int gint_snap_psibeta(gint_ctx *ctx, const double *A, double *S_dev, void *stream);

/* Per-kernel timing on the launch stream.  After gint_set_profiling(ctx, 1) every
 * gint_vlocal call records CUDA events around its kernels on `stream`;
 * gint_get_kernel_ms synchronises on the last call's events and returns durations in
 * milliseconds: ms[0] contraction kernel, ms[1] mirror kernel, ms[2] whole call incl. the
 * memsets, ms[3] psi (orbital evaluation) kernel.  Used by bench.py for the roofline's
 * per-launch duration.  With several batches (stats[30] > 1) ms[0] is the last batch's contraction and ms[3]
 * everything between the first psi kernel and it; ms[2] is always the whole call. */
int gint_set_profiling(gint_ctx *ctx, int32_t on);
int gint_get_kernel_ms(gint_ctx *ctx, double *ms /* [4] */);

/* Statistics of the setup (all host-side, valid for host-only contexts too).
 * stats[0] big cells (regions) total, empty ones included      stats[1] work items
 * stats[2] (atom image, region) list entries                   stats[3] max orbitals listed for one region
 * stats[4] executed tensor flops (512 per DMMA.8x8x4 the kernel will issue)
 * stats[5] accumulator elements flushed (upper bound on red.global.add.f64 per call)
 * stats[6] dynamic shared memory per CTA (bytes)
 * stats[7] number of kernels launched per gint_vlocal call (memsets not counted)
 * stats[8] F_pt = sum_g 2 n(g)^2, n(g) = orbitals non-zero at mesh point g (useful flops, no symmetry)
 * stats[9] F_sym = sum_g n(g) (n(g)+1) (useful flops when H(R)=H(-R)^T is exploited)
 * stats[10] in-sphere (atom image, point) pairs   stats[11] (atom image, point) pairs evaluated per call
 * stats[12] psi scratch buffer (bytes, device)    stats[13] psi bytes streamed back from L2 per call
 * stats[14] 8 KB chunk buffers of the shared-memory ring    stats[15] non-empty regions
 * stats[16..22] k-step / balance statistics of the plan, stats[23..25] big-cell edge actually used,
 * stats[26..29] DMMAs by code path of the contraction kernel (diagonal runs, all-row runs, other) and number of runs
 * stats[30] batches of regions that share the psi scratch (1 unless scratch_max_bytes forces more)
 * Returns the number of entries written (<= n, at most 32). */
int gint_get_stats(const gint_ctx *ctx, double *stats, int32_t n);

/* Copy out the per-cell lists (host logic tests).  cell_start[ncell+1] indexes
 * entry_atom[nentry] / entry_R[nentry][3]; cells are numbered (c1*nc2 + c2)*nc3 + c3.
 * Call with all pointers NULL to get ncell and nentry only. */
int gint_get_cell_lists(const gint_ctx *ctx, int64_t *ncell, int64_t *nentry, int64_t *cell_start,
                        int32_t *entry_atom, int32_t *entry_R);

/* Measure the sustained FP64 tensor-core (DMMA.8x8x4) rate of the current device with
 * a register-resident kernel: the "FP64 tensor peak" of the roofline.  Returns
 * TFLOP/s in *tflops. */
int gint_measure_fp64_peak(int32_t cuda_device, double seconds, double *tflops);

int gint_destroy(gint_ctx *ctx);

/* Text for an error code; gint_last_error() returns the detail of the last
 * failure in this thread (e.g. the CUDA error string). */
const char *gint_strerror(int code);
const char *gint_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GINT_B200_H */
