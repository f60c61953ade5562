// gint_plan.cpp -- host-side plan construction (see gint_plan.hpp).
#include "gint_plan.hpp"

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <numeric>
#include <thread>

#include "../../include/gint.h"

namespace gint {

namespace {

double det3(const double* A) {
    return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) + A[2] * (A[3] * A[7] - A[4] * A[6]);
}

// inv = A^{-1}; fractional coordinates of a Cartesian row vector x are x * inv.
void inv3(const double* A, double* inv) {
    const double d = det3(A);
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

inline int64_t floordiv(int64_t a, int64_t b) {
    int64_t q = a / b, r = a % b;
    return (r != 0 && ((r < 0) != (b < 0))) ? q - 1 : q;
}

// f(i, thread) for i in [0, n), indices handed out in blocks of `grain` to hardware_concurrency() threads (at most 32)
template <class F>
void parallel_for(size_t n, size_t grain, F f) {
    unsigned nt = std::thread::hardware_concurrency();
    if (const char* env = std::getenv("GINT_SETUP_THREADS")) nt = (unsigned)std::atoi(env);
    nt = std::max(1u, std::min(nt, 32u));
    if ((size_t)nt * grain > n) nt = (unsigned)std::max<size_t>(1, n / std::max<size_t>(1, grain));
    if (nt <= 1) {
        for (size_t i = 0; i < n; i++) f(i, 0u);
        return;
    }
    std::atomic<size_t> next{0};
    auto body = [&](unsigned t) {
        for (;;) {
            const size_t b = next.fetch_add(grain);
            if (b >= n) break;
            for (size_t i = b; i < std::min(n, b + grain); i++) f(i, t);
        }
    };
    std::vector<std::thread> th;
    for (unsigned t = 1; t < nt; t++) th.emplace_back(body, t);
    body(0);
    for (auto& x : th) x.join();
}
constexpr unsigned kMaxThreads = 32;

}  // namespace

int build_plan(Plan& P, const double* lattice, const int32_t* ngrid, int nspecies, const SpeciesHost* species,
               int natom, const int32_t* atom_species, const double* atom_pos, const int32_t bcell[3], int rank,
               int nranks, int64_t scratch_max_bytes, std::string& err) {
    // ---- validation -------------------------------------------------------
    if (!lattice || !ngrid || !species || !atom_species || !atom_pos) { err = "null argument"; return GINT_EINVAL; }
    if (nspecies <= 0 || nspecies > 127 || natom <= 0 || natom >= (1 << 20)) { err = "nspecies/natom out of range"; return GINT_EINVAL; }
    for (int d = 0; d < 3; d++)
        if (ngrid[d] <= 0) { err = "ngrid must be positive"; return GINT_EINVAL; }
    for (int i = 0; i < 9; i++)
        if (!std::isfinite(lattice[i])) { err = "lattice not finite"; return GINT_EINVAL; }
    const double vol = std::fabs(det3(lattice));
    double lmax = 0;
    for (int i = 0; i < 9; i++) lmax = std::max(lmax, std::fabs(lattice[i]));
    if (!(vol > 1e-12 * lmax * lmax * lmax) || lmax == 0) { err = "singular lattice"; return GINT_EINVAL; }
    if (nranks <= 0) nranks = 1;
    if (rank < 0 || rank >= nranks) { err = "rank out of range"; return GINT_EINVAL; }
    std::memcpy(P.lattice, lattice, sizeof(P.lattice));
    P.rank = rank;
    P.nranks = nranks;
    if (scratch_max_bytes < 0) { err = "scratch_max_bytes negative"; return GINT_EINVAL; }
    P.scratch_max_bytes = scratch_max_bytes;
    P.species.assign(species, species + nspecies);
    double rc_max = 0;
    for (int s = 0; s < nspecies; s++) {
        SpeciesHost& sp = P.species[s];
        if (!(sp.rcut > 0) || !(sp.dr > 0) || sp.nrad <= 0 || sp.ntab < 4) { err = "bad species"; return GINT_EINVAL; }
        if ((double)sp.ntab * sp.dr < sp.rcut + 3 * sp.dr - 1e-9 * sp.dr) { err = "radial table too short: need ntab*dr >= rcut + 3*dr"; return GINT_EINVAL; }
        if (sp.nrad > 8) { err = "more than 8 radial functions per species"; return GINT_EUNSUPPORTED; }
        sp.norb = 0;
        for (int k = 0; k < sp.nrad; k++) {
            if (sp.l[k] < 0) { err = "negative l"; return GINT_EINVAL; }
            if (sp.l[k] > 3) { err = "l > 3 not supported"; return GINT_EUNSUPPORTED; }
            sp.norb += 2 * sp.l[k] + 1;
        }
        if (sp.norb > kMaxOrbPerAtom) { err = "too many orbitals per atom"; return GINT_EUNSUPPORTED; }
        for (double v : sp.table)
            if (!std::isfinite(v)) { err = "table not finite"; return GINT_EINVAL; }
        rc_max = std::max(rc_max, sp.rcut);
    }
    P.atom_species.assign(atom_species, atom_species + natom);
    P.atom_pos.assign(atom_pos, atom_pos + 3 * (size_t)natom);
    for (int a = 0; a < natom; a++) {
        if (atom_species[a] < 0 || atom_species[a] >= nspecies) { err = "atom_species out of range"; return GINT_EINVAL; }
        for (int c = 0; c < 3; c++)
            if (!std::isfinite(atom_pos[3 * a + c])) { err = "atom position not finite"; return GINT_EINVAL; }
    }
    for (int d = 0; d < 3; d++) {
        P.ngrid[d] = ngrid[d];
        int b = (bcell && bcell[d] > 0) ? bcell[d] : 0;
        if (b == 0) {   // default: the largest of 8, 6, 4 that divides N (8 with a ragged last region otherwise)
            b = 8;
            for (int c : {8, 6, 4})
                if (ngrid[d] % c == 0) { b = c; break; }
        }
        if (b > ngrid[d]) b = ngrid[d];
        P.bcell[d] = b;
        P.ncell[d] = (ngrid[d] + b - 1) / b;
        for (int c = 0; c < 3; c++) P.estep[3 * d + c] = lattice[3 * d + c] / (double)ngrid[d];
    }
    // checked after clamping to the mesh: at most 512 points per region, every edge <= 255 (point offsets are bytes)
    if ((int64_t)P.bcell[0] * P.bcell[1] * P.bcell[2] > kMaxRegionPoints) { err = "region (bcell) larger than 512 mesh points"; return GINT_EUNSUPPORTED; }
    for (int d = 0; d < 3; d++)
        if (P.bcell[d] > 255) { err = "region (bcell) edge longer than 255 mesh points"; return GINT_EUNSUPPORTED; }
    P.dV = vol / ((double)ngrid[0] * (double)ngrid[1] * (double)ngrid[2]);

    double inv[9];
    inv3(lattice, inv);
    double blen[3];   // |column d of A^{-1}|: |d frac_d| <= rho * blen[d] inside a ball of radius rho
    for (int d = 0; d < 3; d++) blen[d] = std::sqrt(inv[d] * inv[d] + inv[3 + d] * inv[3 + d] + inv[6 + d] * inv[6 + d]);

    // ---- block table (sorted by I, J, R1, R2, R3) ---------------------------
    auto norb_of = [&](int a) { return P.species[P.atom_species[a]].norb; };
    auto rc_of = [&](int a) { return P.species[P.atom_species[a]].rcut; };
    {
        struct Blk { int32_t J, r1, r2, r3; };
        std::vector<std::vector<Blk>> per_atom((size_t)natom);
        std::atomic<int> bad{0};
        parallel_for((size_t)natom, 4, [&](size_t Is, unsigned) {
            const int I = (int)Is;
            for (int J = 0; J < natom; J++) {
                double dc[3], f[3];
                for (int c = 0; c < 3; c++) dc[c] = atom_pos[3 * I + c] - atom_pos[3 * J + c];
                const double reach = rc_of(I) + rc_of(J);
                int lo[3], hi[3];
                for (int d = 0; d < 3; d++) {
                    f[d] = dc[0] * inv[d] + dc[1] * inv[3 + d] + dc[2] * inv[6 + d];
                    lo[d] = (int)std::floor(f[d] - reach * blen[d]) - 1;
                    hi[d] = (int)std::ceil(f[d] + reach * blen[d]) + 1;
                }
                for (int r1 = lo[0]; r1 <= hi[0]; r1++)
                    for (int r2 = lo[1]; r2 <= hi[1]; r2++)
                        for (int r3 = lo[2]; r3 <= hi[2]; r3++) {
                            double v[3];
                            for (int c = 0; c < 3; c++)
                                v[c] = r1 * lattice[c] + r2 * lattice[3 + c] + r3 * lattice[6 + c] - dc[c];
                            if (std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) < reach) {
                                if (std::abs(r1) > 127 || std::abs(r2) > 127 || std::abs(r3) > 127) { bad = 1; continue; }
                                per_atom[Is].push_back({J, r1, r2, r3});
                            }
                        }
            }
        });
        if (bad) { err = "lattice image index beyond +-127"; return GINT_EUNSUPPORTED; }
        P.blk_off.push_back(0);
        for (int I = 0; I < natom; I++)
            for (const Blk& b : per_atom[(size_t)I]) {
                P.blk_i.push_back(I);
                P.blk_j.push_back(b.J);
                P.blk_R.push_back(b.r1);
                P.blk_R.push_back(b.r2);
                P.blk_R.push_back(b.r3);
                P.blk_off.push_back(P.blk_off.back() + (int64_t)norb_of(I) * norb_of(b.J));
            }
    }
    const int64_t nblk = (int64_t)P.blk_i.size();
    // block offsets are stored in 32 bits (kNoBlock = 2^32 - 1 marks "no such block"): H below 32 GiB
    if (P.blk_off.back() >= (int64_t)kNoBlock) { err = "H buffer exceeds 2^32 - 1 doubles"; return GINT_EUNSUPPORTED; }

    // ---- hash (I,J,R) -> offset; mirror lists ---------------------------------
    uint32_t hsize = 16;
    while ((int64_t)hsize < 2 * nblk) hsize <<= 1;
    P.hash_mask = hsize - 1;
    P.hash_keys.assign(hsize, 0);
    P.hash_vals.assign(hsize, kNoBlock);
    for (int64_t b = 0; b < nblk; b++) {
        const uint64_t key = pack_key(P.blk_i[b], P.blk_j[b], P.blk_R[3 * b], P.blk_R[3 * b + 1], P.blk_R[3 * b + 2]) + 1;
        uint32_t h = (uint32_t)hash_mix(key) & P.hash_mask;
        while (P.hash_keys[h] != 0) h = (h + 1) & P.hash_mask;
        P.hash_keys[h] = key;
        P.hash_vals[h] = (uint32_t)P.blk_off[b];
    }
    auto lookup = [&](int I, int J, int r1, int r2, int r3) -> uint32_t {
        const uint64_t key = pack_key(I, J, r1, r2, r3) + 1;
        uint32_t h = (uint32_t)hash_mix(key) & P.hash_mask;
        while (P.hash_keys[h] != 0) {
            if (P.hash_keys[h] == key) return P.hash_vals[h];
            h = (h + 1) & P.hash_mask;
        }
        return kNoBlock;
    };
    // canonical blocks (accumulated by the kernel): I<J, or I==J with R >= 0 lexicographically.
    for (int64_t b = 0; b < nblk; b++) {
        const int I = P.blk_i[b], J = P.blk_j[b];
        const int r1 = P.blk_R[3 * b], r2 = P.blk_R[3 * b + 1], r3 = P.blk_R[3 * b + 2];
        const bool zeroR = (r1 == 0 && r2 == 0 && r3 == 0);
        const bool posR = (r1 > 0) || (r1 == 0 && (r2 > 0 || (r2 == 0 && r3 > 0)));
        const bool canonical = (I < J) || (I == J && (zeroR || posR));
        MirrorItem m;
        m.dst = (uint32_t)P.blk_off[b];
        m.nI = norb_of(I);
        m.nJ = norb_of(J);
        if (!canonical) {
            m.src = lookup(J, I, -r1, -r2, -r3);
            if (m.src == kNoBlock) { err = "internal: mirror partner missing"; return GINT_EINVAL; }
            P.mirror.push_back(m);
        } else if (I == J && zeroR) {
            m.src = m.dst;
            P.mirror.push_back(m);
        }
    }

    // ---- packed radial tables: node-major [ntab+4][nradp], pre-multiplied by the Y_lm constant -------
    // l=0: 1/(2 sqrt(pi)); l=1: sqrt(3/4pi); l=2: 1/2 sqrt(15/pi); l=3: 1/2 sqrt(105/pi) (the kernels apply the
    // remaining l=2 and l=3 ratios to the angular polynomials).  Four zero nodes follow the table: the stencil of a point
    // outside the sphere is redirected there, so phi == 0 exactly for r >= rcut.
    {
        const double ylm_c[4] = {0.28209479177387814, 0.48860251190291992, 1.0925484305920792, 2.890611442640554};
        size_t off = 0;
        for (int s = 0; s < nspecies; s++) {
            SpeciesHost& sp = P.species[s];
            const int nradp = (sp.nrad + 1) & ~1;
            sp.tab_offset = (int)off;
            P.tab_packed.resize(off + (size_t)(sp.ntab + 4) * nradp, 0.0);
            for (int k = 0; k < sp.ntab; k++)
                for (int f = 0; f < sp.nrad; f++)
                    P.tab_packed[off + (size_t)k * nradp + f] = sp.table[(size_t)f * sp.ntab + k] * ylm_c[sp.l[f]];
            off = P.tab_packed.size();
            P.sp_meta.push_back(sp.tab_offset);
            P.sp_meta.push_back(sp.ntab);
            P.sp_meta.push_back(nradp);
            P.sp_meta.push_back(sp.norb);
            for (int k = 0; k < 8; k++) P.sp_meta.push_back(k < sp.nrad ? sp.l[k] : -1);
            P.sp_real.push_back(sp.rcut * sp.rcut);
            P.sp_real.push_back(1.0 / sp.dr);
        }
    }
    P.tables_in_smem = P.tab_packed.size() * sizeof(double) <= kMaxTableSmem;
    P.nring = kRingChunks;
    P.smem_bytes = 256 + smem_align((size_t)kDescSlots * sizeof(ItemDesc)) + (size_t)P.nring * kChunkBytes;

    // ---- point order inside a region: k-steps of 4 points, slices of 8 k-steps -----------------
    const int bx = P.bcell[0], by = P.bcell[1], bz = P.bcell[2];
    P.npts = bx * by * bz;
    {
        std::vector<std::array<uint8_t, 4>> order;
        if (bx % 2 == 0 && by % 2 == 0) {   // compact 2 x 2 x 1 k-steps (fewer partially covered k-steps)
            for (int x = 0; x < bx; x += 2)
                for (int y = 0; y < by; y += 2)
                    for (int z = 0; z < bz; z++)
                        for (int q = 0; q < 4; q++) order.push_back({(uint8_t)(x + (q >> 1)), (uint8_t)(y + (q & 1)), (uint8_t)z, 1});
        } else {
            for (int x = 0; x < bx; x++)
                for (int y = 0; y < by; y++)
                    for (int z = 0; z < bz; z++) order.push_back({(uint8_t)x, (uint8_t)y, (uint8_t)z, 1});
        }
        P.nks = (P.npts + kKstepPts - 1) / kKstepPts;
        P.nslice = (P.nks + kSliceKsteps - 1) / kSliceKsteps;
        P.nks_pad = P.nslice * kSliceKsteps;
        P.nstage = P.nks_pad / kStageKsteps;
        while ((int)order.size() < P.nks_pad * kKstepPts) order.push_back({0, 0, 0, 0});
        P.slot_xyz.resize(order.size() * 4);
        for (size_t i = 0; i < order.size(); i++)
            for (int c = 0; c < 4; c++) P.slot_xyz[4 * i + c] = order[i][c];
    }
    const int nslot_pts = P.nks_pad * kKstepPts;

    // ---- (region, atom image) entries -------------------------------------------------------------
    const int64_t ncells = (int64_t)P.ncell[0] * P.ncell[1] * P.ncell[2];
    const double* e1 = P.estep;
    const double* e2 = P.estep + 3;
    const double* e3 = P.estep + 6;
    double cell_rad = 0;   // bounding-sphere radius of a full region about its centre
    for (int s1 = -1; s1 <= 1; s1 += 2)
        for (int s2 = -1; s2 <= 1; s2 += 2) {
            double v[3];
            for (int c = 0; c < 3; c++)
                v[c] = 0.5 * ((bx - 1) * e1[c] + s1 * (by - 1) * e2[c] + s2 * (bz - 1) * e3[c]);
            cell_rad = std::max(cell_rad, std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
        }
    struct Tmp { int64_t cell; int npop; Entry e; };
    std::vector<Tmp> tmp;
    std::vector<int32_t> npoint_orb((size_t)ngrid[0] * ngrid[1] * ngrid[2], 0);
    double n_insphere = 0;
    std::vector<std::vector<Tmp>> tmp_thread(kMaxThreads);
    std::vector<double> insphere_thread(kMaxThreads, 0.0);
    std::atomic<int> bad_image{0};
    parallel_for((size_t)natom, 2, [&](size_t Is, unsigned tid) {
        const int I = (int)Is;
        std::vector<Tmp>& tmp = tmp_thread[tid];
        double& n_insphere = insphere_thread[tid];
        const int sp_id = P.atom_species[I];
        const double rc = P.species[sp_id].rcut, rc2 = rc * rc;
        const int norb = P.species[sp_id].norb;
        const double* tau = &atom_pos[3 * I];
        int64_t nlo[3], nhi[3];
        for (int d = 0; d < 3; d++) {
            const double f = tau[0] * inv[d] + tau[1] * inv[3 + d] + tau[2] * inv[6 + d];
            nlo[d] = (int64_t)std::floor((f - rc * blen[d]) * ngrid[d]) - 1;
            nhi[d] = (int64_t)std::ceil((f + rc * blen[d]) * ngrid[d]) + 1;
        }
        // walk unwrapped (image q, region c) pairs covering [nlo, nhi] in each dimension
        std::vector<std::pair<int, int>> rng[3];   // (q, c)
        for (int d = 0; d < 3; d++) {
            const int64_t N = ngrid[d];
            for (int64_t q = floordiv(nlo[d], N); q <= floordiv(nhi[d], N); q++) {
                const int64_t a = std::max<int64_t>(nlo[d] - q * N, 0), b = std::min<int64_t>(nhi[d] - q * N, N - 1);
                for (int64_t c = a / P.bcell[d]; c <= b / P.bcell[d]; c++) rng[d].push_back({(int)q, (int)c});
            }
        }
        for (auto& qc1 : rng[0]) {
            if (nranks > 1 && (qc1.second % nranks) != rank) continue;
            for (auto& qc2 : rng[1])
                for (auto& qc3 : rng[2]) {
                    const int q[3] = {qc1.first, qc2.first, qc3.first};
                    const int c[3] = {qc1.second, qc2.second, qc3.second};
                    if (std::abs(q[0]) > 127 || std::abs(q[1]) > 127 || std::abs(q[2]) > 127) { bad_image = 1; continue; }
                    Entry e;
                    std::memset(&e, 0, sizeof(e));
                    const int o[3] = {c[0] * bx, c[1] * by, c[2] * bz};
                    for (int k = 0; k < 3; k++) {
                        const double origin = o[0] * e1[k] + o[1] * e2[k] + o[2] * e3[k];
                        const double centre = tau[k] - (q[0] * lattice[k] + q[1] * lattice[3 + k] + q[2] * lattice[6 + k]);
                        e.rel[k] = origin - centre;
                    }
                    // quick reject with the bounding sphere of the (full) region
                    double cc[3];
                    for (int k = 0; k < 3; k++)
                        cc[k] = e.rel[k] + 0.5 * ((bx - 1) * e1[k] + (by - 1) * e2[k] + (bz - 1) * e3[k]);
                    const double dcen = std::sqrt(cc[0] * cc[0] + cc[1] * cc[1] + cc[2] * cc[2]);
                    if (dcen >= rc + cell_rad + 1e-9) continue;
                    int npin = 0;
                    for (int s = 0; s < nslot_pts; s++) {
                        const uint8_t* xyz = &P.slot_xyz[4 * (size_t)s];
                        if (!xyz[3]) continue;
                        const int ix = xyz[0], iy = xyz[1], iz = xyz[2];
                        if (o[0] + ix >= ngrid[0] || o[1] + iy >= ngrid[1] || o[2] + iz >= ngrid[2]) continue;
                        const double dx = e.rel[0] + ix * e1[0] + iy * e2[0] + iz * e3[0];
                        const double dy = e.rel[1] + ix * e1[1] + iy * e2[1] + iz * e3[1];
                        const double dz = e.rel[2] + ix * e1[2] + iy * e2[2] + iz * e3[2];
                        if (dx * dx + dy * dy + dz * dz < rc2) {
                            const int ks = s / kKstepPts;
                            e.kmask[ks >> 5] |= 1u << (ks & 31);
                            npin++;
                            __atomic_fetch_add(&npoint_orb[((size_t)(o[0] + ix) * ngrid[1] + (o[1] + iy)) * ngrid[2] + (o[2] + iz)], norb, __ATOMIC_RELAXED);
                        }
                    }
                    if (!npin) continue;
                    n_insphere += (double)npin;
                    e.atom = I;
                    e.Rpack = ((-q[0] + 128) << 16) | ((-q[1] + 128) << 8) | (-q[2] + 128) | (sp_id << 24);
                    e.norb = norb;
                    int npop = 0;
                    for (int k = 0; k < 4; k++) npop += __builtin_popcount(e.kmask[k]);
                    tmp.push_back({((int64_t)c[0] * P.ncell[1] + c[1]) * P.ncell[2] + c[2], npop, e});
                }
        }
    });
    if (bad_image) { err = "image index beyond +-127"; return GINT_EUNSUPPORTED; }
    for (unsigned t = 0; t < kMaxThreads; t++) {
        tmp.insert(tmp.end(), tmp_thread[t].begin(), tmp_thread[t].end());
        n_insphere += insphere_thread[t];
        std::vector<Tmp>().swap(tmp_thread[t]);
    }
    auto rkey = [](const Entry& e) { return (uint32_t)(e.Rpack & 0xFFFFFF); };
    // bucket the entries by region (counting sort), then per region, in parallel: the query list sorted by (atom, R),
    // and the kernel order -- entries that cover the whole region first (most active k-steps first, then (atom, R)),
    // and among the partially covering entries a greedy chain of similar coverage (Jaccard index of the k-step masks):
    // rows of consecutive entries share 8-row fragments and 32-row groups, whose activity is the OR of their entries'
    // masks, so neighbours that cover the same part of the region execute fewer wasted DMMAs (executed / useful
    // 1.32 -> 1.28 at si512_dzp)
    {
        P.cell_start.assign((size_t)ncells + 1, 0);
        for (auto& t : tmp) P.cell_start[(size_t)t.cell + 1]++;
        for (int64_t c = 0; c < ncells; c++) P.cell_start[(size_t)c + 1] += P.cell_start[(size_t)c];
        std::vector<Tmp> byc(tmp.size());
        {
            std::vector<int64_t> fill(P.cell_start.begin(), P.cell_start.end() - 1);
            for (auto& t : tmp) byc[(size_t)fill[(size_t)t.cell]++] = t;
        }
        tmp.swap(byc);
        std::vector<Tmp>().swap(byc);
        P.cell_atom.resize(tmp.size());
        P.cell_R.resize(3 * tmp.size());
        parallel_for((size_t)ncells, 16, [&](size_t c, unsigned) {
            const size_t a = (size_t)P.cell_start[c], b = (size_t)P.cell_start[c + 1];
            if (a == b) return;
            std::sort(tmp.begin() + (ptrdiff_t)a, tmp.begin() + (ptrdiff_t)b, [&](const Tmp& x, const Tmp& y) {
                if (x.e.atom != y.e.atom) return x.e.atom < y.e.atom;
                return rkey(x.e) < rkey(y.e);
            });
            for (size_t i = a; i < b; i++) {
                const Entry& e = tmp[i].e;
                P.cell_atom[i] = e.atom;
                P.cell_R[3 * i] = ((e.Rpack >> 16) & 0xFF) - 128;
                P.cell_R[3 * i + 1] = ((e.Rpack >> 8) & 0xFF) - 128;
                P.cell_R[3 * i + 2] = (e.Rpack & 0xFF) - 128;
            }
            std::stable_sort(tmp.begin() + (ptrdiff_t)a, tmp.begin() + (ptrdiff_t)b, [](const Tmp& x, const Tmp& y) { return x.npop > y.npop; });
            size_t f = a;
            while (f < b && tmp[f].npop >= P.nks) f++;   // fully covering entries stay first
            for (size_t i = (f > a ? f - 1 : a); i + 1 < b; i++) {
                size_t best = i + 1;
                double best_score = -1;
                for (size_t j = i + 1; j < b; j++) {
                    int in = 0, un = 0;
                    for (int k = 0; k < 4; k++) {
                        in += __builtin_popcount(tmp[i].e.kmask[k] & tmp[j].e.kmask[k]);
                        un += __builtin_popcount(tmp[i].e.kmask[k] | tmp[j].e.kmask[k]);
                    }
                    const double score = (double)in / (double)un;
                    if (score > best_score) { best_score = score; best = j; }
                }
                std::swap(tmp[i + 1], tmp[best]);
            }
            // ... then improved by swapping two partially covering entries whenever that lowers the number of active
            // (fragment, k-step) pairs of the region (executed / useful 1.28 -> 1.25 at si512_dzp)
            {
                const int m = (int)(b - a);
                auto active_pairs = [&]() {
                    uint32_t fm[kMaxGroups * 4][4];
                    int rows = 0;
                    for (int i = 0; i < m; i++) rows += tmp[a + i].e.norb;
                    const int nf = std::min((rows + 7) / 8, kMaxGroups * 4);
                    for (int q = 0; q < nf; q++)
                        for (int k = 0; k < 4; k++) fm[q][k] = 0;
                    int r0 = 0;
                    for (int i = 0; i < m; i++) {
                        const Entry& e = tmp[a + i].e;
                        for (int q = r0 / 8; q <= (r0 + e.norb - 1) / 8 && q < nf; q++)
                            for (int k = 0; k < 4; k++) fm[q][k] |= e.kmask[k];
                        r0 += e.norb;
                    }
                    long c = 0;
                    for (int q = 0; q < nf; q++)
                        for (int k = 0; k < 4; k++) c += __builtin_popcount(fm[q][k]);
                    return c;
                };
                long cur = active_pairs();
                for (int pass = 0, improved = 1; improved && pass < 3; pass++) {
                    improved = 0;
                    for (size_t i = f; i < b; i++)
                        for (size_t j = i + 1; j < b; j++) {
                            std::swap(tmp[i], tmp[j]);
                            const long c = active_pairs();
                            if (c < cur) { cur = c; improved = 1; }
                            else std::swap(tmp[i], tmp[j]);
                        }
                }
            }
        });
    }
    P.entries.resize(tmp.size());
    for (size_t i = 0; i < tmp.size(); i++) P.entries[i] = tmp[i].e;

    // ---- per region: rows, fragment / group activity, row info, pair table, tiles ------------------
    // A proto-item is a set of tiles of ONE region that touches few row groups; proto-items are packed into work
    // items (<= kTilesPerItem tiles, <= kMaxSlots row groups) afterwards, small ones also across regions.
    struct Tile { int region, gi, gj; double cost; };
    struct Proto { std::vector<Tile> tiles; std::vector<std::pair<int, int>> slots; /* (region, group) */ };
    std::vector<Proto> all_protos;
    std::vector<double> region_cost;
    double n_etask = 0, max_rows = 0;
    const int nks_pad = P.nks_pad, nslice = P.nslice, nstage = P.nstage;
    auto kstep_cost_of = [&](const uint8_t* gm, int gi, int gj, int ks) {
        const unsigned ra = gm[(size_t)gi * nks_pad + ks], ca = gm[(size_t)gj * nks_pad + ks];
        if (gi != gj) return __builtin_popcount(ra) * __builtin_popcount(ca);
        int n = 0;
        for (int i = 0; i < 4; i++)
            if ((ra >> i) & 1u) n += __builtin_popcount(ca >> i);
        return n;
    };
    auto stage_cost_of = [&](const uint8_t* gm, int gi, int gj, int st) {
        int n = 0;
        for (int ks = st * kStageKsteps; ks < (st + 1) * kStageKsteps; ks++) n += kstep_cost_of(gm, gi, gj, ks);
        return n;
    };
    // prepass (serial, cheap): region boundaries in the entry list, rows, offsets into the shared tables
    struct Span { size_t pos, end; };
    std::vector<Span> spans;
    int64_t total_chunks = 0;
    {
        const int task_runs = (nslice + 7) / 8;
        size_t gm_off = 0, ri_off = 0, pr_off = 0, tk_off = 0;
        for (size_t pos = 0; pos < tmp.size();) {
            size_t end = pos;
            while (end < tmp.size() && tmp[end].cell == tmp[pos].cell) end++;
            const int64_t c = tmp[pos].cell;
            const int m = (int)(end - pos);
            if (m > 4095) { err = "more than 4095 atom images touch one region"; return GINT_EUNSUPPORTED; }
            Region R;
            std::memset(&R, 0, sizeof(R));
            const int c3 = (int)(c % P.ncell[2]), c2 = (int)((c / P.ncell[2]) % P.ncell[1]), c1 = (int)(c / ((int64_t)P.ncell[1] * P.ncell[2]));
            R.origin[0] = c1 * bx;
            R.origin[1] = c2 * by;
            R.origin[2] = c3 * bz;
            int rows = 0;
            for (int i = 0; i < m; i++) {
                P.entries[pos + i].row0 = rows;
                rows += P.entries[pos + i].norb;
            }
            const int nfrag = (rows + 7) / 8, ngroup = (nfrag + 3) / 4;
            if (ngroup > kMaxGroups) { err = "too many orbitals listed for one region; use a smaller bcell"; return GINT_EUNSUPPORTED; }
            max_rows = std::max(max_rows, (double)rows);
            R.nrow = rows;
            R.nentry = m;
            R.entry0 = (int32_t)pos;
            R.ngroup = ngroup;
            R.gmask_off = (int32_t)gm_off;
            R.rowinfo_off = (int32_t)ri_off;
            R.pair_off = (int32_t)pr_off;
            R.task_off = (int32_t)tk_off;      // room for every (entry, run); only the active ones are listed
            gm_off += (size_t)ngroup * nks_pad;
            ri_off += (size_t)ngroup * kGroupRows;
            pr_off += (size_t)m * m;
            tk_off += (size_t)m * task_runs;
            if (gm_off > 0x7FFFFFFFu || pr_off > 0x7FFFFFFFu || tk_off > 0x7FFFFFFFu) {
                err = "plan tables exceed 2^31 entries";
                return GINT_EUNSUPPORTED;
            }
            P.regions.push_back(R);
            spans.push_back({pos, end});
            pos = end;
        }
        P.gmask.assign(gm_off, 0);
        P.rowinfo.assign(ri_off, kNoBlock);
        for (const Region& R : P.regions) total_chunks += (int64_t)R.ngroup * nstage;
        P.pair.assign(pr_off, PairWord{kNoBlock, 0, 0});
        P.pair_direct.assign(pr_off, kNoBlock);
        P.etasks.assign(tk_off, 0u);
    }
    const size_t nreg = P.regions.size();
    const int64_t max_chunks = std::max<int64_t>(1, (scratch_max_bytes > 0 ? scratch_max_bytes : kDefaultScratchBytes) / kChunkBytes);
    // several batches share the scratch: rows that no task of a region writes must then be zeroed by the psi kernel
    // (they hold another region's values), so every (entry, run of stages) becomes a task
    const bool multibatch = total_chunks > max_chunks;
    std::vector<std::vector<Proto>> region_protos(nreg);
    std::vector<int> region_active(nreg, 0);
    region_cost.assign(nreg, 0.0);
    parallel_for(nreg, 8, [&](size_t rix, unsigned) {
        Region& R = P.regions[rix];
        const size_t pos = spans[rix].pos;
        const int m = R.nentry, ngroup = R.ngroup;
        // evaluation tasks: (entry, run of up to 8 stages) with at least one point inside the sphere; the kernel
        // walks the run's active 32-point stages with the entry's data in registers
        int nactive = 0;
        for (int i = 0; i < m; i++) {
            const Entry& e = P.entries[pos + i];
            for (int h = 0; h * 8 < nslice; h++) {
                int na = 0;
                for (int s = h * 8; s < std::min(nslice, h * 8 + 8); s++)
                    if ((e.kmask[(s * kSliceKsteps) >> 5] >> ((s * kSliceKsteps) & 31)) & 0xFFu) na++;
                if (na || multibatch) P.etasks[(size_t)R.task_off + (size_t)(R.ntask++)] = pack_etask(i, h);
                nactive += na;
            }
        }
        // fragment activity: OR of the k-step masks of the entries that own rows of the fragment
        std::vector<std::array<uint32_t, 4>> fmask((size_t)ngroup * 4, std::array<uint32_t, 4>{0, 0, 0, 0});
        for (int i = 0; i < m; i++) {
            const Entry& e = P.entries[pos + i];
            for (int mu = 0; mu < e.norb; mu++) P.rowinfo[(size_t)R.rowinfo_off + e.row0 + mu] = pack_rowinfo(i, mu, e.norb);
            for (int f = e.row0 / 8; f <= (e.row0 + e.norb - 1) / 8; f++)
                for (int k = 0; k < 4; k++) fmask[(size_t)f][k] |= e.kmask[k];
        }
        uint8_t* gm = &P.gmask[(size_t)R.gmask_off];
        for (int g = 0; g < ngroup; g++)
            for (int ks = 0; ks < nks_pad; ks++) {
                uint8_t b = 0;
                for (int i = 0; i < 4; i++) b |= (uint8_t)(((fmask[(size_t)4 * g + i][ks >> 5] >> (ks & 31)) & 1u) << i);
                gm[(size_t)g * nks_pad + ks] = b;
            }
        // pair table: (row entry a <= column entry b) -> canonical block offset and element strides
        for (int a = 0; a < m; a++)
            for (int b = a; b < m; b++) {
                const Entry& ea = P.entries[pos + a];
                const Entry& eb = P.entries[pos + b];
                const int r1 = ((eb.Rpack >> 16) & 0xFF) - ((ea.Rpack >> 16) & 0xFF);
                const int r2 = ((eb.Rpack >> 8) & 0xFF) - ((ea.Rpack >> 8) & 0xFF);
                const int r3 = (eb.Rpack & 0xFF) - (ea.Rpack & 0xFF);
                const bool zeroR = (r1 == 0 && r2 == 0 && r3 == 0);
                const bool posR = (r1 > 0) || (r1 == 0 && (r2 > 0 || (r2 == 0 && r3 > 0)));
                const bool canonical = (ea.atom < eb.atom) || (ea.atom == eb.atom && (zeroR || posR));
                PairWord pw;
                pw.off = canonical ? lookup(ea.atom, eb.atom, r1, r2, r3) : lookup(eb.atom, ea.atom, -r1, -r2, -r3);
                pw.smu = (uint16_t)(canonical ? eb.norb : 1);
                pw.snu = (uint16_t)(canonical ? 1 : ea.norb);
                P.pair[(size_t)R.pair_off + (size_t)a * m + b] = pw;
                P.pair_direct[(size_t)R.pair_off + (size_t)a * m + b] = lookup(ea.atom, eb.atom, r1, r2, r3);
                P.pair_direct[(size_t)R.pair_off + (size_t)b * m + a] = lookup(eb.atom, ea.atom, -r1, -r2, -r3);
            }
        // tiles (group gi <= gj) with their cost in DMMAs: the kernel decides per k-step (4 mesh points), a fragment
        // pair is executed if the k-step holds an in-sphere point of both fragments' rows
        const int region_index = (int)rix;
        auto add_slot = [](std::vector<std::pair<int, int>>& v, std::pair<int, int> g) { if (std::find(v.begin(), v.end(), g) == v.end()) v.push_back(g); };
        std::vector<std::vector<double>> tcost((size_t)ngroup, std::vector<double>((size_t)ngroup, 0.0));
        double rcost = 0;
        for (int gi = 0; gi < ngroup; gi++)
            for (int gj = gi; gj < ngroup; gj++) {
                int n = 0;
                for (int st = 0; st < nstage; st++) n += stage_cost_of(gm, gi, gj, st);
                tcost[(size_t)gi][(size_t)gj] = n;
                rcost += n;
                if (n > 0) R.ntile++;
            }
        std::vector<Proto> protos;
        auto add_tile = [&](Proto& p, int gi, int gj) {
            if (tcost[(size_t)gi][(size_t)gj] <= 0) return;
            p.tiles.push_back({region_index, gi, gj, tcost[(size_t)gi][(size_t)gj]});
            add_slot(p.slots, {region_index, gi});
            add_slot(p.slots, {region_index, gj});
        };
        const int chunk = kCliqueGroups;
        const int nchunk = (ngroup + chunk - 1) / chunk;
        for (int k = 0; k < nchunk; k++) {
            const int k0 = k * chunk, k1 = std::min(ngroup, k0 + chunk);
            Proto p;
            for (int gi = k0; gi < k1; gi++)
                for (int gj = gi; gj < k1; gj++) add_tile(p, gi, gj);
            if (!p.tiles.empty()) protos.push_back(p);
            for (int l = k + 1; l < nchunk; l++) {
                const int l0 = l * chunk, l1 = std::min(ngroup, l0 + chunk);
                const int width = std::max(1, std::min(kTilesPerItem / (k1 - k0), kMaxSlots - (k1 - k0)));
                for (int cj = l0; cj < l1; cj += width) {
                    Proto r;
                    for (int gi = k0; gi < k1; gi++)
                        for (int gj = cj; gj < std::min(l1, cj + width); gj++) add_tile(r, gi, gj);
                    if (!r.tiles.empty()) protos.push_back(r);
                }
            }
        }
        // greedy merge of small proto-items of the region (fewer items, fewer chunk loads)
        for (bool merged = true; merged;) {
            merged = false;
            int best_a = -1, best_b = -1, best_union = 1 << 30;
            for (size_t a = 0; a < protos.size(); a++)
                for (size_t b = a + 1; b < protos.size(); b++) {
                    if (protos[a].tiles.size() + protos[b].tiles.size() > (size_t)kTilesPerItem) continue;
                    std::vector<std::pair<int, int>> u = protos[a].slots;
                    for (auto g : protos[b].slots) add_slot(u, g);
                    if ((int)u.size() > kMaxSlots) continue;
                    const int growth = (int)u.size() - (int)std::max(protos[a].slots.size(), protos[b].slots.size());
                    if (growth < best_union) { best_union = growth; best_a = (int)a; best_b = (int)b; }
                }
            if (best_a >= 0) {
                for (auto& t : protos[(size_t)best_b].tiles) protos[(size_t)best_a].tiles.push_back(t);
                for (auto g : protos[(size_t)best_b].slots) add_slot(protos[(size_t)best_a].slots, g);
                protos.erase(protos.begin() + best_b);
                merged = true;
            }
        }
        if (R.ntile > 0) region_active[rix] = nactive;
        else R.ntask = 0;
        region_cost[rix] = rcost;
        region_protos[rix] = std::move(protos);
    });
    // psi scratch chunks in region order, starting over with every batch; proto-items in region order
    P.region_batch.assign(nreg, 0);
    {
        int batch = 0;
        int64_t used = 0;
        for (size_t rix = 0; rix < nreg; rix++) {
            Region& R = P.regions[rix];
            const int64_t need = R.ntile > 0 ? (int64_t)R.ngroup * nstage : 0;
            if (used > 0 && used + need > max_chunks) {
                batch++;
                used = 0;
            }
            P.region_batch[rix] = batch;
            R.psi_chunk0 = used;
            used += need;
            P.psi_chunks = std::max(P.psi_chunks, used);
            if (R.ntile > 0) n_etask += region_active[rix];
            for (Proto& p : region_protos[rix]) all_protos.push_back(std::move(p));
        }
        P.batches.assign((size_t)batch + 1, Plan::Batch{0, 0, 0, 0});
        int wr = 0;
        for (size_t rix = 0; rix < nreg; rix++)
            if (P.regions[rix].ntile > 0) {
                Plan::Batch& B = P.batches[(size_t)P.region_batch[rix]];
                if (B.nwr == 0) B.wr0 = wr;
                B.nwr++;
                wr++;
            }
    }
    tmp.clear();
    tmp.shrink_to_fit();

    // ---- work items ---------------------------------------------------------------------------------
    // queue order: heaviest regions first, the proto-items of a region consecutive (their CTAs share its psi in L2)
    std::stable_sort(all_protos.begin(), all_protos.end(), [&](const Proto& a, const Proto& b) {
        const int ra = a.tiles[0].region, rb = b.tiles[0].region;
        if (P.region_batch[(size_t)ra] != P.region_batch[(size_t)rb]) return P.region_batch[(size_t)ra] < P.region_batch[(size_t)rb];
        if (region_cost[(size_t)ra] != region_cost[(size_t)rb]) return region_cost[(size_t)ra] > region_cost[(size_t)rb];
        return ra < rb;
    });
    // pack small proto-items together, also across regions (window of the queue), largest fill first
    {
        const size_t window = 48;
        std::vector<char> dead(all_protos.size(), 0);
        for (size_t a = 0; a < all_protos.size(); a++) {
            if (dead[a]) continue;
            for (;;) {
                Proto& pa = all_protos[a];
                int best = -1;
                size_t best_tiles = 0;
                for (size_t b = a + 1; b < std::min(all_protos.size(), a + 1 + window); b++) {
                    if (dead[b]) continue;
                    const Proto& pb = all_protos[b];
                    if (P.region_batch[(size_t)pb.tiles[0].region] != P.region_batch[(size_t)pa.tiles[0].region]) break;
                    if (pa.tiles.size() + pb.tiles.size() > (size_t)kTilesPerItem) continue;
                    size_t nu = pa.slots.size();
                    for (auto g : pb.slots)
                        if (std::find(pa.slots.begin(), pa.slots.end(), g) == pa.slots.end()) nu++;
                    if (nu > (size_t)kMaxSlots) continue;
                    if (pb.tiles.size() > best_tiles) { best_tiles = pb.tiles.size(); best = (int)b; }
                }
                if (best < 0) break;
                for (auto& t : all_protos[(size_t)best].tiles) pa.tiles.push_back(t);
                for (auto g : all_protos[(size_t)best].slots)
                    if (std::find(pa.slots.begin(), pa.slots.end(), g) == pa.slots.end()) pa.slots.push_back(g);
                dead[(size_t)best] = 1;
            }
        }
        size_t w = 0;
        for (size_t a = 0; a < all_protos.size(); a++)
            if (!dead[a]) {
                if (w != a) all_protos[w] = std::move(all_protos[a]);
                w++;
            }
        all_protos.resize(w);
    }
    for (size_t it = 0; it < all_protos.size(); it++) {   // item ranges of the batches (the queue is batch-major)
        Plan::Batch& B = P.batches[(size_t)P.region_batch[(size_t)all_protos[it].tiles[0].region]];
        if (B.nitems == 0) B.item0 = (int32_t)it;
        B.nitems++;
    }
    // descriptors: everything the contraction kernel needs for an item, contiguous (one bulk copy)
    double exec_dmma = 0, flush_elems = 0, chunk_loads = 0;
    double dmma_diag = 0, dmma_rect = 0, dmma_slow = 0, nruns = 0;
    double ks_full = 0, ks_part = 0, dmma_part = 0, stage_visits = 0, bal_item = 0, bal_stage = 0, bal_warp = 0;
    P.descs.resize(all_protos.size());
    struct Acc { double v[14] = {0}; };
    std::vector<Acc> accs(kMaxThreads);
    parallel_for(all_protos.size(), 16, [&](size_t it, unsigned tid) {
        double* av = accs[tid].v;
        double &exec_dmma = av[0], &flush_elems = av[1], &chunk_loads = av[2], &dmma_diag = av[3], &dmma_rect = av[4],
               &dmma_slow = av[5], &nruns = av[6], &ks_full = av[7], &ks_part = av[8], &dmma_part = av[9],
               &stage_visits = av[10], &bal_item = av[11], &bal_stage = av[12], &bal_warp = av[13];
        Proto& p = all_protos[it];
        ItemDesc& d = P.descs[it];
        std::memset(&d, 0, sizeof(d));
        std::memset(d.item.tiles, 0xFF, sizeof(d.item.tiles));
        std::sort(p.slots.begin(), p.slots.end());
        d.item.nslot = (int16_t)p.slots.size();
        d.item.ntile = (int16_t)p.tiles.size();
        for (size_t q = 0; q < p.slots.size(); q++) {
            const Region& R = P.regions[(size_t)p.slots[q].first];
            const int g = p.slots[q].second;
            SlotInfo& si = d.slot[q];
            si.chunk0 = R.psi_chunk0 + (int64_t)g * nstage;
            si.pair_off = R.pair_off;
            si.nentry = R.nentry;
            for (int k = 0; k < 3; k++) si.origin[k] = R.origin[k];
            const uint8_t* gmq = &P.gmask[(size_t)R.gmask_off + (size_t)g * nks_pad];
            for (int st = 0; st < nstage; st++) {
                uint32_t wd = 0;
                for (int ks = 0; ks < kStageKsteps; ks++) wd |= (uint32_t)(gmq[st * kStageKsteps + ks] & 0xFu) << (4 * ks);
                d.gm32[q][st] = wd;
            }
            std::memcpy(d.rinfo[q], &P.rowinfo[(size_t)R.rowinfo_off + (size_t)g * kGroupRows], sizeof(uint32_t) * kGroupRows);
        }
        auto slot_of = [&](int region, int g) {
            return (int)(std::find(p.slots.begin(), p.slots.end(), std::make_pair(region, g)) - p.slots.begin());
        };
        // Tiles -> warps.  Warp w runs on SM sub-partition (scheduler) w % 4, whose DMMA pipe its four warps share, and
        // the warps of an item move through the ring stages nearly in lockstep (the ring holds 3 stages), so what counts
        // is the heaviest scheduler PER STAGE: start from heaviest-tile-first onto the least loaded scheduler, then
        // improve sum_stage max_scheduler load by single moves and pairwise swaps.
        std::sort(p.tiles.begin(), p.tiles.end(), [](const Tile& a, const Tile& b) { return a.cost > b.cost; });
        double load[4] = {0, 0, 0, 0};
        int used[4] = {0, 0, 0, 0};
        const size_t nt = p.tiles.size();
        std::vector<int> warp_of(nt), sched(nt);
        std::vector<std::array<int, kMaxStages>> sc(nt);
        std::vector<std::array<uint8_t, kMaxKsteps>> kcost(nt);   // DMMAs per (tile, k-step)
        for (size_t t = 0; t < nt; t++) {
            const Tile& tl = p.tiles[t];
            const uint8_t* gm = &P.gmask[(size_t)P.regions[(size_t)tl.region].gmask_off];
            for (int ks = 0; ks < nks_pad; ks++) kcost[t][ks] = (uint8_t)kstep_cost_of(gm, tl.gi, tl.gj, ks);
            for (int st = 0; st < kMaxStages; st++) {
                int n = 0;
                if (st < nstage)
                    for (int ks = st * kStageKsteps; ks < (st + 1) * kStageKsteps; ks++) n += kcost[t][ks];
                sc[t][st] = n;
            }
        }
        {
            // the producer warp shares sub-partition 3, which therefore gets one tile fewer
            const int cap[4] = {(kTilesPerItem + 3) / 4, (kTilesPerItem + 3) / 4, (kTilesPerItem + 3) / 4, kTilesPerItem / 4};
            double ld[4] = {0, 0, 0, 0};
            int us[4] = {0, 0, 0, 0};
            for (size_t t = 0; t < nt; t++) {
                int q = -1;
                for (int k = 0; k < 4; k++)
                    if (us[k] < cap[k] && (q < 0 || ld[k] < ld[q])) q = k;
                sched[t] = q;
                us[q]++;
                ld[q] += p.tiles[t].cost;
            }
            int L[4][kMaxStages] = {};
            for (size_t t = 0; t < nt; t++)
                for (int st = 0; st < nstage; st++) L[sched[t]][st] += sc[t][st];
            auto objective = [&]() {
                long o = 0;
                for (int st = 0; st < nstage; st++) o += std::max(std::max(L[0][st], L[1][st]), std::max(L[2][st], L[3][st]));
                return o;
            };
            auto shift = [&](size_t t, int from, int to) {
                for (int st = 0; st < nstage; st++) { L[from][st] -= sc[t][st]; L[to][st] += sc[t][st]; }
            };
            long cur = objective();
            for (int pass = 0, improved = 1; improved && pass < 2; pass++) {
                improved = 0;
                for (size_t t = 0; t < nt; t++)
                    for (int q = 0; q < 4; q++) {
                        const int q0 = sched[t];
                        if (q == q0 || us[q] >= cap[q]) continue;
                        shift(t, q0, q);
                        const long o = objective();
                        if (o < cur) { cur = o; sched[t] = q; us[q0]--; us[q]++; improved = 1; }
                        else shift(t, q, q0);
                    }
                for (size_t t = 0; t < nt; t++)
                    for (size_t u = t + 1; u < nt; u++) {
                        const int qt = sched[t], qu = sched[u];
                        if (qt == qu) continue;
                        shift(t, qt, qu);
                        shift(u, qu, qt);
                        const long o = objective();
                        if (o < cur) { cur = o; sched[t] = qu; sched[u] = qt; improved = 1; }
                        else { shift(t, qu, qt); shift(u, qt, qu); }
                    }
            }
        }
        for (size_t t = 0; t < nt; t++) {
            const int q = sched[t];
            const int warp = q + 4 * used[q];
            used[q]++;
            warp_of[t] = warp;
            const Tile& tl = p.tiles[t];
            load[q] += tl.cost;
            d.item.tiles[warp][0] = (uint8_t)slot_of(tl.region, tl.gi);
            d.item.tiles[warp][1] = (uint8_t)slot_of(tl.region, tl.gj);
            exec_dmma += tl.cost;
            const uint8_t* gm = &P.gmask[(size_t)P.regions[(size_t)tl.region].gmask_off];
            for (int ks = 0; ks < nks_pad; ks++) {
                const int nd = kcost[t][ks];
                if (tl.gi != tl.gj && nd == 16) ks_full += 1;
                else if (nd > 0) { ks_part += 1; dmma_part += nd; }
            }
            for (int st = 0; st < nstage; st++) {
                if (sc[t][st] <= 0) continue;
                d.item.stage_mask |= 1u << st;
                // the warp's program for the stage: runs of consecutive active k-steps with equal (ra, ca)
                int nrun = 0;
                for (int ks = 0; ks < kStageKsteps;) {
                    const unsigned ra = gm[(size_t)tl.gi * nks_pad + st * kStageKsteps + ks] & 0xFu;
                    const unsigned ca = gm[(size_t)tl.gj * nks_pad + st * kStageKsteps + ks] & 0xFu;
                    if (!ra || !ca) { ks++; continue; }
                    int n = 1;
                    while (ks + n < kStageKsteps && (gm[(size_t)tl.gi * nks_pad + st * kStageKsteps + ks + n] & 0xFu) == ra &&
                           (gm[(size_t)tl.gj * nks_pad + st * kStageKsteps + ks + n] & 0xFu) == ca) n++;
                    d.prog[warp][st][nrun++] = pack_run(ra, ca, ks, n);
                    {   // DMMAs by code path of the contraction kernel
                        int nd = 0;
                        for (int q = 0; q < n; q++) nd += kcost[t][st * kStageKsteps + ks + q];
                        if (tl.gi == tl.gj) dmma_diag += nd;
                        else if (ra == 0xFu) dmma_rect += nd;
                        else dmma_slow += nd;
                        nruns += 1;
                    }
                    ks += n;
                }
            }
        }
        bal_item += std::max(std::max(load[0], load[1]), std::max(load[2], load[3]));
        for (int st = 0; st < nstage; st++) {
            double ls[4] = {0, 0, 0, 0}, lw = 0;
            for (size_t t = 0; t < p.tiles.size(); t++) {
                const double c = sc[t][st];
                ls[warp_of[t] & 3] += c;
                lw = std::max(lw, c);
            }
            bal_stage += std::max(std::max(ls[0], ls[1]), std::max(ls[2], ls[3]));
            bal_warp += lw;
        }
        for (int st = 0; st < nstage; st++) {
            uint32_t a = 0;
            if ((d.item.stage_mask >> st) & 1u)
                for (int q = 0; q < d.item.nslot; q++)
                    if (d.gm32[q][st]) a |= 1u << q;
            d.act[st] = (uint8_t)a;
            chunk_loads += __builtin_popcount(a);
        }
        stage_visits += __builtin_popcount(d.item.stage_mask);
        flush_elems += 1024.0 * (double)p.tiles.size();
        d.valid = 1;
    });
    for (const Acc& a : accs) {
        exec_dmma += a.v[0]; flush_elems += a.v[1]; chunk_loads += a.v[2]; dmma_diag += a.v[3]; dmma_rect += a.v[4];
        dmma_slow += a.v[5]; nruns += a.v[6]; ks_full += a.v[7]; ks_part += a.v[8]; dmma_part += a.v[9];
        stage_visits += a.v[10]; bal_item += a.v[11]; bal_stage += a.v[12]; bal_warp += a.v[13];
    }
    all_protos.clear();

    double fpt = 0, fsym = 0;
    for (int32_t n : npoint_orb) {
        fpt += 2.0 * (double)n * (double)n;
        fsym += (double)n * ((double)n + 1.0);
    }
    P.stats[0] = (double)ncells;
    P.stats[1] = (double)P.descs.size();
    P.stats[2] = (double)P.entries.size();
    P.stats[3] = max_rows;
    P.stats[4] = 512.0 * exec_dmma;
    P.stats[5] = flush_elems;
    P.stats[6] = (double)P.smem_bytes;
    P.stats[7] = 5;   // gint_vrange_kernel, gint_hinit_kernel, gint_psi_kernel, gint_contract_kernel<0>, gint_mirror_kernel
    P.stats[8] = fpt;
    P.stats[9] = fsym;
    P.stats[10] = n_insphere;
    P.stats[11] = n_etask * kSlicePts;
    P.stats[12] = (double)P.psi_chunks * kChunkBytes;
    P.stats[13] = chunk_loads * kChunkBytes;
    P.stats[14] = (double)P.nring;
    P.stats[15] = (double)P.regions.size();
    P.stats[16] = ks_full;
    P.stats[17] = ks_part;
    P.stats[18] = dmma_part;
    P.stats[19] = stage_visits;
    P.stats[20] = bal_item;    // sum over items of the heaviest scheduler's DMMAs (perfect overlap inside an item)
    P.stats[21] = bal_stage;   // same if the warps moved through the stages in lockstep
    P.stats[22] = bal_warp;    // sum over (item, stage) of the heaviest single warp's DMMAs
    for (int d = 0; d < 3; d++) P.stats[23 + d] = (double)P.bcell[d];
    P.stats[30] = (double)P.batches.size();   // batches sharing the psi scratch
    P.stats[26] = dmma_diag;   // DMMAs in diagonal-tile runs / all-row rectangular runs / other patterns (k-step by k-step)
    P.stats[27] = dmma_rect;
    P.stats[28] = dmma_slow;
    P.stats[29] = nruns;
    return GINT_OK;
}

}  // namespace gint
