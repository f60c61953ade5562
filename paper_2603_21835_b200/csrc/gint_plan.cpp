// gint_plan.cpp -- host-side plan construction (see gint_plan.hpp).
#include "gint_plan.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

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

inline size_t align16(size_t x) { return (x + 15) & ~size_t(15); }

}  // namespace

// Must mirror the carve-up in gint_kernels.cu (SmemLayout).
static size_t fixed_smem_bytes(int max_entries, int max_rows_pad, size_t table_bytes) {
    size_t b = 0;
    b += align16(table_bytes);
    b += kMaxItemPoints * sizeof(double);                    // w[p] = V dV
    b += 64;                                                 // counters
    b += align16((size_t)max_entries * 16);                  // entry info (row0, norb, atom, Rpack)
    b += align16((size_t)max_rows_pad * sizeof(uint16_t));   // row -> (entry, mu)
    b += align16((size_t)max_rows_pad / 8 * sizeof(uint32_t));   // per fragment-row k-step masks
    b += align16((size_t)max_entries * max_entries * sizeof(uint32_t));   // pair -> H offset
    return b;
}

size_t item_smem_bytes(int nrow, int npts, int nentry, size_t table_bytes) {
    const int nrow_pad = (nrow + 7) & ~7;
    return fixed_smem_bytes(nentry, nrow_pad, table_bytes) + (size_t)nrow_pad * (npts + 4) * sizeof(double);
}

int build_plan(Plan& P, const double* lattice, const int32_t* ngrid, int nspecies, const SpeciesHost* species,
               int natom, const int32_t* atom_species, const double* atom_pos, const int32_t bcell[3], int rank,
               int nranks, std::string& err) {
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
    P.species.assign(species, species + nspecies);
    double rc_max = 0;
    int tab_off = 0;
    for (int s = 0; s < nspecies; s++) {
        SpeciesHost& sp = P.species[s];
        if (!(sp.rcut > 0) || !(sp.dr > 0) || sp.nrad <= 0 || sp.ntab < 4) { err = "bad species"; return GINT_EINVAL; }
        if ((double)sp.ntab * sp.dr < sp.rcut + 3 * sp.dr - 1e-9 * sp.dr) { err = "radial table too short: need ntab*dr >= rcut + 3*dr"; return GINT_EINVAL; }
        if (sp.nrad > 8) { err = "more than 8 radial functions per species"; return GINT_EUNSUPPORTED; }
        sp.norb = 0;
        for (int k = 0; k < sp.nrad; k++) {
            if (sp.l[k] < 0) { err = "negative l"; return GINT_EINVAL; }
            if (sp.l[k] > 2) { err = "l > 2 not supported"; return GINT_EUNSUPPORTED; }
            sp.norb += 2 * sp.l[k] + 1;
        }
        if (sp.norb > kMaxOrbPerAtom) { err = "too many orbitals per atom"; return GINT_EUNSUPPORTED; }
        for (double v : sp.table)
            if (!std::isfinite(v)) { err = "table not finite"; return GINT_EINVAL; }
        sp.tab_offset = tab_off;
        tab_off += sp.ntab * sp.nrad;
        rc_max = std::max(rc_max, sp.rcut);
    }
    P.atom_species.assign(atom_species, atom_species + natom);
    P.atom_pos.assign(atom_pos, atom_pos + 3 * (size_t)natom);
    for (int a = 0; a < natom; a++) {
        if (atom_species[a] < 0 || atom_species[a] >= nspecies) { err = "atom_species out of range"; return GINT_EINVAL; }
        for (int c = 0; c < 3; c++)
            if (!std::isfinite(atom_pos[3 * a + c])) { err = "atom position not finite"; return GINT_EINVAL; }
    }
    int B = 1;
    for (int d = 0; d < 3; d++) {
        P.ngrid[d] = ngrid[d];
        P.bcell[d] = (bcell && bcell[d] > 0) ? bcell[d] : 4;
        if (P.bcell[d] > ngrid[d]) P.bcell[d] = ngrid[d];
        P.ncell[d] = (ngrid[d] + P.bcell[d] - 1) / P.bcell[d];
        B *= P.bcell[d];
        for (int c = 0; c < 3; c++) P.estep[3 * d + c] = lattice[3 * d + c] / (double)ngrid[d];
    }
    if (B > 64) { err = "big cell larger than 64 mesh points"; return GINT_EUNSUPPORTED; }
    P.dV = vol / ((double)ngrid[0] * (double)ngrid[1] * (double)ngrid[2]);

    double inv[9];
    inv3(lattice, inv);
    double blen[3];   // |column d of A^{-1}|: |d frac_d| <= rho * blen[d] inside a ball of radius rho
    for (int d = 0; d < 3; d++) blen[d] = std::sqrt(inv[d] * inv[d] + inv[3 + d] * inv[3 + d] + inv[6 + d] * inv[6 + d]);

    // ---- block table (sorted by I, J, R1, R2, R3) ---------------------------
    auto norb_of = [&](int a) { return P.species[P.atom_species[a]].norb; };
    auto rc_of = [&](int a) { return P.species[P.atom_species[a]].rcut; };
    P.blk_off.push_back(0);
    for (int I = 0; I < natom; I++)
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
                            if (std::abs(r1) > 127 || std::abs(r2) > 127 || std::abs(r3) > 127) {
                                err = "lattice image index beyond +-127";
                                return GINT_EUNSUPPORTED;
                            }
                            P.blk_i.push_back(I);
                            P.blk_j.push_back(J);
                            P.blk_R.push_back(r1);
                            P.blk_R.push_back(r2);
                            P.blk_R.push_back(r3);
                            P.blk_off.push_back(P.blk_off.back() + (int64_t)norb_of(I) * norb_of(J));
                        }
                    }
        }
    const int64_t nblk = (int64_t)P.blk_i.size();
    if (P.blk_off.back() >= (int64_t)kNoBlock) { err = "H buffer exceeds 2^32 doubles"; return GINT_EUNSUPPORTED; }

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

    // ---- packed radial tables (node-major: [k][nrad]) ---------------------------
    P.tab_packed.resize((size_t)tab_off);
    for (int s = 0; s < nspecies; s++) {
        const SpeciesHost& sp = P.species[s];
        for (int k = 0; k < sp.ntab; k++)
            for (int f = 0; f < sp.nrad; f++)
                P.tab_packed[(size_t)sp.tab_offset + (size_t)k * sp.nrad + f] = sp.table[(size_t)f * sp.ntab + k];
        P.sp_meta.push_back(sp.tab_offset);
        P.sp_meta.push_back(sp.ntab);
        P.sp_meta.push_back(sp.nrad);
        P.sp_meta.push_back(sp.norb);
        for (int k = 0; k < 8; k++) P.sp_meta.push_back(k < sp.nrad ? sp.l[k] : -1);
        P.sp_real.push_back(sp.rcut * sp.rcut);
        P.sp_real.push_back(1.0 / sp.dr);
    }
    const size_t table_bytes_all = P.tab_packed.size() * sizeof(double);
    P.tables_in_smem = table_bytes_all <= 64 * 1024;
    const size_t table_bytes = P.tables_in_smem ? table_bytes_all : 0;

    // ---- per-cell (atom image) lists --------------------------------------------
    const int bx = P.bcell[0], by = P.bcell[1], bz = P.bcell[2];
    const int64_t ncells = (int64_t)P.ncell[0] * P.ncell[1] * P.ncell[2];
    const double* e1 = P.estep;
    const double* e2 = P.estep + 3;
    const double* e3 = P.estep + 6;
    // bounding-sphere radius of a full cell about its centre point
    double cell_rad = 0;
    for (int s1 = -1; s1 <= 1; s1 += 2)
        for (int s2 = -1; s2 <= 1; s2 += 2) {
            double v[3];
            for (int c = 0; c < 3; c++)
                v[c] = 0.5 * ((bx - 1) * e1[c] + s1 * (by - 1) * e2[c] + s2 * (bz - 1) * e3[c]);
            cell_rad = std::max(cell_rad, std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
        }
    struct Tmp { int64_t cell; Entry e; };
    std::vector<Tmp> tmp;
    tmp.reserve((size_t)natom * 2048);
    std::vector<int32_t> npoint_orb((size_t)ngrid[0] * ngrid[1] * ngrid[2], 0);
    double n_insphere = 0;
    for (int I = 0; I < natom; I++) {
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
        // walk unwrapped (image q, cell c) pairs covering [nlo, nhi] in each dimension
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
                    if (std::abs(q[0]) > 127 || std::abs(q[1]) > 127 || std::abs(q[2]) > 127) { err = "image index beyond +-127"; return GINT_EUNSUPPORTED; }
                    Entry e;
                    const int o[3] = {c[0] * bx, c[1] * by, c[2] * bz};
                    for (int k = 0; k < 3; k++) {
                        const double origin = o[0] * e1[k] + o[1] * e2[k] + o[2] * e3[k];
                        const double centre = tau[k] - (q[0] * lattice[k] + q[1] * lattice[3 + k] + q[2] * lattice[6 + k]);
                        e.rel[k] = origin - centre;
                    }
                    // quick reject with the bounding sphere of the (full) cell
                    double cc[3];
                    for (int k = 0; k < 3; k++)
                        cc[k] = e.rel[k] + 0.5 * ((bx - 1) * e1[k] + (by - 1) * e2[k] + (bz - 1) * e3[k]);
                    const double dcen = std::sqrt(cc[0] * cc[0] + cc[1] * cc[1] + cc[2] * cc[2]);
                    if (dcen >= rc + cell_rad + 1e-9) continue;
                    uint64_t mask = 0;
                    for (int ix = 0; ix < bx; ix++) {
                        if (o[0] + ix >= ngrid[0]) break;
                        for (int iy = 0; iy < by; iy++) {
                            if (o[1] + iy >= ngrid[1]) break;
                            for (int iz = 0; iz < bz; iz++) {
                                if (o[2] + iz >= ngrid[2]) break;
                                const double dx = e.rel[0] + ix * e1[0] + iy * e2[0] + iz * e3[0];
                                const double dy = e.rel[1] + ix * e1[1] + iy * e2[1] + iz * e3[1];
                                const double dz = e.rel[2] + ix * e1[2] + iy * e2[2] + iz * e3[2];
                                if (dx * dx + dy * dy + dz * dz < rc2) {
                                    mask |= 1ull << ((ix * by + iy) * bz + iz);
                                    npoint_orb[((size_t)(o[0] + ix) * ngrid[1] + (o[1] + iy)) * ngrid[2] + (o[2] + iz)] += norb;
                                }
                            }
                        }
                    }
                    if (!mask) continue;
                    n_insphere += (double)__builtin_popcountll(mask);
                    e.atom = I;
                    e.Rpack = ((-q[0] + 128) << 16) | ((-q[1] + 128) << 8) | (-q[2] + 128) | (sp_id << 24);
                    e.mask_lo = (uint32_t)mask;
                    e.mask_hi = (uint32_t)(mask >> 32);
                    e.row0 = 0;
                    e.norb = norb;
                    tmp.push_back({((int64_t)c[0] * P.ncell[1] + c[1]) * P.ncell[2] + c[2], e});
                }
        }
    }
    // sort by (cell, atom, R1, R2, R3): inside a cell a<b in list order implies block (I_a,I_b,R_b-R_a) canonical
    auto rkey = [](const Entry& e) { return (uint32_t)(e.Rpack & 0xFFFFFF); };
    std::sort(tmp.begin(), tmp.end(), [&](const Tmp& a, const Tmp& b) {
        if (a.cell != b.cell) return a.cell < b.cell;
        if (a.e.atom != b.e.atom) return a.e.atom < b.e.atom;
        return rkey(a.e) < rkey(b.e);
    });
    P.cell_start.assign((size_t)ncells + 1, 0);
    for (auto& t : tmp) P.cell_start[(size_t)t.cell + 1]++;
    for (int64_t c = 0; c < ncells; c++) P.cell_start[(size_t)c + 1] += P.cell_start[(size_t)c];
    P.entries.resize(tmp.size());
    for (size_t i = 0; i < tmp.size(); i++) P.entries[i] = tmp[i].e;
    tmp.clear();
    tmp.shrink_to_fit();

    // ---- work items ----------------------------------------------------------------
    P.max_entries = 0;
    P.max_rows = 0;
    for (int64_t c = 0; c < ncells; c++) {
        const int64_t s = P.cell_start[(size_t)c], t = P.cell_start[(size_t)c + 1];
        int rows = 0;
        for (int64_t i = s; i < t; i++) {
            P.entries[(size_t)i].row0 = rows;
            rows += P.entries[(size_t)i].norb;
        }
        if (t - s > kMaxEntriesPerItem) { err = "more than 255 atom images touch one big cell"; return GINT_EUNSUPPORTED; }
        P.max_entries = std::max(P.max_entries, (int)(t - s));
        P.max_rows = std::max(P.max_rows, rows);
    }
    const int max_rows_pad = (P.max_rows + 7) & ~7;
    const size_t fixed = fixed_smem_bytes(P.max_entries, max_rows_pad, table_bytes);
    const int Bpad = (B + 3) & ~3;
    double sum_knn = 0, sum_nn = 0, nsplit = 0;
    for (int64_t c = 0; c < ncells; c++) {
        const int64_t s = P.cell_start[(size_t)c], t = P.cell_start[(size_t)c + 1];
        if (s == t) continue;
        const Entry& last = P.entries[(size_t)t - 1];
        const int rows = last.row0 + last.norb;
        const int rows_pad = (rows + 7) & ~7;
        int K = std::min(Bpad, kMaxItemPoints);
        while (K > 4 && fixed + (size_t)rows_pad * (K + 4) * sizeof(double) > kSmemLimit) K = ((K / 2) + 3) & ~3;
        if (fixed + (size_t)rows_pad * (K + 4) * sizeof(double) > kSmemLimit) { err = "big cell does not fit in shared memory"; return GINT_EUNSUPPORTED; }
        const int c3 = (int)(c % P.ncell[2]), c2 = (int)((c / P.ncell[2]) % P.ncell[1]), c1 = (int)(c / ((int64_t)P.ncell[1] * P.ncell[2]));
        if (K < Bpad) nsplit += 1;
        for (int p0 = 0; p0 < Bpad; p0 += K) {
            WorkItem w;
            w.entry0 = (int32_t)s;
            w.nentry = (int32_t)(t - s);
            w.nrow = rows;
            w.p0 = p0;
            w.npts = std::min(K, Bpad - p0);
            w.origin[0] = c1 * bx;
            w.origin[1] = c2 * by;
            w.origin[2] = c3 * bz;
            // skip sub-ranges no sphere reaches
            uint64_t any = 0;
            for (int64_t i = s; i < t; i++) any |= ((uint64_t)P.entries[(size_t)i].mask_hi << 32) | P.entries[(size_t)i].mask_lo;
            const uint64_t range = (w.npts >= 64 ? ~0ull : ((1ull << w.npts) - 1)) << p0;
            if (!(any & range)) continue;
            P.items.push_back(w);
            sum_knn += (double)w.npts * rows * rows;
            sum_nn += (double)rows * rows;
        }
    }
    std::stable_sort(P.items.begin(), P.items.end(), [](const WorkItem& a, const WorkItem& b) {
        return (int64_t)a.npts * a.nrow * a.nrow > (int64_t)b.npts * b.nrow * b.nrow;
    });
    P.smem_bytes = 0;
    for (const WorkItem& w : P.items)
        P.smem_bytes = std::max(P.smem_bytes, fixed + (size_t)((w.nrow + 7) & ~7) * (w.npts + 4) * sizeof(double));
    if (P.items.empty()) P.smem_bytes = fixed;

    double fpt = 0, fsym = 0;
    for (int32_t n : npoint_orb) {
        fpt += 2.0 * (double)n * (double)n;
        fsym += (double)n * ((double)n + 1.0);
    }
    P.stats[0] = (double)ncells;
    P.stats[1] = (double)P.items.size();
    P.stats[2] = (double)P.entries.size();
    P.stats[3] = (double)P.max_rows;
    P.stats[4] = sum_knn;
    P.stats[5] = sum_nn;
    P.stats[6] = (double)P.smem_bytes;
    P.stats[7] = 2;
    P.stats[8] = fpt;
    P.stats[9] = fsym;
    P.stats[10] = n_insphere;
    P.stats[11] = nsplit;
    return GINT_OK;
}

}  // namespace gint
