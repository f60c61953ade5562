// gint_plan.hpp -- host-side plan for gint_vlocal (no CUDA here).
//
// Plays the role of the paper's GintInfo initialisation phase: "The continuous
// real space is discretized into a fine mesh (MeshGrid) ... further grouped into
// coarser blocks (BigGrid) ... Each BigGrid maintains a list of neighboring atoms
// that have non-zero orbital overlap with the grid points contained within it."
// -- PAPER.md:380 (Sec. 3.3.1), Fig. 2 at PAPER.md:368.
//
// Output of the plan (all plain arrays, uploaded verbatim by gint_api.cu):
//   * block table  (I,J,R) sorted, offsets, canonical flag, mirror lists
//   * hash table   (I,J,R) -> H offset, open addressing, for device look-ups
//   * entries      one per (big cell, atom image) whose cutoff sphere holds >=1
//                  mesh point of the cell, sorted by (atom, R) inside a cell
//   * work items   (cell, point sub-range, entry range), sorted by cost
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace gint {

constexpr int kMaxOrbPerAtom = 64;
constexpr int kMaxItemPoints = 64;   // K of one work item (mesh points), multiple of 4
constexpr int kMaxEntriesPerItem = 255;
constexpr uint32_t kNoBlock = 0xFFFFFFFFu;

struct SpeciesHost {
    double rcut = 0, dr = 0;
    int ntab = 0, nrad = 0, norb = 0;
    std::vector<int> l;          // [nrad]
    std::vector<double> table;   // [nrad][ntab]
    int tab_offset = 0;          // first double of this species in the packed device table
};

// One (big cell, atom image) pair.  48 bytes, read by the device as is.
struct Entry {
    double rel[3];     // cell origin minus image centre: r_p - tau = rel + ix e1 + iy e2 + iz e3
    int32_t atom;      // I
    int32_t Rpack;     // image shift R' packed 3 x 8 bit (offset 128), + species << 24
    uint32_t mask_lo;  // bit p: mesh point slot p (0..31) of the cell lies inside the sphere
    uint32_t mask_hi;  // slots 32..63
    int32_t row0;      // first row of this entry in the cell's phi tile
    int32_t norb;
};
static_assert(sizeof(Entry) == 48, "Entry layout is shared with the device");

// One unit of work of the integration kernel.  32 bytes.
struct WorkItem {
    int32_t entry0;    // first entry
    int32_t nentry;    // m
    int32_t nrow;      // n_c = orbitals listed (sum of norb)
    int32_t p0;        // first point slot of the cell handled by this item
    int32_t npts;      // K: number of point slots (multiple of 4, <= kMaxItemPoints)
    int32_t origin[3]; // mesh index of the cell's first point
};
static_assert(sizeof(WorkItem) == 32, "WorkItem layout is shared with the device");

struct MirrorItem {   // dst block (I,J,R) <- transpose of src block (J,I,-R); src == dst: symmetrise lower <- upper
    uint32_t dst, src;
    int32_t nI, nJ;
};

struct Plan {
    // inputs
    double lattice[9];
    int ngrid[3];
    int bcell[3];
    int ncell[3];
    int rank = 0, nranks = 1;
    std::vector<SpeciesHost> species;
    std::vector<int> atom_species;
    std::vector<double> atom_pos;
    double dV = 0;
    double estep[9];             // mesh step vectors e_d = a_d / N_d (rows)
    // blocks
    std::vector<int32_t> blk_i, blk_j, blk_R;   // blk_R [nblk][3]
    std::vector<int64_t> blk_off;               // [nblk+1]
    std::vector<MirrorItem> mirror;
    std::vector<uint64_t> hash_keys;            // 0 = empty (keys are stored +1)
    std::vector<uint32_t> hash_vals;
    uint32_t hash_mask = 0;
    // cells
    std::vector<int64_t> cell_start;            // [ncells+1] into entries (cell-major, before item sorting)
    std::vector<Entry> entries;
    std::vector<WorkItem> items;
    // packed radial tables for the device: per species [ntab][nrad] (node-major)
    std::vector<double> tab_packed;
    std::vector<int32_t> sp_meta;               // per species: tab_offset, ntab, nrad, norb, l[0..7] (12 ints)
    std::vector<double> sp_real;                // per species: rcut^2, 1/dr
    // statistics
    double stats[12] = {0};
    int max_entries = 0, max_rows = 0;
    size_t smem_bytes = 0;
    bool tables_in_smem = true;
};

// Shared-memory budget model (bytes) of the integration kernel for one item.
size_t item_smem_bytes(int nrow, int npts, int nentry, size_t table_bytes);
constexpr size_t kSmemLimit = 232448;   // 227 KB opt-in limit per CTA on sm_100

inline uint64_t pack_key(int I, int J, int r1, int r2, int r3) {
    return ((uint64_t)(uint32_t)I << 44) | ((uint64_t)(uint32_t)J << 24) | ((uint64_t)(uint32_t)(r1 + 128) << 16) |
           ((uint64_t)(uint32_t)(r2 + 128) << 8) | (uint64_t)(uint32_t)(r3 + 128);
}
inline uint64_t hash_mix(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL; k ^= k >> 33;
    return k;
}

// Returns 0 or a negative GINT_* code; err receives a message.
int build_plan(Plan& plan, const double* lattice, const int32_t* ngrid, int nspecies, const SpeciesHost* species,
               int natom, const int32_t* atom_species, const double* atom_pos, const int32_t bcell[3], int rank,
               int nranks, std::string& err);

}  // namespace gint
