// gint_plan.hpp -- host-side plan for gint_vlocal (plain C++, no CUDA here).
//
// Plays the role of the paper's GintInfo initialisation phase: "The continuous
// real space is discretized into a fine mesh (MeshGrid) ... further grouped into
// coarser blocks (BigGrid) ... Each BigGrid maintains a list of neighboring atoms
// that have non-zero orbital overlap with the grid points contained within it."
// -- PAPER.md:380 (Sec. 3.3.1), Fig. 2 at PAPER.md:368.
//
// A *region* is this build's BigGrid: a box of up to 512 mesh points.  Its points
// are ordered into k-steps of 4 points (the K of one DMMA.8x8x4) and slices of 8
// k-steps.  Every (atom image, region) pair whose sphere holds a point of the
// region is an *entry*; entries are sorted densest first and their orbitals are
// packed into consecutive *rows* of the region's phi matrix.  Rows are cut into
// fragments of 8 (one DMMA operand) and groups of 32 (one warp-tile edge).  The
// upper triangle of the region's  C = phi diag(V dV) phi^T  is cut into 32x32
// tiles; tiles are packed 16 at a time (one per warp) into *work items* so that
// an item touches at most kMaxSlots row groups.  An item is what one CTA keeps
// register-resident while it streams the region's points through shared memory.
//
// Output of the plan (plain arrays, uploaded verbatim by gint_api.cu):
//   * block table (I,J,R) sorted, offsets, mirror list
//   * regions, entries, per-group k-step activity bytes, row info, pair->block table
//   * work items (tile lists, slot maps, evaluation tasks), sorted by cost
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#ifdef __CUDACC__
#define GINT_HD __host__ __device__
#else
#define GINT_HD
#endif

namespace gint {

constexpr int kMaxOrbPerAtom = 64;
constexpr int kMaxRegionPoints = 512;          // mesh points of one region
constexpr int kKstepPts = 4;                   // K of DMMA.8x8x4
constexpr int kSliceKsteps = 8;                // k-steps per shared-memory slice
constexpr int kSlicePts = kKstepPts * kSliceKsteps;   // 32
constexpr int kMaxKsteps = kMaxRegionPoints / kKstepPts;   // 128
constexpr int kMaxSlices = kMaxKsteps / kSliceKsteps;      // 16
constexpr int kGroupRows = 32;                 // rows of one row group = warp-tile edge
constexpr int kMaxSlots = 8;                   // row groups one work item may touch
constexpr int kTilesPerItem = 16;              // one 32x32 tile per warp
constexpr int kMaxGroups = 40;                 // row groups per region (<= 1280 orbitals listed)
constexpr int kMaxTasksPerItem = 264;        // 8 groups x 32 rows of 1-orbital atoms + stragglers
constexpr uint32_t kNoBlock = 0xFFFFFFFFu;
constexpr uint32_t kPairTransposed = 0x80000000u;

struct SpeciesHost {
    double rcut = 0, dr = 0;
    int ntab = 0, nrad = 0, norb = 0;
    std::vector<int> l;          // [nrad]
    std::vector<double> table;   // [nrad][ntab]
    int tab_offset = 0;          // first double of this species in the packed device table
};

// ---- structures read by the device as they are -------------------------------------------
// One (region, atom image) pair.  64 bytes.
struct Entry {
    double rel[3];       // region origin minus image centre: r_p - tau = rel + ix e1 + iy e2 + iz e3
    int32_t atom;        // I
    int32_t Rpack;       // image shift R' packed 3 x 8 bit (offset 128), + species << 24
    uint32_t kmask[4];   // bit s: k-step s of the region holds a mesh point inside the sphere
    int32_t row0;        // first row of this entry in the region's phi matrix
    int32_t norb;
    int32_t pad[2];
};
static_assert(sizeof(Entry) == 64, "Entry layout is shared with the device");

struct Region {          // 32 bytes
    int32_t origin[3];   // mesh index of the region's first point
    int32_t nrow;        // orbitals listed
    int32_t gmask_off;   // into gmask: [ngroup][nks_pad] bytes, low nibble = fragment activity of a k-step
    int32_t rowinfo_off; // into rowinfo: [ngroup*32]
    int32_t pair_off;    // into pair: [nentry][nentry]
    int32_t nentry;
};
static_assert(sizeof(Region) == 32, "Region layout is shared with the device");

// One evaluation task of a work item: the orbitals of one entry that fall into the item's row groups.
struct EvalTask {        // 12 bytes
    int32_t entry;       // index into entries
    int16_t row0;        // region row of the entry's first orbital
    int8_t slot[3];      // shared-memory slot of row group (row0>>5)+k, -1 = group not needed by the item
    int8_t pad[3];
};
static_assert(sizeof(EvalTask) == 12, "EvalTask layout is shared with the device");

struct WorkItem {        // 64 bytes
    int32_t region;
    int32_t task0;       // first EvalTask
    int16_t ntask;
    int16_t ntile;
    uint32_t slice_mask; // bit s: slice s holds work for this item
    uint8_t tiles[kTilesPerItem][2];   // (slot of row group, slot of column group), row group <= column group
    uint8_t slot_group[kMaxSlots];     // region row group held by each slot
    int32_t nslot;
    int32_t pad;
};
static_assert(sizeof(WorkItem) == 64, "WorkItem layout is shared with the device");

struct MirrorItem {   // dst block (I,J,R) <- transpose of src block (J,I,-R); src == dst: symmetrise lower <- upper
    uint32_t dst, src;
    int32_t nI, nJ;
};

// rowinfo word: entry index within the region | mu << 12 | norb << 20; kNoBlock for padding rows
inline uint32_t pack_rowinfo(int e, int mu, int norb) { return (uint32_t)e | ((uint32_t)mu << 12) | ((uint32_t)norb << 20); }

struct Plan {
    // inputs
    double lattice[9];
    int ngrid[3];
    int bcell[3];                // region edge in mesh points
    int ncell[3];                // regions per axis
    int rank = 0, nranks = 1;
    std::vector<SpeciesHost> species;
    std::vector<int> atom_species;
    std::vector<double> atom_pos;
    double dV = 0;
    double estep[9];             // mesh step vectors e_d = a_d / N_d (rows)
    // region point order
    int npts = 0, nks = 0, nks_pad = 0, nslice = 0;
    std::vector<uint8_t> slot_xyz;              // [nslice*32][4]: ix, iy, iz, valid
    // blocks
    std::vector<int32_t> blk_i, blk_j, blk_R;   // blk_R [nblk][3]
    std::vector<int64_t> blk_off;               // [nblk+1]
    std::vector<MirrorItem> mirror;
    std::vector<uint64_t> hash_keys;            // 0 = empty (keys are stored +1); host look-ups only
    std::vector<uint32_t> hash_vals;
    uint32_t hash_mask = 0;
    // regions
    std::vector<int64_t> cell_start;            // [ncells+1] into cell_atom / cell_R (sorted by atom, R): query API
    std::vector<int32_t> cell_atom, cell_R;
    std::vector<Region> regions;                // non-empty regions only
    std::vector<Entry> entries;                 // region-major, densest first inside a region
    std::vector<uint8_t> gmask;
    std::vector<uint32_t> rowinfo;
    std::vector<uint32_t> pair;
    std::vector<WorkItem> items;
    std::vector<EvalTask> tasks;
    // packed radial tables for the device: per species [ntab][nrad] (node-major)
    std::vector<double> tab_packed;
    std::vector<int32_t> sp_meta;               // per species: tab_offset, ntab, nrad, norb, l[0..7] (12 ints)
    std::vector<double> sp_real;                // per species: rcut^2, 1/dr
    // statistics
    double stats[12] = {0};
    size_t smem_bytes = 0;
    bool tables_in_smem = true;
};

constexpr size_t kSmemLimit = 232448;   // 227 KB opt-in limit per CTA on sm_100
constexpr int kPhiLD = kSlicePts + 4;   // row stride of the phi slice in doubles (conflict-free fragment loads)

// Shared-memory carve-up of the integration kernel (bytes); used by host and device.
struct SmemLayout {
    uint32_t tab, off, w, gmask, tasks, item, misc, phi, total;
};
GINT_HD inline uint32_t smem_align(size_t x) { return (uint32_t)((x + 127) & ~size_t(127)); }
GINT_HD inline SmemLayout smem_layout(size_t table_bytes) {
    auto al = [](size_t x) { return smem_align(x); };
    SmemLayout L;
    uint32_t o = 0;
    L.tab = o;   o += al(table_bytes);
    L.off = o;   o += al((size_t)3 * kMaxRegionPoints * sizeof(double));
    L.w = o;     o += al((size_t)2 * kSlicePts * sizeof(double));
    L.gmask = o; o += al((size_t)kMaxSlots * kMaxKsteps);
    L.tasks = o; o += al((size_t)kMaxTasksPerItem * sizeof(EvalTask));
    L.item = o;  o += al(sizeof(WorkItem) + sizeof(Region));
    L.misc = o;  o += 128;
    L.phi = o;   o += al((size_t)2 * kMaxSlots * kGroupRows * kPhiLD * sizeof(double));
    L.total = o;
    return L;
}

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
