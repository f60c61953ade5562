// gint_plan.hpp -- host-side plan for gint_vlocal (plain C++, no CUDA here).
//
// Plays the role of the paper's GintInfo initialisation phase: "The continuous
// real space is discretized into a fine mesh (MeshGrid) ... further grouped into
// coarser blocks (BigGrid) ... Each BigGrid maintains a list of neighboring atoms
// that have non-zero orbital overlap with the grid points contained within it."
// -- PAPER.md:380 (Sec. 3.3.1), Fig. 2 at PAPER.md:368.
//
// A *region* is this build's BigGrid: a box of up to 512 mesh points.  Its points
// are ordered into k-steps of 4 points (2x2x1, the K of one DMMA.8x8x4) and stages
// of 8 k-steps (32 points: one shared-memory pipeline stage of the contraction and
// one evaluation slice of the psi kernel, one lane per point).  Every (atom image,
// region) pair whose sphere holds a point of the region is an *entry*; entries that
// cover the whole region come first, the others in a chain of similar coverage, and
// their orbitals are packed into consecutive *rows* of the region's psi matrix.  Rows are cut into fragments of 8
// (one DMMA operand) and groups of 32 (one warp-tile edge).  The upper triangle of
// the region's  C = psi psi^T  (psi = phi sqrt(|V - c| dV), see gint_kernels.cu)  is cut into 32x32 tiles; tiles are
// packed kTilesPerItem at a time (one per consumer warp) into *work items* that
// touch at most kMaxSlots row groups.  gint_psi_kernel writes psi of every region
// once into the scratch buffer (chunks of one (group, stage): [k-step 8][row pair 16]
// [point 4][row parity 2] doubles = 8 KB); gint_contract_kernel streams the chunks an item needs
// through a shared-memory ring with bulk copies.
//
// Output of the plan (plain arrays, uploaded verbatim by gint_api.cu):
//   * block table (I,J,R) sorted, offsets, mirror list
//   * regions, entries, evaluation tasks, per-group k-step activity bytes, row info,
//     pair->block table
//   * work items (tile lists, slot maps), region-major, heaviest regions first
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
constexpr int kStageKsteps = 8;                // k-steps per pipeline stage
constexpr int kStagePts = kKstepPts * kStageKsteps;     // 32: one stage = one evaluation slice (one lane per point)
constexpr int kSlicePts = kStagePts;
constexpr int kSliceKsteps = kStageKsteps;
constexpr int kMaxKsteps = kMaxRegionPoints / kKstepPts;   // 128
constexpr int kMaxStages = kMaxKsteps / kStageKsteps;      // 16
constexpr int kGroupRows = 32;                 // rows of one row group = warp-tile edge
constexpr int kMaxSlots = 8;                   // row groups one work item may touch
constexpr int kTilesPerItem = 15;              // one 32x32 tile per consumer warp; a CTA = 15 consumer warps + 1 producer warp
                                               // (16 + 1 warps get 96 registers each, or 112 after setmaxnreg: measured no faster)
constexpr int kCliqueGroups = 5;               // largest c with c (c + 1) / 2 <= kTilesPerItem
constexpr int kMaxGroups = 40;                 // row groups per region (<= 1280 orbitals listed)
constexpr int kChunkDoubles = kGroupRows * kStagePts;      // 1024: psi of one (group, stage), [k-step][row][point]
constexpr int kChunkBytes = kChunkDoubles * 8;             // 8192
constexpr uint32_t kNoBlock = 0xFFFFFFFFu;

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

struct Region {          // 64 bytes
    int32_t origin[3];   // mesh index of the region's first point
    int32_t nrow;        // orbitals listed
    int32_t gmask_off;   // into gmask: [ngroup][nks_pad] bytes, low nibble = fragment activity of a k-step
    int32_t rowinfo_off; // into rowinfo: [ngroup*32]
    int32_t pair_off;    // into pair: [nentry][nentry]
    int32_t nentry;
    int32_t entry0;      // first entry of the region in entries
    int32_t task_off;    // into etasks
    int32_t ntask;       // evaluation tasks (entry, run of 8 stages) with a point inside the sphere
    int32_t ntile;       // 32x32 tiles of the region's upper triangle that hold work (0: the region is skipped)
    int64_t psi_chunk0;  // first 8 KB chunk of the region in the psi scratch: chunk(g, s) = psi_chunk0 + g*nstage + s
    int32_t ngroup;
    int32_t pad;
};
static_assert(sizeof(Region) == 64, "Region layout is shared with the device");

// evaluation task word: entry index within the region | run << 16 (run h = stages 8h .. 8h+7)
inline uint32_t pack_etask(int e, int run) { return (uint32_t)e | ((uint32_t)run << 16); }

// One row group of one region as a work item sees it (a slot of the shared-memory ring).  A work item may hold
// tiles of several regions (small left-over tile sets are packed together); a tile's two slots always belong to
// the same region.
struct SlotInfo {        // 32 bytes
    int64_t chunk0;      // first chunk of the group in the psi scratch: stage s is chunk0 + s
    int32_t pair_off;    // the region's pair table and its edge
    int32_t nentry;
    int32_t origin[3];   // the region's first mesh point (gint_rho writes rho there)
    int32_t pad;
};
static_assert(sizeof(SlotInfo) == 32, "SlotInfo layout is shared with the device");

struct WorkItem {        // 64 bytes
    uint32_t stage_mask; // bit s: stage s (32 points) holds work for this item
    int16_t ntile, nslot;
    uint8_t tiles[16][2];   // per consumer warp: (slot of row group, slot of column group), 0xFF = no tile
    uint8_t pad[24];
};
static_assert(sizeof(WorkItem) == 64, "WorkItem layout is shared with the device");

struct MirrorItem {   // dst block (I,J,R) <- transpose of src block (J,I,-R); src == dst: symmetrise lower <- upper
    uint32_t dst, src;
    int32_t nI, nJ;
};

// Pair-table entry (row entry a <= column entry b of a region): where element (mu of a, nu of b) of the region's
// C goes in H: off + mu * smu + nu * snu.  (smu, snu) = (n_b, 1) if the block (I_a, I_b, R_b - R_a) is canonical,
// (1, n_a) if it is the transpose of the canonical block (I_b, I_a, R_a - R_b).  off = kNoBlock: no such block.
struct PairWord {
    uint32_t off;
    uint16_t smu, snu;
};
static_assert(sizeof(PairWord) == 8, "PairWord layout is shared with the device");

// rowinfo word: entry index within the region | mu << 12 | norb << 20; kNoBlock for padding rows
inline uint32_t pack_rowinfo(int e, int mu, int norb) { return (uint32_t)e | ((uint32_t)mu << 12) | ((uint32_t)norb << 20); }

constexpr size_t kSmemLimit = 232448;   // 227 KB opt-in limit per CTA on sm_100
constexpr int kDescSlots = 3;           // item descriptors in flight in the contraction kernel

// Per-item descriptor: built by the host, copied to shared memory by the contraction kernel's producer warp with
// one bulk copy.
struct ItemDesc {
    WorkItem item;                                  // 64
    SlotInfo slot[kMaxSlots];                       // 256
    uint32_t gm32[kMaxSlots][kMaxStages];           // 512: per (slot, stage): nibble ks = fragments of the slot's group
                                                    //      with an in-sphere point in k-step ks of the stage
    uint32_t rinfo[kMaxSlots][kGroupRows];          // 1024: row info words of the item's slots (flush)
    uint8_t act[kMaxStages];                        // 16: per stage: bit q = slot q has an active k-step in the stage
    int32_t valid;                                  // 0 = queue exhausted
    int32_t pad[11];
    // 3840: per (consumer warp, stage) the RUNS of consecutive k-steps with one fragment pattern (pack_run), in k-step
    // order, 0-terminated: what the warp executes, decided here so that the kernel's per-stage prologue is one load
    uint16_t prog[kTilesPerItem][kMaxStages][kStageKsteps];
};
// run word: ca | ra << 4 | first k-step << 8 | (k-steps - 1) << 11 | 1 << 15
inline uint16_t pack_run(unsigned ra, unsigned ca, int ks, int n) {
    return (uint16_t)(ca | (ra << 4) | ((unsigned)ks << 8) | ((unsigned)(n - 1) << 11) | 0x8000u);
}
static_assert(kStageKsteps == 8 && kStagePts == 32, "one stage = 8 k-steps = one 32-bit mask word = one lane per point");
static_assert(sizeof(ItemDesc) == 5760 && sizeof(ItemDesc) % 128 == 0, "ItemDesc must keep 128-byte alignment");

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
    int npts = 0, nks = 0, nks_pad = 0, nslice = 0, nstage = 0;   // nks_pad = 8*nslice = 4*nstage
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
    std::vector<PairWord> pair;                 // [nentry][nentry] per region, a <= b filled
    std::vector<uint32_t> pair_direct;          // same indexing: offset of block (I_a, I_b, R_b - R_a) itself, any order (gint_rho)
    // Batches: the psi scratch is reused by consecutive batches of regions when one buffer for all regions would exceed
    // scratch_max_bytes (one batch otherwise).  A batch owns consecutive regions, work-region indices and work items.
    struct Batch { int32_t item0, nitems, wr0, nwr; };
    std::vector<Batch> batches;
    std::vector<int32_t> region_batch;          // [regions]
    int64_t scratch_max_bytes = 0;              // as given (0 = default)
    std::vector<ItemDesc> descs;                // one per work item, queue order (batch-major)
    std::vector<uint32_t> etasks;               // evaluation tasks, region-major
    int64_t psi_chunks = 0;                     // 8 KB chunks of the psi scratch buffer
    // packed radial tables for the device: per species [ntab+4][nradp] (node-major, nradp = nrad rounded up
    // to even, every function pre-multiplied by its Y_lm constant, four zero nodes appended)
    std::vector<double> tab_packed;
    std::vector<int32_t> sp_meta;               // per species: tab_offset, ntab, nradp, norb, l[0..7] (12 ints)
    std::vector<double> sp_real;                // per species: rcut^2, 1/dr
    // statistics
    double stats[32] = {0};
    size_t smem_bytes = 0;
    bool tables_in_smem = true;
    int nring = 0;                              // 8 KB chunk buffers of the psi ring in shared memory
};

GINT_HD inline uint32_t smem_align(size_t x) { return (uint32_t)((x + 127) & ~size_t(127)); }
constexpr int kRingChunks = 26;         // 26 x 8 KB of psi in flight per CTA: stages occupy only their active chunks
constexpr int kRingMaxStages = 8;       // stages in flight (one full / empty mbarrier pair each)
constexpr size_t kMaxTableSmem = 56 * 1024;   // larger radial tables stay in global memory (L1/L2-cached)

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
               int nranks, int64_t scratch_max_bytes, std::string& err);
constexpr int64_t kDefaultScratchBytes = int64_t(16) << 30;   // psi scratch limit when the caller gives none

}  // namespace gint
