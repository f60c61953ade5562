// gint_device.hpp -- kernel parameter block and launchers shared by gint_api.cu and gint_kernels.cu.
// The plan structures (Entry, Region, WorkItem, ItemDesc, MirrorItem, PairWord) are plain
// C++ and come from gint_plan.hpp; the device reads them exactly as the host wrote them.
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "gint_plan.hpp"

namespace gint {

// Shift of the potential chosen per gint_vlocal call (gint_hinit_kernel): H = c S - C (neg = 1) or c S + C (neg = 0),
// C = sum_g phi |V - c| phi dV.
struct ShiftDev {
    double c;
    uint32_t neg, pad;
};

// Kernel parameter block (passed by value as a __grid_constant__).
struct DevicePlan {
    const ItemDesc* descs;    // one per work item, queue order
    const Region* regions;
    const Entry* entries;
    const uint32_t* etasks;   // evaluation tasks: entry within region | run of 8 stages << 16
    const PairWord* pair;     // (entry a <= entry b) -> where C[mu of a][nu of b] goes in H (gint_vlocal flush)
    const uint32_t* pair_direct;   // (entry a, entry b) -> offset of block (I_a, I_b, R_b - R_a) (gint_rho)
    const uint8_t* slot_xyz;  // [nslice*32][4]
    const double* tab;        // packed radial tables, per species [ntab+4][nradp]
    const int32_t* sp_meta;   // per species 12 ints: tab_offset, ntab, nradp, norb, l[8]
    const double* sp_real;    // per species: rcut^2, 1/dr
    const MirrorItem* mirror;
    const double* S;          // grid overlap blocks (Eq. 45 with V = 1), H layout; built once at setup
    ShiftDev* shift;          // this call's shift of the potential
    double* vpart;            // per-block (min, max) of V
    double* psi;              // scratch: psi_chunks x 1024 doubles, zero-filled once at setup
    unsigned int* counter;    // work-queue head, reset before every launch
    const int32_t* work_regions;   // indices of the regions that own work items
    const uint8_t* gmask;     // per region [ngroup][nks_pad]: fragment activity nibble per k-step (Region::gmask_off)
    double estep[9];          // mesh step vectors a_d / N_d (rows)
    double dV;
    int32_t ngrid[3];
    int32_t nks_pad, nslice, nstage;
    int32_t nitems, nmirror, nregions, nwork_regions;
    int32_t tab_doubles;
    int32_t nspecies;
    int32_t nring;
    int32_t multibatch;       // several batches of regions reuse the psi scratch: the psi kernel zero-fills what it skips
    int32_t never;            // always 0: a branch condition the compiler cannot fold (see KROW in gint_kernels.cu)
};

// k-space assembly (gint_fold.cu): the block table as the device needs it
struct FoldPlan {
    const int32_t* blk_i;      // [nblk]
    const int32_t* blk_j;      // [nblk]
    const int32_t* blk_R;      // [nblk][3]
    const int64_t* blk_off;    // [nblk+1]
    const int32_t* run_start;  // [nrun+1]: blocks run_start[r] .. run_start[r+1]-1 share (I, J)
    const int32_t* first;      // [natom+1]: first orbital of each atom in the dense matrix
    const int32_t* row_run0;   // [natom+1]: first run of each row atom
    const int32_t* col_atom;   // [norb_tot]: atom of each column of the dense matrix
    double2* phase;            // [nblk] scratch: exp(2 pi i kfrac . R) of every block, rewritten by each call
    int32_t nrun, norb_tot, nblk, natom;
};
// local Pulay force (gint_fvl.cu): what its kernels need beyond DevicePlan; built at the first gint_fvl call
struct FvlPlan {
    const uint8_t* gmask;      // per region [ngroup][nks_pad]: fragment activity nibble per k-step (Region::gmask_off)
    const uint32_t* rowinfo;   // per region [ngroup * 32]: entry | mu << 12 | norb << 20 (Region::rowinfo_off)
    const int64_t* e_chunk0;   // per region: first 8 KB chunk of its E = D + D^T in escratch ([ga][gb] sub-blocks)
    const int4* tg_tasks;      // CTA tasks of gint_tgemm_kernel: (region, row quad, stage quad, 0)
    double* escratch;
    double* tscratch;          // T = E Phi, psi chunk layout (same chunk indices as the psi scratch)
    int32_t ntg, nks_pad;
};
// spherical-grid overlaps < phi | exp(-i A.r) | beta > (gint_snap.cu)
struct SnapSpecies {           // orbitals of a species, or its projectors: plain tables [nrad][ntab] at tab + tab_off
    int32_t tab_off, ntab, nrad, ncomp;
    int32_t l[8];
    double rcut, inv_dr;
};
struct SnapPair {              // projectors of atom I against the orbitals of the image of atom J at tau_J + R
    double d[3];               // tau_I - (tau_J + R)
    double tauI[3];
    int64_t off;               // first complex element of the block [n_J][m_I] in S
    int32_t spI, spJ;
};
struct SnapPlan {
    const SnapSpecies* orb;    // [nspecies]
    const SnapSpecies* proj;   // [nspecies]
    const double* tab;
    const SnapPair* pairs;
    const double* rad_x;       // [nrad] nodes on (0, 1)
    const double* rad_w;       // [nrad] weights, sum 1
    const double* ang_xyz;     // [nang][3] unit vectors
    const double* ang_w;       // [nang] weights, sum 4 pi
    const int32_t* groups;     // [ngroup][2]: first pair and number of pairs (<= kSnapGroupPairs, same atom I) of a CTA
    int32_t npair, nrad, nang, ngroup;
};
constexpr int kSnapGroupPairs = 2;   // 3: spills at 128 registers (si512_tzdp slower), 4: worse still (measured)
cudaError_t launch_snap(const SnapPlan& P, int fr, int fc, const double* A, double* S, cudaStream_t stream);

// The launchers walk the plan's batches (regions that share the psi scratch one after the other): nbatch entries of
// (first item, items, first work region, work regions).
struct BatchRange { int32_t item0, nitems, wr0, nwr; };
size_t force_kernel_smem(size_t table_bytes, int nspecies);
cudaError_t configure_fvl(size_t force_smem, bool tab_smem);
cudaError_t launch_fvl(const DevicePlan& P, const FvlPlan& F, size_t psi_smem, size_t force_smem, bool tab_smem, int nsm,
                       int natom, const BatchRange* batches, const int32_t* tg0, int nbatch, const double* V, const double* D,
                       double* Fout, cudaStream_t stream);
DevicePlan batch_plan(const DevicePlan& P, const BatchRange& B);
cudaError_t launch_psi(const DevicePlan& P, size_t psi_smem, bool tab_smem, int nsm, const double* V, cudaStream_t stream);
cudaError_t launch_rho(const DevicePlan& P, size_t psi_smem, size_t contract_smem_bytes, bool tab_smem, int nsm,
                       const BatchRange* batches, int nbatch, const double* D, double* rho, cudaStream_t stream);
cudaError_t launch_fold(const FoldPlan& F, const double* H, const double* kfrac, double* Hk, cudaStream_t stream);
// gint_fold_k_static: phases in a file-scope device array of kFoldStaticMaxBlocks entries (gint_fold.cu)
constexpr int kFoldStaticMaxBlocks = 1 << 18;
cudaError_t fold_static_scratch(int device, double2** out);   // `device` must be current; address cached per device
cudaError_t launch_fold_static(const FoldPlan& F, double2* static_phase, const double* H, const double* kfrac, double* Hk,
                               cudaStream_t stream);

size_t psi_kernel_smem(size_t table_bytes, int nspecies);
size_t contract_kernel_smem(int nring);
cudaError_t configure_kernels(size_t psi_smem, size_t contract_smem_bytes, bool tab_smem);
// ev: nullptr, or 5 events recorded at call start / before psi / before contraction / after it / after mirror (with
// several batches: before the first psi kernel / -- / after the last contraction)
// raw: integrate a non-negative V without the shift (builds S at setup)
cudaError_t launch_vlocal(const DevicePlan& P, size_t psi_smem, size_t contract_smem_bytes, bool tab_smem, int nsm,
                          const BatchRange* batches, int nbatch, size_t h_len, const double* V, double* H, bool raw,
                          cudaStream_t stream, cudaEvent_t* ev);
cudaError_t measure_dmma_peak(double seconds, int nsm, double* tflops);

}  // namespace gint
