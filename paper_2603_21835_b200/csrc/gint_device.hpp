// gint_device.hpp -- structures shared by the host API (gint_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

namespace gint {

constexpr uint32_t kNoBlockDev = 0xFFFFFFFFu;
constexpr int kMaxItemPointsDev = 64;

struct EntryDev {   // == gint::Entry (gint_plan.hpp), 48 bytes
    double rel[3];
    int32_t atom;
    int32_t Rpack;
    uint32_t mask_lo, mask_hi;
    int32_t row0, norb;
};
struct WorkItemDev {   // == gint::WorkItem, 32 bytes
    int32_t entry0, nentry, nrow, p0, npts;
    int32_t origin[3];
};
struct MirrorItemDev {   // == gint::MirrorItem
    uint32_t dst, src;
    int32_t nI, nJ;
};

// Kernel parameter block (passed by value as a __grid_constant__).
struct DevicePlan {
    const WorkItemDev* items;
    const EntryDev* entries;
    const uint64_t* hash_keys;
    const uint32_t* hash_vals;
    const double* tab;        // packed radial tables, per species [ntab][nrad]
    const int32_t* sp_meta;   // per species 12 ints: tab_offset, ntab, nrad, norb, l[8]
    const double* sp_real;    // per species: rcut^2, 1/dr
    const MirrorItemDev* mirror;
    unsigned int* counter;    // work-queue head, reset before every launch
    double estep[9];          // mesh step vectors a_d / N_d (rows)
    double dV;
    int32_t ngrid[3];
    int32_t bcell[3];
    int32_t nitems, nmirror;
    int32_t tab_doubles;
    int32_t max_entries, max_rows_pad;
    uint32_t hash_mask;
};

cudaError_t configure_kernels(const DevicePlan& P, size_t smem_bytes, bool tab_smem);
// ev: nullptr, or 4 events recorded at call start / before main / after main / after mirror
cudaError_t launch_vlocal(const DevicePlan& P, size_t smem_bytes, bool tab_smem, int nsm, size_t h_len,
                          const double* V, double* H, cudaStream_t stream, cudaEvent_t* ev);
cudaError_t measure_dmma_peak(double seconds, int nsm, double* tflops);

}  // namespace gint
