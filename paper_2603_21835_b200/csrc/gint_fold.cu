// gint_fold.cu -- k-space assembly of the real-space blocks,
//
//   H_mu,nu(k) = sum_R exp(i k.R) H_mu,nu(R)                      (Sec. 2.1, Eq. 5)
//
// with k = kfrac . (b1, b2, b3), a_i . b_j = 2 pi delta_ij, so k.R = 2 pi kfrac . (R1, R2, R3).  The block table is
// sorted by (I, J, R), so the blocks of an atom pair are consecutive (a "run").  Single pass, every element of the
// dense matrix written exactly once, zeros included (no memset): one CTA per row atom I sweeps the n_I rows of the
// dense matrix, consecutive threads on consecutive columns (coalesced 16-byte stores, one column per thread); a column's atom J comes from a
// table, the run (I, J) from a binary search in the row's run list (shared memory), the phases exp(2 pi i kfrac . R)
// of all blocks from a small kernel run first.  HBM-bound: H read once, H(k) written once.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "gint_device.hpp"

namespace gint {

__global__ void __launch_bounds__(256) gint_fold_phase_kernel(const FoldPlan F, double k1, double k2, double k3) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= F.nblk) return;
    const double x = k1 * F.blk_R[3 * b] + k2 * F.blk_R[3 * b + 1] + k3 * F.blk_R[3 * b + 2];
    double s, c;
    sincospi(2.0 * x, &s, &c);
    F.phase[b] = make_double2(c, s);
}

constexpr int kFoldRunsSmem = 4096;   // run list of a row atom kept in shared memory up to this length
constexpr int kFoldCols = 1;          // columns per thread: a CTA covers 256 consecutive columns of one row atom (1 beats 2 and 4: the kernel
                                      // lives on threads in flight for its dependent block-offset -> H loads)

__global__ void __launch_bounds__(256) gint_fold_kernel(const FoldPlan F, const double* __restrict__ H, double2* __restrict__ Hk) {
    __shared__ int32_t s_runJ[kFoldRunsSmem];
    const int I = blockIdx.y;
    const int run0 = F.row_run0[I], nrun = F.row_run0[I + 1] - run0;
    const int r0 = F.first[I], nI = F.first[I + 1] - r0;
    const bool in_smem = nrun <= kFoldRunsSmem;
    if (in_smem)
        for (int i = threadIdx.x; i < nrun; i += blockDim.x) s_runJ[i] = F.blk_j[F.run_start[run0 + i]];
    __syncthreads();
    // this thread's columns: the run (I, J) of each is looked up once and reused for the n_I rows
    int b0[kFoldCols], b1[kFoldCols], e0[kFoldCols], nJ[kFoldCols];
#pragma unroll
    for (int q = 0; q < kFoldCols; q++) {
        const int c = (blockIdx.x * kFoldCols + q) * 256 + threadIdx.x;
        b0[q] = b1[q] = e0[q] = nJ[q] = 0;
        if (c >= F.norb_tot) continue;
        const int J = __ldg(F.col_atom + c);
        int lo = 0, hi = nrun;   // first run of the row with atom >= J
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const int Jm = in_smem ? s_runJ[mid] : __ldg(F.blk_j + __ldg(F.run_start + run0 + mid));
            if (Jm < J) lo = mid + 1;
            else hi = mid;
        }
        if (lo < nrun && (in_smem ? s_runJ[lo] : __ldg(F.blk_j + __ldg(F.run_start + run0 + lo))) == J) {
            const int c0 = __ldg(F.first + J);
            nJ[q] = __ldg(F.first + J + 1) - c0;
            e0[q] = c - c0;
            b0[q] = __ldg(F.run_start + run0 + lo);
            b1[q] = __ldg(F.run_start + run0 + lo + 1);
        }
    }
    for (int mu = 0; mu < nI; mu++) {
#pragma unroll
        for (int q = 0; q < kFoldCols; q++) {
            const int c = (blockIdx.x * kFoldCols + q) * 256 + threadIdx.x;
            if (c >= F.norb_tot) continue;
            double re = 0.0, im = 0.0;
            for (int b = b0[q]; b < b1[q]; b++) {
                const double2 ph = F.phase[b];
                const double h = __ldg(H + __ldg(F.blk_off + b) + mu * nJ[q] + e0[q]);
                re = fma(ph.x, h, re);
                im = fma(ph.y, h, im);
            }
            Hk[(size_t)(r0 + mu) * F.norb_tot + c] = make_double2(re, im);
        }
    }
}

cudaError_t launch_fold(const FoldPlan& F, const double* H, const double* kfrac, double* Hk, cudaStream_t stream) {
    if (F.natom <= 0) return cudaSuccess;
    if (F.nblk > 0) gint_fold_phase_kernel<<<(F.nblk + 255) / 256, 256, 0, stream>>>(F, kfrac[0], kfrac[1], kfrac[2]);
    const dim3 grid((unsigned)((F.norb_tot + kFoldCols * 256 - 1) / (kFoldCols * 256)), (unsigned)F.natom);
    gint_fold_kernel<<<grid, 256, 0, stream>>>(F, H, reinterpret_cast<double2*>(Hk));
    return cudaGetLastError();
}

// ---- gint_fold_k_static: the same two kernels with the phase scratch in a file-scope array ---------------------
// For callers that may not allocate (CUDA graph capture, serving loops): the phases exp(2 pi i kfrac . R) go to a fixed
// array that every GPU loading the library holds until exit (kFoldStaticMaxBlocks x 16 bytes = 4 MiB) instead of the
// context's own buffer.  In host code the array's name is only a stand-in; its device address comes from
// cudaGetSymbolAddress, once per device with that device current (fold_static_scratch, called by the set-up), and is
// handed to the kernels in FoldPlan::phase.  Nothing has to start at zero: gint_fold_phase_kernel rewrites entries
// 0 .. nblk-1 before gint_fold_kernel reads them on the same stream.  All contexts of a device share the array, so
// calls that overlap on the GPU (two streams, two contexts) race on it.
static __device__ __align__(256) double2 g_fold_static_phase[kFoldStaticMaxBlocks];

cudaError_t fold_static_scratch(int device, double2** out) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static double2* addr[kMaxDevices] = {};
    *out = nullptr;
    int current = -1;
    cudaError_t e = cudaGetDevice(&current);
    if (e != cudaSuccess) return e;
    if (device < 0 || device >= kMaxDevices || current != device) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_fold_static_phase);
        if (e != cudaSuccess) return e;
        addr[device] = reinterpret_cast<double2*>(p);
    }
    *out = addr[device];
    return cudaSuccess;
}

cudaError_t launch_fold_static(const FoldPlan& F, double2* static_phase, const double* H, const double* kfrac, double* Hk,
                               cudaStream_t stream) {
    if (!static_phase || F.nblk > kFoldStaticMaxBlocks) return cudaErrorInvalidValue;
    FoldPlan G = F;
    G.phase = static_phase;
    return launch_fold(G, H, kfrac, Hk, stream);
}

}  // namespace gint
