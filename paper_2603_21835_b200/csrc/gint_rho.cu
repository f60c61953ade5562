// gint_rho.cu -- charge density on the mesh from density-matrix blocks (first cut),
//
//   rho(r_g) = sum_{R,R'} sum_{mu,nu} rho_mu,nu(R) phi_mu(r_g - tau_I - R') phi_nu(r_g - tau_J - R - R')
//                                                              (Sec. 3.3.1, Eq. 44)
//
// In the region picture: rho(p) = sum over ORDERED pairs (a, b) of the region's (atom image) entries of
// phi_a(p)^T D(I_a, I_b, R_b - R_a) phi_b(p).  phi comes from gint_psi_kernel run with unit weights (the same scratch
// and fragment layout as gint_vlocal).  One CTA per (region, 32-point stage): the stage's phi of all row groups is
// staged in shared memory, the 8 warps share the entry pairs (lane = mesh point), partial sums are reduced through
// shared memory and every mesh point is written once (no atomics).  FP64 FMA, not yet on the tensor pipe.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

namespace {
constexpr int kRhoThreads = 256;
constexpr int kRhoWarps = kRhoThreads / 32;
static_assert(kStagePts == 32, "gint_rho_kernel assumes 32-point stages (one lane per point)");

// element (row R, point lane) of a (group, stage) chunk in DMMA fragment order (see gint_kernels.cu)
__device__ __forceinline__ int chunk_index(int R, int lane) {
    return (R >> 5) * kChunkDoubles + ((((R >> 3) & 3) * kStagePairs + (lane >> 3)) * 32 + (R & 7) * 4 + (lane & 3)) * 2 +
           ((lane >> 2) & 1);
}
}  // namespace

__global__ void __launch_bounds__(kRhoThreads) gint_rho_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ D,
                                                               double* __restrict__ rho) {
    extern __shared__ __align__(16) double s_phi[];   // [ngroup][1024] + [8 warps][32] partial sums
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nst = P.nstage;
    for (int unit = blockIdx.x; unit < P.nwork_regions * nst; unit += gridDim.x) {
        const int reg_index = __ldg(P.work_regions + unit / nst), st = unit % nst;
        const Region* reg = P.regions + reg_index;
        const int ngroup = __ldg(&reg->ngroup), m = __ldg(&reg->nentry);
        const Entry* entries = P.entries + __ldg(&reg->entry0);
        const uint32_t* pdir = P.pair_direct + __ldg(&reg->pair_off);
        const double* psi = P.psi + ((size_t)__ldg(&reg->psi_chunk0) + st) * kChunkDoubles;
        double* s_part = s_phi + (size_t)ngroup * kChunkDoubles;
        __syncthreads();   // previous unit done with shared memory
        for (int g = 0; g < ngroup; g++) {
            const double2* src = reinterpret_cast<const double2*>(psi + (size_t)g * nst * kChunkDoubles);
            double2* dst = reinterpret_cast<double2*>(s_phi + (size_t)g * kChunkDoubles);
            for (int i = tid; i < kChunkDoubles / 2; i += kRhoThreads) dst[i] = src[i];
        }
        __syncthreads();
        double acc = 0.0;
        const int ks0 = st * kStageKsteps;   // the stage's 8 k-steps: one byte of the entries' k-step masks
        for (int t = warp; t < m * m; t += kRhoWarps) {
            const int a = t / m, b = t - a * m;
            const Entry* ea = entries + a;
            const Entry* eb = entries + b;
            if ((((ea->kmask[ks0 >> 5] >> (ks0 & 31)) & 0xFFu) == 0u) || (((eb->kmask[ks0 >> 5] >> (ks0 & 31)) & 0xFFu) == 0u))
                continue;   // one of the two orbitals sets vanishes on all 32 points
            const uint32_t off = __ldg(pdir + t);
            if (off == kNoBlock) continue;
            const int nI = ea->norb, nJ = eb->norb, ra = ea->row0, rb = eb->row0;
            const double* Db = D + off;
            for (int mu = 0; mu < nI; mu++) {
                double tsum = 0.0;
                for (int nu = 0; nu < nJ; nu++) tsum = fma(__ldg(Db + mu * nJ + nu), s_phi[chunk_index(rb + nu, lane)], tsum);
                acc = fma(s_phi[chunk_index(ra + mu, lane)], tsum, acc);
            }
        }
        s_part[warp * 32 + lane] = acc;
        __syncthreads();
        if (warp == 0) {
            double v = 0.0;
            for (int w2 = 0; w2 < kRhoWarps; w2++) v += s_part[w2 * 32 + lane];
            const uchar4 c = reinterpret_cast<const uchar4*>(P.slot_xyz)[st * kStagePts + lane];
            const int g1 = __ldg(&reg->origin[0]) + c.x, g2 = __ldg(&reg->origin[1]) + c.y, g3 = __ldg(&reg->origin[2]) + c.z;
            if (c.w && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2])
                rho[((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3] = v;
        }
    }
}

cudaError_t configure_rho(size_t* smem_out, int max_groups) {
    const size_t smem = ((size_t)max_groups * kChunkDoubles + kRhoWarps * 32) * sizeof(double);
    *smem_out = smem;
    return cudaFuncSetAttribute(gint_rho_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

cudaError_t launch_rho_kernel(const DevicePlan& P, size_t smem, int nsm, const double* D, double* rho, cudaStream_t stream) {
    const size_t npts = (size_t)P.ngrid[0] * P.ngrid[1] * P.ngrid[2];
    cudaError_t e = cudaMemsetAsync(rho, 0, npts * sizeof(double), stream);   // mesh points no orbital reaches
    if (e != cudaSuccess || P.nwork_regions <= 0) return e;
    const long long units = (long long)P.nwork_regions * P.nstage;
    const int per_sm = smem > 110 * 1024 ? 1 : 2;
    const int grid = (int)(units < (long long)per_sm * nsm * 4 ? units : (long long)per_sm * nsm * 4);
    gint_rho_kernel<<<grid, kRhoThreads, smem, stream>>>(P, D, rho);
    return cudaGetLastError();
}

}  // namespace gint
