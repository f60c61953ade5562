// gint_fold.cu -- k-space assembly of the real-space blocks,
//
//   H_mu,nu(k) = sum_R exp(i k.R) H_mu,nu(R)                      (Sec. 2.1, Eq. 5)
//
// with k = kfrac . (b1, b2, b3), a_i . b_j = 2 pi delta_ij, so k.R = 2 pi kfrac . (R1, R2, R3).  The block table is
// sorted by (I, J, R), so the blocks of an atom pair are consecutive: one warp owns a pair, sums its images in
// registers and writes each element of the dense matrix once (no atomics).  Pairs without a block stay zero from the
// memset.  The kernel is HBM-bound: it reads H once and writes the touched part of H(k) once.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

__global__ void __launch_bounds__(256) gint_fold_kernel(const FoldPlan F, const double* __restrict__ H, double k1, double k2,
                                                        double k3, double2* __restrict__ Hk) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= F.nrun) return;
    const int b0 = F.run_start[w], b1 = F.run_start[w + 1];
    const int I = F.blk_i[b0], J = F.blk_j[b0];
    const int r0 = F.first[I], c0 = F.first[J];
    const int nI = F.first[I + 1] - r0, nJ = F.first[J + 1] - c0;
    const int n = nI * nJ;
    for (int idx = lane; idx < n; idx += 32) {
        double re = 0.0, im = 0.0;
        for (int b = b0; b < b1; b++) {
            const double x = k1 * F.blk_R[3 * b] + k2 * F.blk_R[3 * b + 1] + k3 * F.blk_R[3 * b + 2];
            double s, c;
            sincospi(2.0 * x, &s, &c);
            const double h = H[F.blk_off[b] + idx];
            re = fma(c, h, re);
            im = fma(s, h, im);
        }
        const int mu = idx / nJ, nu = idx - mu * nJ;
        Hk[(size_t)(r0 + mu) * F.norb_tot + (c0 + nu)] = make_double2(re, im);
    }
}

cudaError_t launch_fold(const FoldPlan& F, const double* H, const double* kfrac, double* Hk, cudaStream_t stream) {
    cudaError_t e = cudaMemsetAsync(Hk, 0, sizeof(double) * 2 * (size_t)F.norb_tot * F.norb_tot, stream);
    if (e != cudaSuccess) return e;
    if (F.nrun > 0) {
        const int wpb = 256 / 32;
        gint_fold_kernel<<<(F.nrun + wpb - 1) / wpb, 256, 0, stream>>>(F, H, kfrac[0], kfrac[1], kfrac[2],
                                                                        reinterpret_cast<double2*>(Hk));
        e = cudaGetLastError();
    }
    return e;
}

}  // namespace gint
