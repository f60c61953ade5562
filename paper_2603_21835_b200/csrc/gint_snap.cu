// gint_snap.cu -- spherical-grid integration of the velocity-gauge nonlocal overlaps (the paper's snap_psibeta),
// PAPER.md:415-426 (Sec. 3.3.2, Eq. 47):
//
//   S(I, J, R)[mu][b] = < phi_mu(r - tau_J - R) | exp(-i A.r) | beta_b(r - tau_I) >
//                     = sum_i sum_a  w_i rb r_i^2  w_a  phi_mu(tau_I + r_i n_a - tau_J - R)
//                                    exp(-i A.(tau_I + r_i n_a))  beta_b(r_i n_a),
//
// quadrature centred on the projector's atom: radial nodes r_i = x_i rb_I (Gauss-Legendre, 140 in the paper), angular
// nodes n_a (Lebedev-Laikov, 110 in the paper), both tables given by the caller.  beta_{l m zeta} = b(|r|) Y_lm like an
// orbital.  One CTA per two consecutive (I, J, R) pairs of an atom I (the paper batches all neighbours of a central atom
// into one launch; here all pairs of all atoms are one launch).  The 128 threads walk the nr x na quadrature points; a thread evaluates the n_J
// orbitals and the m_I weighted, phase-modulated projector components of its point into its warp's staging tile in
// shared memory, and the warp contracts 32 points at a time on the FP64 tensor pipe:
//   C[mu][c] += sum_p Phi[p][mu] G[p][c],   G[p][2b] = Re, G[p][2b+1] = Im of  w_p beta_b(p) exp(-i A.r_p)
// (DMMA.8x8x4, K = points).  No atomics: the four warps' partial C are added through shared memory in a fixed order
// and every element of S is written once (the paper's kernel reduces with shuffles and shared memory for the same
// reason).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <string>
#include <vector>

#include "gint_device.hpp"

namespace gint {

namespace {

__device__ __forceinline__ void dmma_s(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// Values of all components of a species (orbitals or projectors) at distance r (< rcut) and direction (x, y, z) from
// its centre, times `scale`, written to out[0], out[os], .. out[(ncomp-1) os]: cubic Lagrange interpolation on the
// forward stencil k .. k+3, k = floor(r / dr); real Y_lm as in include/gint.h (l <= 3); nz = 0 marks r < 1e-12, where
// the direction is (0, 0, 0).
__device__ __forceinline__ void snap_eval_core(const SnapSpecies& sp, const double* __restrict__ tab, double r, double x, double y, double z,
                                               double nz, double scale, double* __restrict__ out, int os) {
    const double s = r * sp.inv_dr;
    const int k = __double2int_rd(s);
    const double t = s - (double)k;
    const double t1 = 1.0 - t, t2 = 2.0 - t, t3 = 3.0 - t;
    const double a23 = t2 * t3, b01 = t * t1;
    const double L0 = (t1 * a23) * (scale * (1.0 / 6.0));
    const double L1 = (t * a23) * (scale * 0.5);
    const double L2 = (b01 * t3) * (scale * -0.5);
    const double L3 = (b01 * t2) * (scale * (1.0 / 6.0));
    int c = 0;
    for (int f = 0; f < sp.nrad; f++) {
        const double* T = tab + sp.tab_off + (size_t)f * sp.ntab + k;
        const double fv = fma(T[0], L0, fma(T[1], L1, fma(T[2], L2, T[3] * L3)));
        const int l = sp.l[f];
        if (l == 0) {
            out[os * c++] = 0.28209479177387814 * fv;
        } else if (l == 1) {
            const double g = 0.48860251190291992 * fv;
            out[os * c++] = g * y; out[os * c++] = g * z; out[os * c++] = g * x;
        } else if (l == 2) {
            const double g = 1.0925484305920792 * fv;
            out[os * c++] = g * (x * y);
            out[os * c++] = g * (y * z);
            out[os * c++] = (0.31539156525252005 * fv) * fma(3.0 * z, z, -nz);
            out[os * c++] = g * (x * z);
            out[os * c++] = (0.54627421529603959 * fv) * fma(x, x, -(y * y));
        } else {
            const double x2 = x * x, y2 = y * y, q = fma(5.0 * z, z, -nz);
            const double g3 = 0.59004358992664352 * fv, g1 = 0.45704579946446577 * fv;
            out[os * c++] = (g3 * y) * fma(3.0, x2, -y2);
            out[os * c++] = (2.8906114426405538 * fv) * (x * y * z);
            out[os * c++] = (g1 * y) * q;
            out[os * c++] = (0.37317633259011540 * fv * z) * fma(5.0 * z, z, -3.0 * nz);
            out[os * c++] = (g1 * x) * q;
            out[os * c++] = (1.4453057213202769 * fv * z) * (x2 - y2);
            out[os * c++] = (g3 * x) * fma(-3.0, y2, x2);
        }
    }
}

// orbitals at displacement (dx, dy, dz): zero for r >= rcut; 1/r from the hardware seed and one cubic correction
__device__ __forceinline__ void snap_eval(const SnapSpecies& sp, const double* __restrict__ tab, double dx, double dy, double dz,
                                          double* __restrict__ out, int os) {
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    if (!(r2 < sp.rcut * sp.rcut)) {
        for (int c = 0; c < sp.ncomp; c++) out[c * os] = 0.0;
        return;
    }
    double rinv = 0.0, nz = 0.0;
    if (r2 >= 1e-24) {
        double y0;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));   // relative error ~2^-22
        const double e = fma(-(r2 * y0), y0, 1.0);                   // 1 - r2 y0^2
        rinv = fma(e * y0, fma(0.375, e, 0.5), y0);                  // y0 (1 + e/2 + 3 e^2/8): error ~e^3
        nz = 1.0;
    }
    snap_eval_core(sp, tab, r2 * rinv, dx * rinv, dy * rinv, dz * rinv, nz, 1.0, out, os);
}

constexpr int kSnapThreads = 128;
constexpr int kSnapStride = 36;   // staging tiles are [column][point]: 32 points + 4, so that the lanes' writes (one column,
                                  // 32 points) and the fragment reads (4 points x 8 columns) are both free of bank conflicts

}  // namespace

// FR x FC accumulator fragments of 8 x 8: rows = orbitals of J (n_J <= 8 FR), columns = (Re, Im) of the projector
// components of I (2 m_I <= 8 FC)
template <int FR, int FC>
__global__ void __launch_bounds__(kSnapThreads, 4) gint_snap_kernel(const SnapPlan P, double ax, double ay, double az, double* __restrict__ S) {
    extern __shared__ __align__(16) double snap_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* sPhi = snap_smem + (size_t)warp * (FR + FC) * 8 * kSnapStride;   // [8 FR columns: orbitals][36]
    double* sG = sPhi + FR * 8 * kSnapStride;                                // [8 FC columns: Re, Im of the projectors][36]
    // a CTA takes up to kSnapGroupPairs consecutive pairs of ONE projector atom: the projector side of a point (beta,
    // weight, phase) is evaluated once and contracted with the orbitals of each of them
    const int g0 = P.groups[2 * blockIdx.x], gn = P.groups[2 * blockIdx.x + 1];
    const SnapPair pr = P.pairs[g0];
    const SnapSpecies& sb = P.proj[pr.spI];
    const int mI = sb.ncomp;
    const double rb = sb.rcut;
    const int npts = P.nrad * P.nang;
    double dq[kSnapGroupPairs][3];
    int spq[kSnapGroupPairs];
#pragma unroll
    for (int nb = 0; nb < kSnapGroupPairs; nb++) {
        const SnapPair& q = P.pairs[g0 + (nb < gn ? nb : 0)];
        dq[nb][0] = q.d[0]; dq[nb][1] = q.d[1]; dq[nb][2] = q.d[2];
        spq[nb] = q.spJ;
    }
    double acc[kSnapGroupPairs][FR][FC][2];
#pragma unroll
    for (int nb = 0; nb < kSnapGroupPairs; nb++)
#pragma unroll
        for (int i = 0; i < FR; i++)
#pragma unroll
            for (int j = 0; j < FC; j++) acc[nb][i][j][0] = acc[nb][i][j][1] = 0.0;
    // zero the staging tiles once: columns that are never written stay zero
    for (int e = lane; e < (FR + FC) * 8 * kSnapStride; e += 32) sPhi[e] = 0.0;
    __syncwarp();
    const int frow = lane >> 2, fk = lane & 3;
    for (int p0 = warp * 32; p0 < npts; p0 += kSnapThreads) {
        const int p = p0 + lane;
        double* myPhi = sPhi + lane;   // column c of this lane's point: myPhi[c * kSnapStride]
        double* myG = sG + lane;
        double ux = 0.0, uy = 0.0, uz = 0.0;
        if (p < npts) {
            const int ir = p / P.nang, ia = p - ir * P.nang;
            const double r = P.rad_x[ir] * rb;
            const double nx = P.ang_xyz[3 * ia], ny = P.ang_xyz[3 * ia + 1], nz_ = P.ang_xyz[3 * ia + 2];
            ux = r * nx; uy = r * ny; uz = r * nz_;
            const double w = P.rad_w[ir] * rb * r * r * P.ang_w[ia];
            // weighted real projector values through the Phi columns of this point, then G = beta (cos - i sin)(A.r)
            // (the quadrature point sits at distance r < rb in direction n_a by construction: no square root)
            snap_eval_core(sb, P.tab, r, nx, ny, nz_, 1.0, w, myPhi, kSnapStride);
            double sn, cs;
            sincos(ax * (pr.tauI[0] + ux) + ay * (pr.tauI[1] + uy) + az * (pr.tauI[2] + uz), &sn, &cs);
            for (int b = 0; b < mI; b++) {
                const double bv = myPhi[b * kSnapStride];
                myG[(2 * b) * kSnapStride] = bv * cs;
                myG[(2 * b + 1) * kSnapStride] = -(bv * sn);
            }
        } else {
            for (int c = 0; c < 2 * mI; c++) myG[c * kSnapStride] = 0.0;
        }
#pragma unroll
        for (int nb = 0; nb < kSnapGroupPairs; nb++) {
            if (nb < gn) {
                const SnapSpecies& so = P.orb[spq[nb]];
                if (p < npts) {
                    // rows beyond n_J keep what the step before left there (projector values or another neighbour's
                    // orbitals): they only reach accumulator rows that are never written out
                    snap_eval(so, P.tab, ux + dq[nb][0], uy + dq[nb][1], uz + dq[nb][2], myPhi, kSnapStride);
                } else {
                    for (int c = 0; c < FR * 8; c++) myPhi[c * kSnapStride] = 0.0;
                }
                __syncwarp();
                // 32 points = 8 k-steps of 4 points: A[row mu = 8 i + lane / 4][k = lane % 4], B[k = lane % 4][col = 8 j + lane / 4]
#pragma unroll
                for (int q = 0; q < 8; q++) {
                    double a[FR], b[FC];
#pragma unroll
                    for (int i = 0; i < FR; i++) a[i] = sPhi[(8 * i + frow) * kSnapStride + 4 * q + fk];
#pragma unroll
                    for (int j = 0; j < FC; j++) b[j] = sG[(8 * j + frow) * kSnapStride + 4 * q + fk];
#pragma unroll
                    for (int i = 0; i < FR; i++)
#pragma unroll
                        for (int j = 0; j < FC; j++) dmma_s(acc[nb][i][j][0], acc[nb][i][j][1], a[i], b[j]);
                }
                __syncwarp();
            }
        }
    }
    // cross-warp sum in a fixed order: warp w writes its fragments, then thread e adds the four copies of element e
    double* red = snap_smem;   // [4 warps][FR * 8][FC * 8]
    constexpr int kCols = FC * 8;
#pragma unroll
    for (int nb = 0; nb < kSnapGroupPairs; nb++) {
        if (nb < gn) {
            __syncthreads();
#pragma unroll
            for (int i = 0; i < FR; i++)
#pragma unroll
                for (int j = 0; j < FC; j++) {
                    // C fragment: lane holds (row lane / 4, columns 2 (lane % 4), 2 (lane % 4) + 1)
                    double* dst = red + ((size_t)warp * FR * 8 + 8 * i + frow) * kCols + 8 * j + 2 * fk;
                    dst[0] = acc[nb][i][j][0];
                    dst[1] = acc[nb][i][j][1];
                }
            __syncthreads();
            const int nJ = P.orb[spq[nb]].ncomp;
            double* out = S + 2 * P.pairs[g0 + nb].off;   // block [n_J][m_I] complex = [n_J][2 m_I] doubles
            for (int e = tid; e < nJ * 2 * mI; e += kSnapThreads) {
                const int mu = e / (2 * mI), c = e - mu * 2 * mI;
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < kSnapThreads / 32; w++) v += red[((size_t)w * FR * 8 + mu) * kCols + c];
                out[e] = v;
            }
        }
    }
}

size_t snap_kernel_smem(int fr, int fc) {
    const size_t stage = (size_t)(kSnapThreads / 32) * (fr + fc) * 8 * kSnapStride * sizeof(double);
    const size_t red = (size_t)(kSnapThreads / 32) * fr * 8 * fc * 8 * sizeof(double);
    return std::max(stage, red);
}

template <int FR, int FC>
static cudaError_t launch_snap_t(const SnapPlan& P, const double* A, double* S, cudaStream_t stream) {
    const size_t smem = snap_kernel_smem(FR, FC);
    cudaError_t e = cudaFuncSetAttribute(gint_snap_kernel<FR, FC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    gint_snap_kernel<FR, FC><<<P.ngroup, kSnapThreads, smem, stream>>>(P, A[0], A[1], A[2], S);
    return cudaGetLastError();
}

// fr = ceil(max orbitals per atom / 8) <= 4, fc = ceil(2 max projector components / 8) <= 4
cudaError_t launch_snap(const SnapPlan& P, int fr, int fc, const double* A, double* S, cudaStream_t stream) {
    if (P.npair <= 0) return cudaSuccess;
    if (fr < 1 || fr > 4 || fc < 1 || fc > 4) return cudaErrorInvalidValue;
#define SNAP_CASE(R, C) case (R) * 4 + (C): return launch_snap_t<R, C>(P, A, S, stream);
    switch (fr * 4 + fc) {
        SNAP_CASE(1, 1) SNAP_CASE(1, 2) SNAP_CASE(1, 3) SNAP_CASE(1, 4)
        SNAP_CASE(2, 1) SNAP_CASE(2, 2) SNAP_CASE(2, 3) SNAP_CASE(2, 4)
        SNAP_CASE(3, 1) SNAP_CASE(3, 2) SNAP_CASE(3, 3) SNAP_CASE(3, 4)
        SNAP_CASE(4, 1) SNAP_CASE(4, 2) SNAP_CASE(4, 3) SNAP_CASE(4, 4)
    }
#undef SNAP_CASE
    return cudaErrorInvalidValue;
}

}  // namespace gint
