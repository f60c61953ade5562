// gint_rho.cu -- charge density on the mesh from density-matrix blocks (first cut),
//
//   rho(r_g) = sum_{R,R'} sum_{mu,nu} rho_mu,nu(R) phi_mu(r_g - tau_I - R') phi_nu(r_g - tau_J - R - R')
//                                                              (Sec. 3.3.1, Eq. 44)
//
// In the region picture: rho(p) = sum over ORDERED pairs (a, b) of the region's (atom image) entries of
// phi_a(p)^T D(I_a, I_b, R_b - R_a) phi_b(p).  phi comes from gint_psi_kernel run with unit weights (the same scratch
// and fragment layout as gint_vlocal).  One CTA per (region, 32-point stage): the stage's phi of all row groups is
// staged in shared memory, the 16 warps share the entry pairs (lane = mesh point), partial sums are reduced through
// shared memory and every mesh point is written once (no atomics).  FP64 FMA, not yet on the tensor pipe.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

namespace {
constexpr int kRhoThreads = 512;
constexpr int kRhoWarps = kRhoThreads / 32;


constexpr int kMaxEntries = 64;   // entries of a region whose info and pair table are staged in shared memory
constexpr int kMaxBlock = 256;   // D blocks up to 16 x 16 orbitals are staged per warp in shared memory
constexpr int kRowLD = 33;   // shared-memory row stride in doubles: conflict-free for the transposing store and the reads
}  // namespace

__global__ void __launch_bounds__(kRhoThreads) gint_rho_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ D,
                                                               double* __restrict__ rho) {
    extern __shared__ __align__(16) double s_phi[];   // [ngroup * 32 rows][33] (row = orbital, column = mesh point) + [8 warps][32] partial sums
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nst = P.nstage;
    for (int unit = blockIdx.x; unit < P.nwork_regions * nst; unit += gridDim.x) {
        const int reg_index = __ldg(P.work_regions + unit / nst), st = unit % nst;
        const Region* reg = P.regions + reg_index;
        const int ngroup = __ldg(&reg->ngroup), m = __ldg(&reg->nentry);
        const Entry* entries = P.entries + __ldg(&reg->entry0);
        const uint32_t* pdir = P.pair_direct + __ldg(&reg->pair_off);
        const double* psi = P.psi + ((size_t)__ldg(&reg->psi_chunk0) + st) * kChunkDoubles;
        double* s_part = s_phi + (size_t)ngroup * kGroupRows * kRowLD;
        __syncthreads();   // previous unit done with shared memory
        // stage phi of the stage's 32 points, transposed out of the DMMA fragment order (gint_kernels.cu: element
        // j of a chunk is row 8 i + frow, point (2 kp + kk) 4 + fk with j = (((i 4 + kp) 32 + frow 4 + fk) 2 + kk)
        for (int g = 0; g < ngroup; g++) {
            const double* src = psi + (size_t)g * nst * kChunkDoubles;
            for (int j = tid; j < kChunkDoubles; j += kRhoThreads) {
                const int kk = j & 1, t = j >> 1, fk = t & 3, frow = (t >> 2) & 7, q = t >> 5, kp = q & 3, i = q >> 2;
                s_phi[(g * kGroupRows + i * 8 + frow) * kRowLD + (2 * kp + kk) * 4 + fk] = src[j];
            }
        }
        // the region's entries (active on this stage?, orbitals, first row) and its pair table, once per unit
        const int ks0 = st * kStageKsteps;   // the stage's 8 k-steps: one byte of the entries' k-step masks
        int4* s_ent = reinterpret_cast<int4*>(s_part + kRhoWarps * 32 + kRhoWarps * kMaxBlock);
        uint32_t* s_pdir = reinterpret_cast<uint32_t*>(s_ent + kMaxEntries);
        for (int i = tid; i < m; i += kRhoThreads)
            s_ent[i] = make_int4((int)((entries[i].kmask[ks0 >> 5] >> (ks0 & 31)) & 0xFFu), entries[i].norb, entries[i].row0, 0);
        for (int i = tid; i < m * m; i += kRhoThreads) s_pdir[i] = __ldg(pdir + i);
        __syncthreads();
        double acc = 0.0;
        double* s_D = s_part + kRhoWarps * 32 + warp * kMaxBlock;   // this warp's copy of the current D block
        // the warp's pairs, with the next pair's block already in flight (registers) while the current one is used
        // pairs t = a m + b, t = warp, warp + 16, ...: (a, b) advanced without divisions; the next pair that
        // contributes on this stage (both entries active, block exists) is looked up in shared memory
        struct PairIt { int t, a, b; uint32_t off; };
        auto advance = [&](PairIt& it) {   // to the next contributing pair at or after it.t
            while (it.t < m * m) {
                while (it.b >= m) { it.b -= m; it.a++; }
                if (s_ent[it.a].x != 0 && s_ent[it.b].x != 0) {
                    it.off = s_pdir[it.t];
                    if (it.off != kNoBlock) return;
                }
                it.t += kRhoWarps;
                it.b += kRhoWarps;
            }
            it.off = kNoBlock;
        };
        PairIt cur{warp, 0, warp, kNoBlock};
        advance(cur);
        double dreg[kMaxBlock / 32];
        auto fetch = [&](const PairIt& it) {
            if (it.t >= m * m) return;
            const uint32_t o = it.off;
            const int n = s_ent[it.a].y * s_ent[it.b].y;
#pragma unroll
            for (int k = 0; k < kMaxBlock / 32; k++) dreg[k] = (lane + 32 * k < n) ? __ldg(D + o + lane + 32 * k) : 0.0;
        };
        fetch(cur);
        while (cur.t < m * m) {
            const int a = cur.a, b = cur.b;
            const uint32_t off = cur.off;
            const int nI = s_ent[a].y, nJ = s_ent[b].y, ra = s_ent[a].z, rb = s_ent[b].z;
            __syncwarp();
            if (nI <= 16 && nJ <= 16) {   // rows padded to 16 columns: aligned 16-byte broadcast loads
                const float inv_nJ = 1.0f / (float)nJ;
#pragma unroll
                for (int k = 0; k < kMaxBlock / 32; k++) {
                    const int idx = lane + 32 * k;
                    const int r = (int)(((float)idx + 0.5f) * inv_nJ);   // idx / nJ for idx < 256, nJ <= 16
                    if (idx < nI * nJ) s_D[r * 16 + (idx - r * nJ)] = dreg[k];
                }
            }
            __syncwarp();
            PairIt nxt{cur.t + kRhoWarps, cur.a, cur.b + kRhoWarps, kNoBlock};
            advance(nxt);
            fetch(nxt);
            if (nI <= 16 && nJ <= 16) {
                const double* pa = s_phi + ra * kRowLD + lane;
                const double* pb = s_phi + rb * kRowLD + lane;
                double vb[16];   // the column orbitals at this lane's point, in registers across the rows
#pragma unroll
                for (int nu = 0; nu < 16; nu++) vb[nu] = nu < nJ ? pb[nu * kRowLD] : 0.0;
                for (int mu = 0; mu < nI; mu++) {
                    const double2* Dr = reinterpret_cast<const double2*>(s_D + mu * 16);
                    double t0 = 0.0, t1 = 0.0;
#pragma unroll
                    for (int q = 0; q < 8; q++) {
                        if (2 * q < nJ) {   // columns past nJ hold stale numbers times vb = 0: skipped anyway
                            const double2 d = Dr[q];
                            t0 = fma(d.x, vb[2 * q], t0);
                            if (2 * q + 1 < nJ) t1 = fma(d.y, vb[2 * q + 1], t1);
                        }
                    }
                    acc = fma(pa[mu * kRowLD], t0 + t1, acc);
                }
            } else {   // large blocks (more than 16 x 16 orbitals): straight from global memory
                const double* Db = D + off;
                const double* pa = s_phi + ra * kRowLD + lane;
                const double* pb = s_phi + rb * kRowLD + lane;
                for (int mu = 0; mu < nI; mu++) {
                    double tsum = 0.0;
                    for (int nu = 0; nu < nJ; nu++) tsum = fma(__ldg(Db + mu * nJ + nu), pb[nu * kRowLD], tsum);
                    acc = fma(pa[mu * kRowLD], tsum, acc);
                }
            }
            cur = nxt;
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
    const size_t smem = ((size_t)max_groups * kGroupRows * kRowLD + kRhoWarps * 32 + kRhoWarps * kMaxBlock) * sizeof(double) + kMaxEntries * 16 + kMaxEntries * kMaxEntries * 4;
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
