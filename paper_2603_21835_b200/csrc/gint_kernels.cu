// gint_kernels.cu -- sm_100a kernels of gint_vlocal.
//
//   H_mu,nu(R) = sum_g phi_mu(r_g - tau_I) V(r_g) phi_nu(r_g - tau_J - R) dV   (Eq. 45)
//
// One persistent CTA per SM pulls work items (big cell x point range) from a
// global queue.  Per item (the paper's "BigGrid" batch):
//   A. stage V*dV of the cell's points, the row map and the (entry,entry)->H-offset
//      table in shared memory;
//   B. evaluate phi for every listed (atom image, point) into a dense shared-memory
//      tile  phi[row = orbital][col = point]  (Eq. 1: 4-point Lagrange radial table x
//      real Y_lm) -- each phi value is computed exactly once per call;
//   C. contract  C = phi diag(V dV) phi^T  on the FP64 tensor cores
//      (mma.sync.m8n8k4.f64 -> DMMA.8x8x4; tcgen05 has no FP64 kind), upper
//      triangle only, skipping (8-row fragment, 4-point k-step) pairs that hold no
//      in-sphere point, and add the fragments into the canonical H blocks with
//      red.global.add.f64.
// A second kernel writes every non-canonical block as the transpose of its
// partner, H(J,I,-R) = H(I,J,R)^T, and symmetrises the (I,I,0) blocks.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kTileFrags = 4;   // warp tile = 4 x 4 fragments of 8 x 8

__device__ __forceinline__ void dmma8x8x4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t align16u(uint32_t x) { return (x + 15u) & ~15u; }

__device__ __forceinline__ uint64_t hash_mix(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdULL; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ULL; k ^= k >> 33;
    return k;
}

__device__ __forceinline__ uint32_t block_lookup(const DevicePlan& P, int I, int J, int r1, int r2, int r3) {
    const uint64_t key = (((uint64_t)(uint32_t)I << 44) | ((uint64_t)(uint32_t)J << 24) |
                          ((uint64_t)(uint32_t)(r1 + 128) << 16) | ((uint64_t)(uint32_t)(r2 + 128) << 8) |
                          (uint64_t)(uint32_t)(r3 + 128)) + 1;
    uint32_t h = (uint32_t)hash_mix(key) & P.hash_mask;
    while (true) {
        const uint64_t k = __ldg(P.hash_keys + h);
        if (k == key) return __ldg(P.hash_vals + h);
        if (k == 0) return kNoBlockDev;
        h = (h + 1) & P.hash_mask;
    }
}

struct EInfo {   // per entry, in shared memory
    int32_t row0, norb, atom, Rpack;
};

// k-step mask of an entry restricted to the item's point range: bit s <=> any of
// the 4 points p0+4s .. p0+4s+3 lies inside the entry's sphere.
__device__ __forceinline__ uint32_t kstep_mask(uint32_t mlo, uint32_t mhi, int p0, int npts) {
    uint64_t m = (((uint64_t)mhi << 32) | mlo) >> p0;
    if (npts < 64) m &= (1ull << npts) - 1ull;
    m |= m >> 1;
    m |= m >> 2;             // bit 4s now holds the OR of bits 4s..4s+3
    uint32_t out = 0;
#pragma unroll
    for (int s = 0; s < 16; s++) out |= (uint32_t)((m >> (4 * s)) & 1ull) << s;
    return out;
}

}  // namespace

template <bool TAB_SMEM>
__global__ void __launch_bounds__(kThreads, 1)
gint_vlocal_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ V, double* __restrict__ H) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- shared memory carve-up (mirrors fixed_smem_bytes() in gint_plan.cpp) ----
    uint32_t off = 0;
    double* s_tab = reinterpret_cast<double*>(smem_raw);
    off += TAB_SMEM ? align16u((uint32_t)P.tab_doubles * 8u) : 0u;
    double* s_w = reinterpret_cast<double*>(smem_raw + off);
    off += kMaxItemPointsDev * 8;
    int* s_misc = reinterpret_cast<int*>(smem_raw + off);   // [0] item index, [1] tile counter
    off += 64;
    EInfo* s_einfo = reinterpret_cast<EInfo*>(smem_raw + off);
    off += align16u((uint32_t)P.max_entries * 16u);
    uint16_t* s_rowinfo = reinterpret_cast<uint16_t*>(smem_raw + off);
    off += align16u((uint32_t)P.max_rows_pad * 2u);
    uint32_t* s_fragmask = reinterpret_cast<uint32_t*>(smem_raw + off);
    off += align16u((uint32_t)(P.max_rows_pad / 8) * 4u);
    uint32_t* s_pair = reinterpret_cast<uint32_t*>(smem_raw + off);
    off += align16u((uint32_t)(P.max_entries * P.max_entries) * 4u);
    double* s_phi = reinterpret_cast<double*>(smem_raw + off);

    if (TAB_SMEM) {
        for (int i = tid; i < P.tab_doubles; i += kThreads) s_tab[i] = __ldg(P.tab + i);
    }
    const double* tab = TAB_SMEM ? s_tab : P.tab;

    const int by = P.bcell[1], bz = P.bcell[2];
    const int byz = by * bz;

    while (true) {
        if (tid == 0) s_misc[0] = (int)atomicAdd(P.counter, 1u);
        __syncthreads();   // also: every warp has left phase C of the previous item
        const int item = s_misc[0];
        if (item >= P.nitems) break;
        const WorkItemDev wi = P.items[item];
        const int m = wi.nentry, nrow = wi.nrow, nrow_pad = (nrow + 7) & ~7, npts = wi.npts, p0 = wi.p0;
        const int LD = npts + 4;
        const EntryDev* ent = P.entries + wi.entry0;

        // ---------------- phase A: staging ----------------------------------------
        if (tid == 0) s_misc[1] = 0;
        for (int e = tid; e < m; e += kThreads) {
            EInfo ei;
            ei.row0 = ent[e].row0;
            ei.norb = ent[e].norb;
            ei.atom = ent[e].atom;
            ei.Rpack = ent[e].Rpack;
            s_einfo[e] = ei;
            for (int mu = 0; mu < ei.norb; mu++) s_rowinfo[ei.row0 + mu] = (uint16_t)((e << 6) | mu);
        }
        for (int r = nrow + tid; r < nrow_pad; r += kThreads) s_rowinfo[r] = 0xFFFFu;
        for (int c = tid; c < kMaxItemPointsDev; c += kThreads) {
            double wv = 0.0;
            if (c < npts) {
                const int p = p0 + c;
                const int ix = p / byz, iy = (p - ix * byz) / bz, iz = p - ix * byz - iy * bz;
                const int g1 = wi.origin[0] + ix, g2 = wi.origin[1] + iy, g3 = wi.origin[2] + iz;
                if (ix < P.bcell[0] && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2])
                    wv = __ldg(V + ((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3) * P.dV;
            }
            s_w[c] = wv;
        }
        for (int f = tid; f < nrow_pad / 8; f += kThreads) {
            uint32_t msk = 0;
            for (int e = 0; e < m; e++) {
                const int r0 = ent[e].row0, r1 = r0 + ent[e].norb;
                if (r0 < 8 * f + 8 && r1 > 8 * f) msk |= kstep_mask(ent[e].mask_lo, ent[e].mask_hi, p0, npts);
            }
            s_fragmask[f] = msk;
        }
        for (int idx = tid; idx < m * m; idx += kThreads) {
            const int ea = idx / m, eb = idx - ea * m;
            if (ea > eb) continue;
            const int Ra = ent[ea].Rpack, Rb = ent[eb].Rpack;
            s_pair[idx] = block_lookup(P, ent[ea].atom, ent[eb].atom, ((Rb >> 16) & 0xFF) - ((Ra >> 16) & 0xFF),
                                       ((Rb >> 8) & 0xFF) - ((Ra >> 8) & 0xFF), (Rb & 0xFF) - (Ra & 0xFF));
        }
        for (int idx = tid; idx < (nrow_pad - nrow) * LD; idx += kThreads) s_phi[nrow * LD + idx] = 0.0;

        // ---------------- phase B: phi tile (Eq. 1) ----------------------------------
        {
            const int ngroups = (npts + 31) >> 5;
            for (int task = warp; task < m * ngroups; task += kWarps) {
                const int e = task / ngroups, g = task - e * ngroups;
                const EntryDev en = ent[e];
                const int col = 32 * g + lane;
                const int p = p0 + col;
                const bool colvalid = col < npts;
                const uint32_t mword = (p < 32) ? en.mask_lo : en.mask_hi;
                const bool inside = colvalid && ((mword >> (p & 31)) & 1u);
                double* dst = s_phi + en.row0 * LD + col;
                if (__ballot_sync(0xffffffffu, inside) == 0u) {
                    if (colvalid)
                        for (int mu = 0; mu < en.norb; mu++) dst[mu * LD] = 0.0;
                    continue;
                }
                const int sp = (en.Rpack >> 24) & 0x7F;
                const int32_t* meta = P.sp_meta + 12 * sp;
                const int tab_off = __ldg(meta + 0), ntab = __ldg(meta + 1), nrad = __ldg(meta + 2);
                const double inv_dr = __ldg(P.sp_real + 2 * sp + 1);
                const int ix = p / byz, iy = (p - ix * byz) / bz, iz = p - ix * byz - iy * bz;
                const double dx = en.rel[0] + ix * P.estep[0] + iy * P.estep[3] + iz * P.estep[6];
                const double dy = en.rel[1] + ix * P.estep[1] + iy * P.estep[4] + iz * P.estep[7];
                const double dz = en.rel[2] + ix * P.estep[2] + iy * P.estep[5] + iz * P.estep[8];
                const double r2 = dx * dx + dy * dy + dz * dz;
                double x = 0.0, y = 0.0, z = 0.0, r = 0.0, lnz = 0.0;   // lnz: 1 if l>0 components survive
                if (r2 >= 1e-24) {
                    const double rinv = rsqrt(r2);
                    r = r2 * rinv;
                    x = dx * rinv;
                    y = dy * rinv;
                    z = dz * rinv;
                    lnz = 1.0;
                }
                const double s = r * inv_dr;
                int k = (int)s;
                k = min(k, ntab - 4);
                const double t = s - (double)k;
                const double t1 = 1.0 - t, t2 = 2.0 - t, t3 = 3.0 - t;
                const double in = inside ? 1.0 : 0.0;
                const double L0 = in * (t1 * t2 * t3 * (1.0 / 6.0));
                const double L1 = in * (t * t2 * t3 * 0.5);
                const double L2 = in * (-t * t1 * t3 * 0.5);
                const double L3 = in * (t * t1 * t2 * (1.0 / 6.0));
                const double* Tk = tab + tab_off + (inside ? k : 0) * nrad;
                // real Y_lm, l <= 2 (no Condon-Shortley phase; order fixed in include/gint.h)
                const double Y00 = 0.28209479177387814;
                const double c1 = 0.48860251190291992 * lnz;
                const double c2a = 1.0925484305920792, c2b = 0.31539156525252005 * lnz, c2c = 0.54627421529603959;
                double* o = dst;
                for (int f = 0; f < nrad; f++) {
                    const double fv = Tk[f] * L0 + Tk[nrad + f] * L1 + Tk[2 * nrad + f] * L2 + Tk[3 * nrad + f] * L3;
                    const int l = __ldg(meta + 4 + f);
                    if (l == 0) {
                        if (colvalid) o[0] = fv * Y00;
                        o += LD;
                    } else if (l == 1) {
                        const double g1 = fv * c1;
                        if (colvalid) {
                            o[0] = g1 * y;
                            o[LD] = g1 * z;
                            o[2 * LD] = g1 * x;
                        }
                        o += 3 * LD;
                    } else {
                        const double ga = fv * c2a;
                        if (colvalid) {
                            o[0] = ga * (x * y);
                            o[LD] = ga * (y * z);
                            o[2 * LD] = (fv * c2b) * (3.0 * z * z - 1.0);
                            o[3 * LD] = ga * (x * z);
                            o[4 * LD] = (fv * c2c) * (x * x - y * y);
                        }
                        o += 5 * LD;
                    }
                }
            }
        }
        __syncthreads();

        // ---------------- phase C: C = phi diag(w) phi^T, upper triangle ----------------
        {
            const int NF = nrow_pad >> 3;
            const int NT = (NF + kTileFrags - 1) / kTileFrags;
            const int ntiles = NT * (NT + 1) / 2;
            const int nk = npts >> 2;
            const int frow = lane >> 2, fk = lane & 3;
            while (true) {
                int t = 0;
                if (lane == 0) t = atomicAdd(&s_misc[1], 1);
                t = __shfl_sync(0xffffffffu, t, 0);
                if (t >= ntiles) break;
                // tile index -> (ti <= tj), column-major over the upper triangle, large tj first
                t = ntiles - 1 - t;
                int tj = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
                while ((tj + 1) * (tj + 2) / 2 <= t) tj++;
                while (tj * (tj + 1) / 2 > t) tj--;
                const int ti = t - tj * (tj + 1) / 2;
                const int fi0 = kTileFrags * ti, fj0 = kTileFrags * tj;
                uint32_t rmask[kTileFrags], cmask[kTileFrags];
#pragma unroll
                for (int i = 0; i < kTileFrags; i++) {
                    rmask[i] = (fi0 + i < NF) ? s_fragmask[fi0 + i] : 0u;
                    cmask[i] = (fj0 + i < NF) ? s_fragmask[fj0 + i] : 0u;
                }
                double acc[kTileFrags][kTileFrags][2];
#pragma unroll
                for (int i = 0; i < kTileFrags; i++)
#pragma unroll
                    for (int j = 0; j < kTileFrags; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
                const double* pa = s_phi + (8 * fi0 + frow) * LD + fk;
                const double* pb = s_phi + (8 * fj0 + frow) * LD + fk;
                for (int s = 0; s < nk; s++) {
                    uint32_t ra = 0, ca = 0;
#pragma unroll
                    for (int i = 0; i < kTileFrags; i++) {
                        ra |= ((rmask[i] >> s) & 1u) << i;
                        ca |= ((cmask[i] >> s) & 1u) << i;
                    }
                    if (ra == 0u || ca == 0u) continue;
                    const double wv = s_w[4 * s + fk];
                    double a[kTileFrags], b[kTileFrags];
#pragma unroll
                    for (int i = 0; i < kTileFrags; i++) {
                        a[i] = ((ra >> i) & 1u) ? pa[(8 * i) * LD + 4 * s] : 0.0;
                        b[i] = ((ca >> i) & 1u) ? wv * pb[(8 * i) * LD + 4 * s] : 0.0;
                    }
#pragma unroll
                    for (int i = 0; i < kTileFrags; i++)
#pragma unroll
                        for (int j = 0; j < kTileFrags; j++)
                            if (((ra >> i) & 1u) && ((ca >> j) & 1u) && (fi0 + i <= fj0 + j))
                                dmma8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
                // ---- flush: add the fragments into the canonical H blocks ----
#pragma unroll
                for (int i = 0; i < kTileFrags; i++) {
                    if (rmask[i] == 0u) continue;
                    const int r = 8 * (fi0 + i) + frow;
                    const uint32_t ri = s_rowinfo[r];
                    if (ri == 0xFFFFu) continue;
                    const int ea = ri >> 6, mu = ri & 63;
#pragma unroll
                    for (int j = 0; j < kTileFrags; j++) {
                        if ((rmask[i] & cmask[j]) == 0u || (fi0 + i > fj0 + j)) continue;
#pragma unroll
                        for (int h = 0; h < 2; h++) {
                            const int c = 8 * (fj0 + j) + 2 * fk + h;
                            const uint32_t ci = s_rowinfo[c];
                            if (ci == 0xFFFFu || r > c) continue;
                            const int eb = ci >> 6, nu = ci & 63;
                            const uint32_t base = s_pair[ea * m + eb];
                            if (base == kNoBlockDev) continue;
                            atomicAdd(H + (size_t)base + (size_t)(mu * s_einfo[eb].norb + nu), acc[i][j][h]);
                        }
                    }
                }
            }
        }
        // loop-top __syncthreads separates phase C from the next item's staging
    }
}

// H(J,I,-R) = H(I,J,R)^T for every non-canonical block; lower <- upper for (I,I,0).
__global__ void __launch_bounds__(256) gint_mirror_kernel(const MirrorItemDev* __restrict__ items, int nitems,
                                                          double* __restrict__ H) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= nitems) return;
    const MirrorItemDev it = items[w];
    const int n = it.nI * it.nJ;
    if (it.src == it.dst) {
        for (int idx = lane; idx < n; idx += 32) {
            const int mu = idx / it.nJ, nu = idx - mu * it.nJ;
            if (mu > nu) H[(size_t)it.dst + idx] = H[(size_t)it.dst + nu * it.nJ + mu];
        }
    } else {
        for (int idx = lane; idx < n; idx += 32) {
            const int mu = idx / it.nJ, nu = idx - mu * it.nJ;
            H[(size_t)it.dst + idx] = H[(size_t)it.src + nu * it.nI + mu];
        }
    }
}

// ---- launchers -----------------------------------------------------------------------
cudaError_t configure_kernels(const DevicePlan& P, size_t smem_bytes, bool tab_smem) {
    (void)P;
    if (tab_smem)
        return cudaFuncSetAttribute(gint_vlocal_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    return cudaFuncSetAttribute(gint_vlocal_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
}

cudaError_t launch_vlocal(const DevicePlan& P, size_t smem_bytes, bool tab_smem, int nsm, size_t h_len,
                          const double* V, double* H, cudaStream_t stream, cudaEvent_t* ev) {
    if (ev) cudaEventRecord(ev[0], stream);
    cudaError_t e = cudaMemsetAsync(H, 0, h_len * sizeof(double), stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int), stream);
    if (e != cudaSuccess) return e;
    if (ev) cudaEventRecord(ev[1], stream);
    if (P.nitems > 0) {
        const int grid = P.nitems < nsm ? P.nitems : nsm;
        if (tab_smem)
            gint_vlocal_kernel<true><<<grid, kThreads, smem_bytes, stream>>>(P, V, H);
        else
            gint_vlocal_kernel<false><<<grid, kThreads, smem_bytes, stream>>>(P, V, H);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[2], stream);
    if (P.nmirror > 0) {
        const int wpb = 256 / 32;
        gint_mirror_kernel<<<(P.nmirror + wpb - 1) / wpb, 256, 0, stream>>>(P.mirror, P.nmirror, H);
        e = cudaGetLastError();
    }
    if (ev) cudaEventRecord(ev[3], stream);
    return e;
}

// ---- FP64 tensor peak: register-resident DMMA.8x8x4 loop --------------------------------
__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out, int iters, double a0, double b0) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = 0.0;
    const double a = a0 + threadIdx.x * 1e-9, b = b0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma8x8x4(c[i][0], c[i][1], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

cudaError_t measure_dmma_peak(double seconds, int nsm, double* tflops) {
    double* out = nullptr;
    cudaError_t e = cudaMalloc(&out, 64);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 20000, grid = nsm * 4, threads = 256;   // 32 warps per SM
    dmma_peak_kernel<<<grid, threads>>>(out, iters, 1.0, 1.0);
    e = cudaDeviceSynchronize();
    double best = 0, total_ms = 0;
    while (e == cudaSuccess && total_ms < seconds * 1e3) {
        cudaEventRecord(e0);
        dmma_peak_kernel<<<grid, threads>>>(out, iters, 1.0, 1.0);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms;
        const double tf = (double)grid * (threads / 32) * (double)iters * 8.0 * 512.0 / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = best;
    return e;
}

}  // namespace gint
