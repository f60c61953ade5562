// gint_fvl.cu -- local Pulay force (the paper's cal_gint_fvl), PAPER.md:400-411 (Sec. 3.3.1, Eq. 46):
//
//   F_K = - sum_blocks sum_{mu nu} D(I,J,R)[mu][nu] dH(I,J,R)[mu][nu] / d tau_K      at fixed V and D,
//
// the derivative acting on phi_mu when K = I and on phi_nu when K = J; "the derivatives of the NAOs are computed
// analytically for the angular part (real spherical harmonics) and numerically for the radial part"
// -- here the derivative of the same cubic Lagrange interpolant that defines f(r).
//
// Per region (the plan's BigGrid) with its entries (atom images) c, e and rows kappa, lambda:
//
//   F_{I_c} += sum_p V(p) dV sum_{kappa in c} grad phi_kappa(p) T_kappa(p),     T = E Phi,
//   E[kappa of c][lambda of e] = D(I_c, I_e, R_e - R_c)[kappa][lambda] + D(I_e, I_c, R_c - R_e)[lambda][kappa],
//
// i.e. entry c collects its row role in the blocks (I_c, I_e, .) and its column role in the blocks (I_e, I_c, .).
// Three kernels after gint_psi_kernel (unit weights, Phi in the psi scratch):
//   gint_egather_kernel  E of every region, dense, in DMMA A-fragment order (32 x 32 sub-blocks of 8 KB)
//   gint_tgemm_kernel    T = E Phi per region on the FP64 tensor pipe (DMMA.8x8x4): CTA tile 128 rows x 128 points,
//                        16 warps x (32 rows x 32 points), K = the region's row groups streamed through a 3-deep
//                        shared-memory ring with cp.async.bulk + full / empty mbarriers; (row group, stage) pairs without an
//                        in-sphere point are skipped; T is written in the psi chunk layout
//   gint_force_kernel    per (entry, 32-point stage): V dV, grad phi (analytic angular part, interpolant derivative),
//                        dot with T, warp reduction, three atomics per task into F
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

namespace {

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bar_expect(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D_%=;\n\t"
        "bra W_%=;\n\t"
        "D_%=:\n\t}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_copy(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// a (row group, stage) pair holds an in-sphere point
__device__ __forceinline__ bool group_stage_active(const FvlPlan& F, const Region* reg, int g, int stage) {
    const uint8_t* gm = F.gmask + __ldg(&reg->gmask_off) + (size_t)g * F.nks_pad + (size_t)stage * kStageKsteps;
    return *reinterpret_cast<const unsigned long long*>(gm) != 0ull;
}

// 16 bits: nibble j = fragments of row group g with an in-sphere point in k-pair j (8 points) of the stage
__device__ __forceinline__ uint32_t kpair_masks(const FvlPlan& F, const Region* reg, int g, int stage) {
    const uint8_t* gm = F.gmask + __ldg(&reg->gmask_off) + (size_t)g * F.nks_pad + (size_t)stage * kStageKsteps;
    const uint2 w = __ldg(reinterpret_cast<const uint2*>(gm));   // 8 k-steps, one byte each (low nibble)
    const uint32_t a = (w.x | (w.x >> 8)) & 0x000F000Fu, b = (w.y | (w.y >> 8)) & 0x000F000Fu;
    return (a & 0xFu) | ((a >> 12) & 0xF0u) | ((b & 0xFu) << 8) | ((b >> 4) & 0xF000u);
}

}  // namespace

// ---- E = D + D^T of every region, A-fragment order -------------------------------------------------------
// chunk (ga, gb) of region r sits at (e_chunk0[r] + ga * ngroup + gb) * 1024 doubles; inside: [kc 8][i 4][lane 32],
// element = E[row 32 ga + 8 i + lane / 4][column 32 gb + 4 kc + lane % 4].
__global__ void __launch_bounds__(256) gint_egather_kernel(const __grid_constant__ DevicePlan P, const __grid_constant__ FvlPlan F,
                                                           const double* __restrict__ D) {
    const int reg_index = __ldg(P.work_regions + blockIdx.x);
    const Region* reg = P.regions + reg_index;
    const int ngroup = __ldg(&reg->ngroup), m = __ldg(&reg->nentry);
    const uint32_t* rinfo = F.rowinfo + __ldg(&reg->rowinfo_off);
    const uint32_t* pdir = P.pair_direct + __ldg(&reg->pair_off);
    double* E = F.escratch + (size_t)__ldg(F.e_chunk0 + reg_index) * kChunkDoubles;
    const int nchunk = ngroup * ngroup;
    for (int idx = threadIdx.x; idx < nchunk * kChunkDoubles; idx += blockDim.x) {
        const int ch = idx >> 10, e = idx & 1023;
        const int ga = ch / ngroup, gb = ch - ga * ngroup;
        const int kc = e >> 7, i = (e >> 5) & 3, lane = e & 31;
        const uint32_t ri = __ldg(rinfo + ga * 32 + 8 * i + (lane >> 2));
        const uint32_t ci = __ldg(rinfo + gb * 32 + 4 * kc + (lane & 3));
        double v = 0.0;
        if (ri != kNoBlock && ci != kNoBlock) {
            const int ea = ri & 0xFFF, mu = (ri >> 12) & 0xFF, nI = ri >> 20;
            const int eb = ci & 0xFFF, nu = (ci >> 12) & 0xFF, nJ = ci >> 20;
            const uint32_t o1 = __ldg(pdir + ea * m + eb), o2 = __ldg(pdir + eb * m + ea);
            if (o1 != kNoBlock) v += __ldg(D + o1 + mu * nJ + nu);
            if (o2 != kNoBlock) v += __ldg(D + o2 + nu * nI + mu);
        }
        E[idx] = v;
    }
}

// ---- T = E Phi ----------------------------------------------------------------------------------------------
constexpr int kTgThreads = 512;
constexpr int kTgBufBytes = 8 * kChunkBytes;          // 4 E sub-blocks + 4 psi chunks
constexpr int kTgRing = 3;                            // K steps in flight
constexpr int kTgSmem = kTgRing * kTgBufBytes + 64;

__global__ void __launch_bounds__(kTgThreads, 1)
gint_tgemm_kernel(const __grid_constant__ DevicePlan P, const __grid_constant__ FvlPlan F) {
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kTgRing * kTgBufBytes);   // full[3], empty[3]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int4 task = __ldg(F.tg_tasks + blockIdx.x);   // region, row quad, stage quad
    const Region* reg = P.regions + task.x;
    const int ngroup = __ldg(&reg->ngroup), nstage = P.nstage;
    const int ga = 4 * task.y + (warp >> 2), stage = 4 * task.z + (warp & 3);
    const bool mine = ga < ngroup && stage < nstage && group_stage_active(F, reg, ga, stage);
    const double* Ebase = F.escratch + (size_t)__ldg(F.e_chunk0 + task.x) * kChunkDoubles;
    const double* psi_region = P.psi + (size_t)__ldg(&reg->psi_chunk0) * kChunkDoubles;
    if (tid == 0) {
        for (int i = 0; i < kTgRing; i++) {
            bar_init(smem_addr(bars + i), 1);
            bar_init(smem_addr(bars + kTgRing + i), kTgThreads / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async;" ::: "memory");
    __syncthreads();
    // thread 0 streams, per column group gb: E(4 rq + i, gb) and Phi(gb, 4 sq + j), i, j = 0..3
    auto issue = [&](int gb) {
        const uint32_t buf = smem_addr(smem) + (gb % kTgRing) * kTgBufBytes, bar = smem_addr(bars + gb % kTgRing);
        uint32_t n = 0;
        bool e_on[4], p_on[4];
        for (int i = 0; i < 4; i++) {
            e_on[i] = 4 * task.y + i < ngroup;
            p_on[i] = 4 * task.z + i < nstage && group_stage_active(F, reg, gb, 4 * task.z + i);
            n += (e_on[i] ? 1u : 0u) + (p_on[i] ? 1u : 0u);
        }
        if (n) bar_expect(bar, n * kChunkBytes);
        else bar_arrive(bar);
        for (int i = 0; i < 4; i++) {
            if (e_on[i])
                bulk_copy(buf + i * kChunkBytes, Ebase + ((size_t)(4 * task.y + i) * ngroup + gb) * kChunkDoubles, kChunkBytes, bar);
            if (p_on[i])
                bulk_copy(buf + (4 + i) * kChunkBytes, psi_region + ((size_t)gb * nstage + 4 * task.z + i) * kChunkDoubles, kChunkBytes, bar);
        }
    };
    if (tid == 0) {
        issue(0);
        if (ngroup > 1) issue(1);
    }
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
    const int q = lane >> 2, r = lane & 3;
    // B operand of (kc, j): Phi[row 4 kc + r of gb][point 8 j + q]; point 8 j + q is point q % 4 of k-step 2 j + q / 4
    const int boff = (q >> 2) * 128 + (r >> 1) * 8 + (q & 3) * 2 + (r & 1);
    const uint32_t rp = mine ? kpair_masks(F, reg, ga, stage) : 0u;   // row fragments of ga active per k-pair
    // bit j: some row fragment of ga is active in k-pair j
    const uint32_t rj_any = ((rp & 0xFu) ? 1u : 0u) | ((rp & 0xF0u) ? 2u : 0u) | ((rp & 0xF00u) ? 4u : 0u) | ((rp & 0xF000u) ? 8u : 0u);
    for (int gb = 0; gb < ngroup; gb++) {
        // K step gb + 2 goes into the buffer of K step gb - 1 once all 16 warps have released it; the warps take turns at
        // waiting for that (no block-wide barrier: a warp whose tile is sparse runs ahead by up to two K steps)
        if (warp == (gb & 15) && gb + 2 < ngroup) {
            if (lane == 0) {
                if (gb >= 1) bar_wait(smem_addr(bars + kTgRing + (gb + 2) % kTgRing), (uint32_t)((gb + 2) / kTgRing - 1) & 1u);
                issue(gb + 2);
            }
            __syncwarp();
        }
        bar_wait(smem_addr(bars + gb % kTgRing), (uint32_t)(gb / kTgRing) & 1u);
        const uint32_t cp = mine ? kpair_masks(F, reg, gb, stage) : 0u;   // column fragments of gb active per k-pair
        if (cp) {
            const double* bufE = reinterpret_cast<const double*>(smem + (gb % kTgRing) * kTgBufBytes + (warp >> 2) * kChunkBytes) + lane;
            const double* bufP = reinterpret_cast<const double*>(smem + (gb % kTgRing) * kTgBufBytes + (4 + (warp & 3)) * kChunkBytes) + boff;
            if ((rp & cp) == 0xFFFFu) {   // every fragment active in every k-pair: dense
#pragma unroll 2
                for (int kc = 0; kc < 8; kc++) {
                    double a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) a[i] = bufE[(kc * 4 + i) * 32];
#pragma unroll
                    for (int j = 0; j < 4; j++) b[j] = bufP[j * 256 + kc * 16];
#pragma unroll
                    for (int i = 0; i < 4; i++)
#pragma unroll
                        for (int j = 0; j < 4; j++) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            } else {
                // blocks of 8 DMMAs (column fragment f = columns 8 f .. 8 f + 7, k-pair j = 8 points, all four row
                // fragments) only where the column fragment holds an in-sphere point in the k-pair and some row of the
                // group does too.  Real, warp-uniform branches (a predicated-off DMMA still costs its pipe cycles, hence
                // the never-taken back edges); 8 DMMAs on 4 accumulators keep the pipe busy by themselves.
#pragma unroll
                for (int f = 0; f < 4; f++) {
                    const uint32_t jm = ((cp >> f) & 1u) | (((cp >> (4 + f)) & 1u) << 1) | (((cp >> (8 + f)) & 1u) << 2) | (((cp >> (12 + f)) & 1u) << 3);
                    if ((jm & rj_any) == 0u) continue;
                    double a0[4], a1[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        a0[i] = bufE[(8 * f + i) * 32];
                        a1[i] = bufE[(8 * f + 4 + i) * 32];
                    }
#pragma unroll
                    for (int j = 0; j < 4; j++) {
                        if ((jm & rj_any) & (1u << j)) {
                            do {
                                const double b0 = bufP[j * 256 + (2 * f) * 16], b1 = bufP[j * 256 + (2 * f + 1) * 16];
#pragma unroll
                                for (int i = 0; i < 4; i++) dmma(acc[i][j][0], acc[i][j][1], a0[i], b0);
#pragma unroll
                                for (int i = 0; i < 4; i++) dmma(acc[i][j][0], acc[i][j][1], a1[i], b1);
                            } while (P.never);
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) bar_arrive(smem_addr(bars + kTgRing + gb % kTgRing));   // this warp is done with the buffer
    }
    if (mine) {   // T tile -> scratch, psi chunk layout: (row R, point 4 ks + k) at ks * 128 + (R / 2) * 8 + k * 2 + R % 2
        double* Tc = F.tscratch + ((size_t)__ldg(&reg->psi_chunk0) + (size_t)ga * nstage + stage) * kChunkDoubles;
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < 4; j++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int R = 8 * i + q, pp = 2 * r + h;
                    Tc[(2 * j + (pp >> 2)) * 128 + (R >> 1) * 8 + (pp & 3) * 2 + (R & 1)] = acc[i][j][h];
                }
    }
}

// ---- F_c += sum_p V dV sum_kappa grad phi_kappa T_kappa ----------------------------------------------------------
namespace {

struct SpeciesF {
    int32_t tab_off, ntab, nradp, nrad;
    int32_t l[8];
    double rc2, inv_dr;
};

__device__ __forceinline__ double rsqrt_seed_f(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

}  // namespace

constexpr int kFvThreads = 256;

template <bool TAB_SMEM>
__global__ void __launch_bounds__(kFvThreads, 2)
gint_force_kernel(const __grid_constant__ DevicePlan P, const __grid_constant__ FvlPlan F, const double* __restrict__ V,
                  double* __restrict__ Fout) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* s_off = reinterpret_cast<double*>(smem_raw);                              // [3][512]
    uchar4* s_xyz = reinterpret_cast<uchar4*>(smem_raw + 3 * kMaxRegionPoints * 8);    // [512]
    double* s_w = reinterpret_cast<double*>(smem_raw + 3 * kMaxRegionPoints * 8 + kMaxRegionPoints * 4);   // [512]
    SpeciesF* s_spec = reinterpret_cast<SpeciesF*>(smem_raw + 4 * kMaxRegionPoints * 8 + kMaxRegionPoints * 4);
    double* s_tab = reinterpret_cast<double*>(smem_raw + 4 * kMaxRegionPoints * 8 + kMaxRegionPoints * 4 +
                                              smem_align((size_t)P.nspecies * sizeof(SpeciesF)));
    if (TAB_SMEM)
        for (int i = tid; i < P.tab_doubles; i += kFvThreads) s_tab[i] = __ldg(P.tab + i);
    for (int i = tid; i < P.nspecies; i += kFvThreads) {
        const int32_t* meta = P.sp_meta + 12 * i;
        SpeciesF sd;
        sd.tab_off = meta[0]; sd.ntab = meta[1]; sd.nradp = meta[2];
        sd.nrad = 0;
        for (int k = 0; k < 8; k++) { sd.l[k] = meta[4 + k]; if (meta[4 + k] >= 0) sd.nrad = k + 1; }
        sd.rc2 = P.sp_real[2 * i]; sd.inv_dr = P.sp_real[2 * i + 1];
        s_spec[i] = sd;
    }
    const double* tab = TAB_SMEM ? s_tab : P.tab;
    const int npt = P.nstage * kStagePts;
    for (int p = tid; p < npt; p += kFvThreads) {
        const uchar4 c = reinterpret_cast<const uchar4*>(P.slot_xyz)[p];
        for (int k = 0; k < 3; k++)
            s_off[k * kMaxRegionPoints + p] = c.x * P.estep[k] + c.y * P.estep[3 + k] + c.z * P.estep[6 + k];
        s_xyz[p] = c;
    }
    for (int rr = blockIdx.x; rr < P.nwork_regions; rr += gridDim.x) {
        __syncthreads();
        const Region* reg = P.regions + __ldg(P.work_regions + rr);
        const int ox = __ldg(&reg->origin[0]), oy = __ldg(&reg->origin[1]), oz = __ldg(&reg->origin[2]);
        for (int p = tid; p < npt; p += kFvThreads) {
            const uchar4 c = s_xyz[p];
            const int g1 = ox + c.x, g2 = oy + c.y, g3 = oz + c.z;
            double wv = 0.0;
            if (c.w && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2])
                wv = __ldg(V + ((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3) * P.dV;
            s_w[p] = wv;
        }
        __syncthreads();
        const int ntask = __ldg(&reg->ntask);
        const uint32_t* tasks = P.etasks + __ldg(&reg->task_off);
        const Entry* entries = P.entries + __ldg(&reg->entry0);
        const double* T_region = F.tscratch + (size_t)__ldg(&reg->psi_chunk0) * kChunkDoubles;
        const int gstride = P.nstage * kChunkDoubles;
        for (int t = warp; t < ntask; t += kFvThreads / 32) {
            const uint32_t tk = __ldg(tasks + t);
            const Entry* en = entries + (tk & 0xFFFFu);
            const int s0 = (int)(tk >> 16) * 8;
            const double relx = __ldg(&en->rel[0]), rely = __ldg(&en->rel[1]), relz = __ldg(&en->rel[2]);
            const int spi = (__ldg(&en->Rpack) >> 24) & 0x7F, row0 = __ldg(&en->row0), atom = __ldg(&en->atom);
            const uint2 km = __ldg(reinterpret_cast<const uint2*>(&en->kmask[s0 >> 2]));
            const SpeciesF& sp = s_spec[spi];
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int qs = 0; qs < 8 && s0 + qs < P.nstage; qs++) {
                if ((((qs < 4 ? km.x : km.y) >> (8 * (qs & 3))) & 0xFFu) == 0u) continue;
                const int stage = s0 + qs, p = stage * kStagePts + lane;
                const double dx = relx + s_off[p], dy = rely + s_off[kMaxRegionPoints + p], dz = relz + s_off[2 * kMaxRegionPoints + p];
                const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
                const bool inside = r2 < sp.rc2;
                double rinv = 0.0;
                const bool nz = r2 >= 1e-24;   // r >= 1e-12
                if (nz) {
                    const double y0 = rsqrt_seed_f(r2);
                    const double e = fma(-(r2 * y0), y0, 1.0);
                    rinv = fma(e * y0, fma(0.375, e, 0.5), y0);
                }
                const double r = r2 * rinv;
                const double x = dx * rinv, y = dy * rinv, z = dz * rinv;
                const double s = r * sp.inv_dr;
                int k = __double2int_rd(s);
                const double tt = s - (double)k;
                k = inside ? min(k, sp.ntab) : sp.ntab;   // outside: the four zero nodes after the table
                const double t1 = 1.0 - tt, t2 = 2.0 - tt, t3 = 3.0 - tt;
                const double L0 = t1 * t2 * t3 * (1.0 / 6.0), L1 = tt * t2 * t3 * 0.5, L2 = tt * t1 * t3 * -0.5, L3 = tt * t1 * t2 * (1.0 / 6.0);
                // d/dt of the four Lagrange weights, times 1 / dr
                const double D0 = -(t2 * t3 + t1 * t3 + t1 * t2) * (1.0 / 6.0) * sp.inv_dr;
                const double D1 = (t2 * t3 - tt * t3 - tt * t2) * 0.5 * sp.inv_dr;
                const double D2 = -(t1 * t3 - tt * t3 - tt * t1) * 0.5 * sp.inv_dr;
                const double D3 = (t1 * t2 - tt * t2 - tt * t1) * (1.0 / 6.0) * sp.inv_dr;
                const double* Tk = tab + sp.tab_off + k * sp.nradp;
                const double* Tl = T_region + (size_t)stage * kChunkDoubles + (lane >> 2) * 128 + (lane & 3) * 2;
                int R = row0;
                auto tval = [&]() {
                    const double v = Tl[(R >> 5) * gstride + ((R & 31) >> 1) * 8 + (R & 1)];
                    R++;
                    return v;
                };
                double gx = 0.0, gy = 0.0, gz = 0.0;
                for (int f = 0; f < sp.nrad; f++) {
                    const double a0 = Tk[f], a1 = Tk[sp.nradp + f], a2 = Tk[2 * sp.nradp + f], a3 = Tk[3 * sp.nradp + f];
                    const double fv = fma(a0, L0, fma(a1, L1, fma(a2, L2, a3 * L3)));
                    const double fd = fma(a0, D0, fma(a1, D1, fma(a2, D2, a3 * D3)));
                    const int l = sp.l[f];
                    if (l == 0) {
                        const double c = fd * tval();
                        gx = fma(c, x, gx); gy = fma(c, y, gy); gz = fma(c, z, gz);
                    } else if (l == 1) {
                        const double qq = nz ? fv * rinv : fd;   // f / r, and its limit f'(0) at r = 0
                        const double ty = tval(), tz = tval(), tx = tval();
                        const double A = fma(ty, y, fma(tz, z, tx * x)) * (fd - qq);
                        gx = fma(A, x, fma(qq, tx, gx)); gy = fma(A, y, fma(qq, ty, gy)); gz = fma(A, z, fma(qq, tz, gz));
                    } else if (l == 3) {
                        // homogeneous cubic forms (table carries 1/2 sqrt(105/pi)) and their gradients
                        const double qq = fv * rinv;
                        const double ca = 0.20412414523193151, cc = 0.15811388300841897, cd = 0.12909944487358055;
                        const double u0 = tval() * ca, u1 = tval(), u2 = tval() * cc, u3 = tval() * cd, u4 = tval() * cc, u5 = tval() * 0.5, u6 = tval() * ca;
                        const double x2 = x * x, y2 = y * y, z2 = z * z, h = 4.0 * z2 - x2 - y2;
                        const double A = (u0 * y * (3.0 * x2 - y2) + u1 * x * y * z + u2 * y * h + u3 * z * (2.0 * z2 - 3.0 * x2 - 3.0 * y2) +
                                          u4 * x * h + u5 * z * (x2 - y2) + u6 * x * (x2 - 3.0 * y2)) * (fd - 3.0 * qq);
                        const double bx = u0 * 6.0 * x * y + u1 * y * z - 2.0 * u2 * x * y - 6.0 * u3 * x * z + u4 * (h - 2.0 * x2) + 2.0 * u5 * x * z + 3.0 * u6 * (x2 - y2);
                        const double by = 3.0 * u0 * (x2 - y2) + u1 * x * z + u2 * (h - 2.0 * y2) - 6.0 * u3 * y * z - 2.0 * u4 * x * y - 2.0 * u5 * y * z - 6.0 * u6 * x * y;
                        const double bz = u1 * x * y + 8.0 * u2 * y * z + u3 * (6.0 * z2 - 3.0 * x2 - 3.0 * y2) + 8.0 * u4 * x * z + u5 * (x2 - y2);
                        gx = fma(A, x, fma(qq, bx, gx)); gy = fma(A, y, fma(qq, by, gy)); gz = fma(A, z, fma(qq, bz, gz));
                    } else {
                        const double qq = fv * rinv;
                        const double c2 = 0.28867513459481288;
                        const double u0 = tval(), u1 = tval(), u2 = tval() * c2, u3 = tval(), u4 = tval();
                        const double zz = nz ? 1.0 : 0.0;
                        const double A = (u0 * (x * y) + u1 * (y * z) + u2 * fma(3.0 * z, z, -zz) + u3 * (x * z) + u4 * (0.5 * fma(x, x, -(y * y)))) *
                                         (fd - 2.0 * qq);
                        const double bx = fma(u0, y, fma(-2.0 * u2, x, fma(u3, z, u4 * x)));
                        const double by = fma(u0, x, fma(u1, z, fma(-2.0 * u2, y, -(u4 * y))));
                        const double bz = fma(u1, y, fma(4.0 * u2, z, u3 * x));
                        gx = fma(A, x, fma(qq, bx, gx)); gy = fma(A, y, fma(qq, by, gy)); gz = fma(A, z, fma(qq, bz, gz));
                    }
                }
                const double w = s_w[p];
                fx = fma(w, gx, fx); fy = fma(w, gy, fy); fz = fma(w, gz, fz);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                fx += __shfl_xor_sync(0xffffffffu, fx, o);
                fy += __shfl_xor_sync(0xffffffffu, fy, o);
                fz += __shfl_xor_sync(0xffffffffu, fz, o);
            }
            if (lane == 0) {
                atomicAdd(Fout + 3 * atom, fx);
                atomicAdd(Fout + 3 * atom + 1, fy);
                atomicAdd(Fout + 3 * atom + 2, fz);
            }
        }
    }
}

// ---- launcher ---------------------------------------------------------------------------------------------------
size_t force_kernel_smem(size_t table_bytes, int nspecies) {
    return 4 * kMaxRegionPoints * 8 + kMaxRegionPoints * 4 + smem_align((size_t)nspecies * sizeof(SpeciesF)) + smem_align(table_bytes);
}

cudaError_t configure_fvl(size_t force_smem, bool tab_smem) {
    cudaError_t e = cudaFuncSetAttribute(gint_tgemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTgSmem);
    if (e != cudaSuccess) return e;
    return tab_smem ? cudaFuncSetAttribute(gint_force_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)force_smem)
                    : cudaFuncSetAttribute(gint_force_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)force_smem);
}

// F <- 0; per batch of regions: Phi (psi kernel with unit weights), E gather, T = E Phi, force kernel
cudaError_t launch_fvl(const DevicePlan& P, const FvlPlan& F, size_t psi_smem, size_t force_smem, bool tab_smem, int nsm,
                       int natom, const BatchRange* batches, const int32_t* tg0, int nbatch, const double* V, const double* D,
                       double* Fout, cudaStream_t stream) {
    cudaError_t e = cudaMemsetAsync(Fout, 0, (size_t)natom * 3 * sizeof(double), stream);
    if (e != cudaSuccess) return e;
    for (int b = 0; b < nbatch; b++) {
        const DevicePlan Q = batch_plan(P, batches[b]);
        if (Q.nwork_regions <= 0 || Q.nitems <= 0) continue;
        if ((e = launch_psi(Q, psi_smem, tab_smem, nsm, nullptr, stream)) != cudaSuccess) return e;
        gint_egather_kernel<<<Q.nwork_regions, 256, 0, stream>>>(Q, F, D);
        FvlPlan G = F;
        G.tg_tasks = F.tg_tasks + tg0[b];
        G.ntg = tg0[b + 1] - tg0[b];
        if (G.ntg > 0) gint_tgemm_kernel<<<G.ntg, kTgThreads, kTgSmem, stream>>>(Q, G);
        const int grid = Q.nwork_regions < 2 * nsm ? Q.nwork_regions : 2 * nsm;
        if (tab_smem) gint_force_kernel<true><<<grid, kFvThreads, force_smem, stream>>>(Q, F, V, Fout);
        else gint_force_kernel<false><<<grid, kFvThreads, force_smem, stream>>>(Q, F, V, Fout);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace gint
