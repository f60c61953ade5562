// gint_kernels.cu -- sm_100a kernels of gint_vlocal.
//
//   H_mu,nu(R) = sum_g phi_mu(r_g - tau_I) V(r_g) phi_nu(r_g - tau_J - R) dV   (Eq. 45)
//
// Two kernels per call, both behind gint_vlocal (plus a tiny mirror kernel):
//
//   gint_psi_kernel     psi = phi sqrt(|V dV|) for every (atom image, mesh point) pair listed by
//       the plan, evaluated exactly once -- Eq. 1: 4-point Lagrange radial table x real Y_lm, one
//       lane per mesh point -- and stored to a scratch buffer in DMMA fragment order, together
//       with the sign bits of V per region.  The V dV weighting of Eq. 45 is thereby folded into
//       the operand: C = psi diag(sign V) psi^T.
//   gint_contract_kernel<0>  (gint_vlocal) output-stationary contraction (the paper's per-BigGrid dense contraction,
//       PAPER.md:380, 413).  One persistent CTA per SM pulls work items from a global queue; a
//       work item is a set of up to 15 32x32 tiles (one per consumer warp) of the upper triangle
//       of one region's C.  A producer warp stages the item descriptor and streams the row groups
//       the tiles need through a ring of shared-memory stages (32 points each) with
//       cp.async.bulk + mbarrier, running ahead across item boundaries; the 15 consumer warps
//       keep their tile in registers and issue mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4; tcgen05 has
//       no FP64 kind).  (fragment, k-step) pairs that hold no in-sphere point are skipped by
//       warp-uniform branches on host-built activity nibbles (a predicated-off DMMA still costs
//       its 16 pipe cycles).  After the last stage the warp adds its tile into the canonical H
//       blocks with red.global.add.f64 (once per item, not once per BigGrid).
//   gint_mirror_kernel  writes every non-canonical block as the transpose of its partner,
//       H(J,I,-R) = H(I,J,R)^T, and symmetrises the (I,I,0) blocks.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"

namespace gint {

namespace {

#ifdef GINT_TIMING   // development only: per-CTA clock64 breakdown written behind the ready counters
#define TIMER_DECL long long tm_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; long long t0_ = 0; (void)t0_;
#define TIMER_START t0_ = clock64();
#define TIMER_ADD(k) tm_[k] += clock64() - t0_;
#define TIMER_COUNT(k) tm_[k] += 1;
#else
#define TIMER_DECL
#define TIMER_START
#define TIMER_ADD(k)
#define TIMER_COUNT(k)
#endif

constexpr int kConsumerWarps = kTilesPerItem;          // 7
constexpr int kConsumerThreads = kConsumerWarps * 32;  // 224
constexpr int kThreads = kConsumerThreads + 32;        // + 1 producer warp
constexpr int kStageBytes = kMaxSlots * kChunkBytes;   // 32 KB

__device__ __forceinline__ void dmma8x8x4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// DMMAs under warp-uniform conditions.  A predicated-off DMMA still holds the FP64 tensor pipe for its
// 16 cycles (measured), and ptxas if-converts a plain `if` around a few of them into exactly that; a
// never-taken back edge (`never` is always 0 at run time) makes the guarded block a loop, which is not
// if-converted.
// One k-pair (two k-steps = a 2x2x2 box of mesh points) of an off-diagonal tile: row fragments ra x
// column fragments ca (4-bit masks, OR over the two k-steps).  The code is selected by the column
// pattern (a jump on a warp-uniform value), the rows are guarded one by one; .x / .y of an operand are
// its values for the first / second k-step.
#define KROW(i, body)                                  \
    if (ra & (1u << i)) {                              \
        do { body } while (never);                     \
    }
#define KX(i, j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a##i.x, b##j.x);
#define KY(i, j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a##i.y, b##j.y);
#define K1(i, p) KX(i, p) KY(i, p)
#define K2(i, p, q) KX(i, p) KX(i, q) KY(i, p) KY(i, q)
#define K3(i, p, q, r) KX(i, p) KX(i, q) KX(i, r) KY(i, p) KY(i, q) KY(i, r)
#define K4(i) KX(i, 0) KX(i, 1) KX(i, 2) KX(i, 3) KY(i, 0) KY(i, 1) KY(i, 2) KY(i, 3)
#define KCASE1(c, p) case c: KROW(0, K1(0, p)) KROW(1, K1(1, p)) KROW(2, K1(2, p)) KROW(3, K1(3, p)) break;
#define KCASE2(c, p, q) case c: KROW(0, K2(0, p, q)) KROW(1, K2(1, p, q)) KROW(2, K2(2, p, q)) KROW(3, K2(3, p, q)) break;
#define KCASE3(c, p, q, r) \
    case c: KROW(0, K3(0, p, q, r)) KROW(1, K3(1, p, q, r)) KROW(2, K3(2, p, q, r)) KROW(3, K3(3, p, q, r)) break;
__device__ __forceinline__ void kpair_rect(double (&acc)[4][4][2], uint32_t ra, uint32_t ca, double2 a0, double2 a1, double2 a2,
                                           double2 a3, double2 b0, double2 b1, double2 b2, double2 b3, int never) {
    switch (ca) {
        KCASE1(1, 0)
        KCASE1(2, 1)
        KCASE2(3, 0, 1)
        KCASE1(4, 2)
        KCASE2(5, 0, 2)
        KCASE2(6, 1, 2)
        KCASE3(7, 0, 1, 2)
        KCASE1(8, 3)
        KCASE2(9, 0, 3)
        KCASE2(10, 1, 3)
        KCASE3(11, 0, 1, 3)
        KCASE2(12, 2, 3)
        KCASE3(13, 0, 2, 3)
        KCASE3(14, 1, 2, 3)
        case 15: KROW(0, K4(0)) KROW(1, K4(1)) KROW(2, K4(2)) KROW(3, K4(3)) break;
        default: break;
    }
}
// The same with all four row fragments active (the usual case: rows come from the denser groups):
// straight-line code per column pattern, no row guards.
// (all first-k-step DMMAs, then all second-k-step ones: no accumulator is reused within 28 cycles)
#define KALL1(c, p) case c: KX(0, p) KX(1, p) KX(2, p) KX(3, p) KY(0, p) KY(1, p) KY(2, p) KY(3, p) break;
#define KALL2(c, p, q) \
    case c: KX(0, p) KX(0, q) KX(1, p) KX(1, q) KX(2, p) KX(2, q) KX(3, p) KX(3, q) \
            KY(0, p) KY(0, q) KY(1, p) KY(1, q) KY(2, p) KY(2, q) KY(3, p) KY(3, q) break;
#define KALL3(c, p, q, r) \
    case c: KX(0, p) KX(0, q) KX(0, r) KX(1, p) KX(1, q) KX(1, r) KX(2, p) KX(2, q) KX(2, r) KX(3, p) KX(3, q) KX(3, r) \
            KY(0, p) KY(0, q) KY(0, r) KY(1, p) KY(1, q) KY(1, r) KY(2, p) KY(2, q) KY(2, r) KY(3, p) KY(3, q) KY(3, r) break;
__device__ __forceinline__ void kpair_rect_allrows(double (&acc)[4][4][2], uint32_t ca, double2 a0, double2 a1, double2 a2,
                                                   double2 a3, double2 b0, double2 b1, double2 b2, double2 b3) {
    switch (ca) {
        KALL1(1, 0)
        KALL1(2, 1)
        KALL2(3, 0, 1)
        KALL1(4, 2)
        KALL2(5, 0, 2)
        KALL2(6, 1, 2)
        KALL3(7, 0, 1, 2)
        KALL1(8, 3)
        KALL2(9, 0, 3)
        KALL2(10, 1, 3)
        KALL3(11, 0, 1, 3)
        KALL2(12, 2, 3)
        KALL3(13, 0, 2, 3)
        KALL3(14, 1, 2, 3)
        default: break;
    }
}
#undef KALL1
#undef KALL2
#undef KALL3
// One k-pair of a diagonal tile (row group == column group): fragment pairs i <= j with both active.
#define KX_IF(cond, i, j) \
    if (cond) {           \
        do { KX(i, j) } while (never); \
    }
#define KY_IF(cond, i, j) \
    if (cond) {           \
        do { KY(i, j) } while (never); \
    }
__device__ __forceinline__ void kpair_diag(double (&acc)[4][4][2], uint32_t ra, double2 a0, double2 a1, double2 a2, double2 a3,
                                           double2 b0, double2 b1, double2 b2, double2 b3, int never) {
    if (ra == 0xFu) {   // all ten fragment pairs
        KX(0, 0) KX(0, 1) KX(0, 2) KX(0, 3) KX(1, 1) KX(1, 2) KX(1, 3) KX(2, 2) KX(2, 3) KX(3, 3)
        KY(0, 0) KY(0, 1) KY(0, 2) KY(0, 3) KY(1, 1) KY(1, 2) KY(1, 3) KY(2, 2) KY(2, 3) KY(3, 3)
        return;
    }
    // first k-step of every active pair, then the second: no accumulator is reused back to back
    KROW(0, KX(0, 0) KX_IF(ra & 2u, 0, 1) KX_IF(ra & 4u, 0, 2) KX_IF(ra & 8u, 0, 3))
    KROW(1, KX(1, 1) KX_IF(ra & 4u, 1, 2) KX_IF(ra & 8u, 1, 3))
    KROW(2, KX(2, 2) KX_IF(ra & 8u, 2, 3))
    KROW(3, KX(3, 3))
    KROW(0, KY(0, 0) KY_IF(ra & 2u, 0, 1) KY_IF(ra & 4u, 0, 2) KY_IF(ra & 8u, 0, 3))
    KROW(1, KY(1, 1) KY_IF(ra & 4u, 1, 2) KY_IF(ra & 8u, 1, 3))
    KROW(2, KY(2, 2) KY_IF(ra & 8u, 2, 3))
    KROW(3, KY(3, 3))
}
#undef KROW
#undef KX
#undef KY
#undef K1
#undef K2
#undef K3
#undef K4
#undef KCASE1
#undef KCASE2
#undef KCASE3
#undef KX_IF
#undef KY_IF

// ---- mbarrier / bulk-copy helpers (shared::cta addresses) --------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

__device__ __forceinline__ double rsqrt_seed(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

// psi = phi sqrt(|V dV|) of one entry on the 32 points of a slice (lane = point), Eq. 1, stored
// to the region's scratch in fragment order: element (row R, point p of stage s) sits at
//   chunk(R >> 5, s) + (((R >> 3 & 3) * 2 + kp) * 32 + (R & 7) * 4 + fk) * 2 + kk,
// p = (2 kp + kk) * 4 + fk, so that one LDS.128 per lane feeds two k-steps of a DMMA operand.
__device__ __forceinline__ void eval_task(const DevicePlan& P, const double* __restrict__ tab, const Entry* __restrict__ en,
                                          int slice, int lane, const double* __restrict__ s_off,
                                          const double* __restrict__ s_sqrtw, double* __restrict__ psi_region) {
    const int sp = (en->Rpack >> 24) & 0x7F;
    const int32_t* meta = P.sp_meta + 12 * sp;
    const int tab_off = __ldg(meta + 0), ntab = __ldg(meta + 1), nradp = __ldg(meta + 2);
    const double rc2 = __ldg(P.sp_real + 2 * sp), inv_dr = __ldg(P.sp_real + 2 * sp + 1);
    const int p = slice * kSlicePts + lane;
    const double dx = en->rel[0] + s_off[p];
    const double dy = en->rel[1] + s_off[kMaxRegionPoints + p];
    const double dz = en->rel[2] + s_off[2 * kMaxRegionPoints + p];
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const bool inside = r2 < rc2;
    double rinv = 0.0, lnz = 0.0;   // lnz: 1 if the l>0 components survive (r >= 1e-12)
    if (r2 >= 1e-24) {
        const double y0 = rsqrt_seed(r2);              // relative error ~2^-22
        const double e = fma(-(r2 * y0), y0, 1.0);     // 1 - r2 y0^2
        rinv = fma(e * y0, fma(0.375, e, 0.5), y0);    // y0 (1 + e/2 + 3 e^2/8): cubic convergence
        lnz = 1.0;
    }
    const double r = r2 * rinv;
    const double x = dx * rinv, y = dy * rinv, z = dz * rinv;
    const double s = r * inv_dr;
    int k = __double2int_rd(s);
    const double t = s - (double)k;
    k = inside ? min(k, ntab) : ntab;                  // outside: the four zero nodes after the table
    const double t1 = 1.0 - t, t2 = 2.0 - t, t3 = 3.0 - t;
    const double a23 = t2 * t3, b01 = t * t1;
    const double sq = s_sqrtw[p];
    const double L0 = (t1 * a23) * (sq * (1.0 / 6.0));
    const double L1 = (t * a23) * (sq * 0.5);
    const double L2 = (b01 * t3) * (sq * -0.5);
    const double L3 = (b01 * t2) * (sq * (1.0 / 6.0));
    const double* Tk = tab + tab_off + k * nradp;
    // store addressing
    const int row0 = en->row0;
    double* out = psi_region + ((lane / kStagePts) * kChunkDoubles + (((lane % kStagePts) >> 3) * 64) + (lane & 3) * 2 + ((lane >> 2) & 1));
    const int gstride = P.nstage * kChunkDoubles;
    int R = row0;
    auto put = [&](double v) {
        out[(R >> 5) * gstride + ((R >> 3) & 3) * (kStagePairs * 64) + (R & 7) * 8] = v;
        R++;
    };
    auto emit = [&](int l, double fv) {
        if (l == 0) {
            put(fv);
        } else if (l == 1) {
            put(fv * y);
            put(fv * z);
            put(fv * x);
        } else {
            // table carries 1/2 sqrt(15/pi); ratios: 1/4 sqrt(5/pi) / that = 1/(2 sqrt 3), 1/4 sqrt(15/pi) / that = 1/2
            put(fv * (x * y));
            put(fv * (y * z));
            put(fv * (fma(3.0 * z, z, -lnz) * 0.28867513459481288));
            put(fv * (x * z));
            put(fv * (fma(x, x, -(y * y)) * 0.5));
        }
    };
    for (int f = 0; f < nradp; f += 2) {
        const double2 T0 = *reinterpret_cast<const double2*>(Tk + f);
        const double2 T1 = *reinterpret_cast<const double2*>(Tk + nradp + f);
        const double2 T2 = *reinterpret_cast<const double2*>(Tk + 2 * nradp + f);
        const double2 T3 = *reinterpret_cast<const double2*>(Tk + 3 * nradp + f);
        const int l0 = __ldg(meta + 4 + f);
        const int l1 = (f + 1 < 8) ? __ldg(meta + 4 + f + 1) : -1;
        emit(l0, fma(T0.x, L0, fma(T1.x, L1, fma(T2.x, L2, T3.x * L3))));
        if (l1 >= 0) emit(l1, fma(T0.y, L0, fma(T1.y, L1, fma(T2.y, L2, T3.y * L3))));
    }
}

}  // namespace
// ---- kernel 1: psi = phi sqrt(|V dV|) of every region, evaluated once ---------------------------
// One CTA per region (with work): stage sqrt(|V dV|) of the region's points and their sign bits, then
// the warps walk the region's (atom image, 32-point slice) tasks.  Plenty of warps per SM (4 CTAs of 8
// warps) hide the table and entry latencies; the output is 8.5 GB at si512_dzp, so the kernel runs at
// the HBM write rate.
constexpr int kEvalThreads = 256;

struct EvalSmem {
    uint32_t off, xyz, sqrtw, tab, total;
};
GINT_HD inline EvalSmem eval_smem(size_t table_bytes) {
    EvalSmem L;
    uint32_t o = 0;
    L.off = o;   o += 3 * kMaxRegionPoints * 8;
    L.xyz = o;   o += kMaxRegionPoints * 4;
    L.sqrtw = o; o += kMaxRegionPoints * 8;
    L.tab = o;   o += smem_align(table_bytes);
    L.total = o;
    return L;
}

template <bool TAB_SMEM>
__global__ void __launch_bounds__(kEvalThreads, 3)
gint_psi_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ V) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const EvalSmem L = eval_smem(TAB_SMEM ? (size_t)P.tab_doubles * sizeof(double) : 0);
    double* s_off = reinterpret_cast<double*>(smem_raw + L.off);
    uchar4* s_xyz = reinterpret_cast<uchar4*>(smem_raw + L.xyz);
    double* s_sqrtw = reinterpret_cast<double*>(smem_raw + L.sqrtw);
    double* s_tab = reinterpret_cast<double*>(smem_raw + L.tab);
    if (TAB_SMEM) {
        for (int i = tid; i < P.tab_doubles; i += kEvalThreads) s_tab[i] = __ldg(P.tab + i);
    }
    const double* tab = TAB_SMEM ? s_tab : P.tab;
    const int npt = P.nslice * kSlicePts;
    for (int p = tid; p < npt; p += kEvalThreads) {
        const uchar4 c = reinterpret_cast<const uchar4*>(P.slot_xyz)[p];
        for (int k = 0; k < 3; k++)
            s_off[k * kMaxRegionPoints + p] = c.x * P.estep[k] + c.y * P.estep[3 + k] + c.z * P.estep[6 + k];
        s_xyz[p] = c;
    }
    for (int r = blockIdx.x; r < P.nwork_regions; r += gridDim.x) {
        __syncthreads();   // previous region's sqrtw no longer read (first pass: tables and offsets staged)
        const int reg_index = __ldg(P.work_regions + r);
        const Region* reg = P.regions + reg_index;
        const int ox = __ldg(&reg->origin[0]), oy = __ldg(&reg->origin[1]), oz = __ldg(&reg->origin[2]);
        const int item0 = __ldg(&reg->item0), nitem = __ldg(&reg->nitem);
        for (int p = tid; p < npt; p += kEvalThreads) {   // npt is a multiple of 32: whole warps
            const uchar4 c = s_xyz[p];
            const int g1 = ox + c.x, g2 = oy + c.y, g3 = oz + c.z;
            double wv = 0.0;
            if (c.w && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2])   // V == nullptr: plain phi (gint_rho)
                wv = V ? __ldg(V + ((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3) * P.dV : 1.0;
            s_sqrtw[p] = sqrt(fabs(wv));
            const unsigned int neg = __ballot_sync(0xffffffffu, wv < 0.0);
            if (lane == 0)   // every work item of the region carries the sign bits in its descriptor
                for (int q = 0; q < nitem; q++) P.descs[item0 + q].sign[p >> 5] = neg;
        }
        __syncthreads();
        const int ntask = __ldg(&reg->ntask);
        const uint32_t* tasks = P.etasks + __ldg(&reg->task_off);
        const Entry* entries = P.entries + __ldg(&reg->entry0);
        double* psi_region = P.psi + (size_t)__ldg(&reg->psi_chunk0) * kChunkDoubles;
        for (int t = warp; t < ntask; t += kEvalThreads / 32) {
            const uint32_t tk = __ldg(tasks + t);
            const Entry* en = entries + (tk & 0xFFFFu);
            const int s0 = (int)(tk >> 16) * 8;
            // activity of the run's 8 slices: byte s of the 64 k-step bits starting at slice s0
            const uint2 km = *reinterpret_cast<const uint2*>(&en->kmask[s0 >> 2]);
            for (int q = 0; q < 8 && s0 + q < P.nslice; q++) {
                if ((((q < 4 ? km.x : km.y) >> (8 * (q & 3))) & 0xFFu) == 0u) continue;
                const int slice = s0 + q;
                eval_task(P, tab, en, slice, lane, s_off, s_sqrtw,
                          psi_region + (size_t)(slice * (kSlicePts / kStagePts)) * kChunkDoubles);
            }
        }
    }
}

// ---- kernel 2: contraction -------------------------------------------------------------------
struct ContractSmem {
    uint32_t bar, desc, ring, total;
};
GINT_HD inline ContractSmem contract_smem(int nring) {
    ContractSmem L;
    uint32_t o = 0;
    L.bar = o;   o += 256;   // mbarriers: full[8], empty[8], desc_full[4], desc_empty[4]
    L.desc = o;  o += smem_align((size_t)kDescSlots * sizeof(ItemDesc));
    L.ring = o;  o += (uint32_t)nring * kStageBytes;
    L.total = o;
    return L;
}

// ---- gint_rho on the tensor pipe (MODE 1 of the contraction kernel) --------------------------------
//   rho(p) = sum over tiles (ga <= gb) of  Phi_ga(p)^T E Phi_gb(p),   E = D[ga][gb] + D[gb][ga]^T  (ga < gb),
//                                                                      E = D[ga][ga]               (ga = gb),
// D[.][.] being the region's density matrix gathered from the blocks (entry a, entry b) -> (I_a, I_b, R_b - R_a)
// (Eq. 44; no symmetry of D is assumed).  The warp holds E as 4 x 8 A fragments
// (rows 8 i + lane/4, columns 4 kc + lane%4) in registers for the whole item.  Per k-pair (8 mesh points) it
// forms T = E Phi_gb as 4 accumulator fragments (rows x 8 points) with the B operand read from the stage
// (rows of gb are the K dimension, the 8 points the N dimension: conflict-free 8-byte loads in the fragment
// layout), multiplies by Phi_ga in the accumulator layout, reduces over the rows by shuffles and adds the 8 point
// values into rho with red.global.add.f64.
#define RHO_GUARD(cond, body)          \
    if (cond) {                        \
        do { body } while (never);     \
    }
#define RHO_ROW(i)                                                           \
    RHO_GUARD(ra & (1u << i), {                                              \
        dmma8x8x4(C[i][0], C[i][1], A[i][2 * j], b0);                        \
        dmma8x8x4(C[i][0], C[i][1], A[i][2 * j + 1], b1);                    \
    })
__device__ __forceinline__ void rho_consumer(const DevicePlan& P, const double* __restrict__ D, double* __restrict__ rho,
                                             uint64_t* s_full, uint64_t* s_empty, uint64_t* s_dfull, uint64_t* s_dempty,
                                             const ItemDesc* s_desc, const unsigned char* s_ring, int nring, int never,
                                             int lane, int cidx) {
    if (kStagePts != 32) return;   // the 16-point-stage build variant (GINT_CTAS_PER_SM=2) uses the FMA kernel of gint_rho.cu
    const int frow = lane >> 2, fk = lane & 3;
    uint32_t cs = 0, cph = 0;
    for (int it = 0;; it++) {
        const int ds = it % kDescSlots;
        mbar_wait(smem_u32(s_dfull + ds), ((uint32_t)it / kDescSlots) & 1u);
        const ItemDesc* cur = &s_desc[ds];
        if (!cur->valid) break;
        const int sa = cur->item.tiles[cidx][0], sb = cur->item.tiles[cidx][1];
        const bool has_tile = sa != 0xFF;
        const bool diag = sa == sb;
        // ---- gather the tile of E into A fragments ----
        double A[4][8];
        if (has_tile) {
            const uint32_t* pdir = P.pair_direct + cur->item.reg.pair_off;
            const int m = cur->item.reg.nentry;
            uint32_t ci[8];
#pragma unroll
            for (int kc = 0; kc < 8; kc++) ci[kc] = cur->rinfo[sb][4 * kc + fk];
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const uint32_t ri = cur->rinfo[sa][8 * i + frow];
                const int ea = ri & 0xFFF, mu = (ri >> 12) & 0xFF, nI = ri >> 20;
                // all pair-table look-ups of the row first, then all block elements (independent loads in flight)
                uint32_t o1[8], o2[8];
#pragma unroll
                for (int kc = 0; kc < 8; kc++) {
                    const bool ok = ri != kNoBlock && ci[kc] != kNoBlock;
                    const int eb = ci[kc] & 0xFFF;
                    o1[kc] = ok ? __ldg(pdir + ea * m + eb) : kNoBlock;
                    o2[kc] = (ok && !diag) ? __ldg(pdir + eb * m + ea) : kNoBlock;
                }
#pragma unroll
                for (int kc = 0; kc < 8; kc++) {
                    const int nu = (ci[kc] >> 12) & 0xFF, nJ = ci[kc] >> 20;
                    const double e1 = o1[kc] != kNoBlock ? __ldg(D + o1[kc] + mu * nJ + nu) : 0.0;
                    const double e2 = o2[kc] != kNoBlock ? __ldg(D + o2[kc] + nu * nI + mu) : 0.0;
                    A[i][kc] = e1 + e2;
                }
            }
        }
        const int ox = cur->item.reg.origin[0], oy = cur->item.reg.origin[1], oz = cur->item.reg.origin[2];
        uint32_t todo = cur->item.stage_mask;
        while (todo) {
            const int s = __ffs(todo) - 1;
            todo &= todo - 1;
            uint32_t ma = 0, mb = 0;
            if (has_tile) {
                const uint64_t ma8 = *reinterpret_cast<const uint64_t*>(&cur->gmask[sa][s * 8]);
                const uint64_t mb8 = *reinterpret_cast<const uint64_t*>(&cur->gmask[sb][s * 8]);
                const uint64_t qa = (ma8 | (ma8 >> 8)) & 0x000F000F000F000Full, qb = (mb8 | (mb8 >> 8)) & 0x000F000F000F000Full;
                ma = (uint32_t)qa | (uint32_t)(qa >> 28);
                mb = (uint32_t)qb | (uint32_t)(qb >> 28);
            }
            mbar_wait(smem_u32(s_full + cs), cph);
            if (has_tile) {
                const unsigned char* stage = s_ring + (size_t)cs * kStageBytes;
                const double* chA = reinterpret_cast<const double*>(stage + sa * kChunkBytes);
                const double* chB = reinterpret_cast<const double*>(stage + sb * kChunkBytes);
#pragma unroll 1
                for (int kp = 0; kp < kStagePairs; kp++) {
                    const uint32_t ra = (ma >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
                    const uint32_t ca = (mb >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
                    if (ra == 0u || ca == 0u) continue;
                    double C[4][2];
#pragma unroll
                    for (int i = 0; i < 4; i++) C[i][0] = C[i][1] = 0.0;
                    // B operand of k-step kc = 2 j + h2: Phi_gb[row 8 j + 4 h2 + lane%4][point lane/4 of the k-pair]
                    const double* bsrc = chB + ((kp * 32 + fk * 4 + (frow & 3)) * 2 + (frow >> 2));
                    if ((ra & ca) == 0xFu) {
#pragma unroll
                        for (int kc = 0; kc < 8; kc++) {
                            const double b = bsrc[((kc >> 1) * kStagePairs * 32 + (kc & 1) * 16) * 2];
#pragma unroll
                            for (int i = 0; i < 4; i++) dmma8x8x4(C[i][0], C[i][1], A[i][kc], b);
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 4; j++) {
                            RHO_GUARD(ca & (1u << j), {
                                const double b0 = bsrc[(j * kStagePairs * 32) * 2];
                                const double b1 = bsrc[(j * kStagePairs * 32 + 16) * 2];
                                RHO_ROW(0) RHO_ROW(1) RHO_ROW(2) RHO_ROW(3)
                            })
                        }
                    }
                    // C[i][h] = T[row 8 i + lane/4][point 2 (lane%4) + h]: times Phi_ga there, summed over the rows
                    double p0 = 0.0, p1 = 0.0;
                    const double* asrc = chA + ((kp * 32 + frow * 4 + ((2 * fk) & 3)) * 2 + (fk >> 1));
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        if ((ra >> i) & 1u) {
                            p0 = fma(asrc[(i * kStagePairs * 32) * 2], C[i][0], p0);
                            p1 = fma(asrc[(i * kStagePairs * 32) * 2 + 2], C[i][1], p1);
                        }
                    }
                    // sum over the 8 row lanes (lane/4): lanes with even lane/4 end up with the first point's total,
                    // odd ones with the second's (one exchange), then two plain butterfly steps
                    const bool odd = (frow & 1) != 0;
                    double keep = odd ? p1 : p0;
                    keep += __shfl_xor_sync(0xffffffffu, odd ? p0 : p1, 4);
                    keep += __shfl_xor_sync(0xffffffffu, keep, 8);
                    keep += __shfl_xor_sync(0xffffffffu, keep, 16);
                    if (frow < 2) {   // lanes 0..7: point 8 kp + 2 fk + lane/4 of the stage
                        const uchar4 c = reinterpret_cast<const uchar4*>(P.slot_xyz)[s * kStagePts + kp * 8 + 2 * fk + frow];
                        const int g1 = ox + c.x, g2 = oy + c.y, g3 = oz + c.z;
                        if (c.w && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2] && keep != 0.0)
                            atomicAdd(rho + ((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3, keep);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(s_empty + cs));
            if (++cs == (uint32_t)nring) { cs = 0; cph ^= 1u; }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(s_dempty + ds));
    }
}
#undef RHO_ROW
#undef RHO_GUARD

// MODE 0: gint_vlocal (H += psi diag(sign V) psi^T, Eq. 45).  MODE 1: gint_rho (Eq. 44): the same items, stages and
// producer; a consumer warp keeps its 32x32 tile of the region's density matrix in registers as the A operand,
// forms T = E Phi_b on the tensor pipe per 8 points and dots it with Phi_a (see the consumer code below).
template <int MODE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm)
gint_contract_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ Din, double* __restrict__ H) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const ContractSmem L = contract_smem(P.nring);
    uint64_t* s_full = reinterpret_cast<uint64_t*>(smem_raw + L.bar);         // [8] stage filled (tx bytes)
    uint64_t* s_empty = s_full + 8;                                           // [8] stage released by the 15 consumer warps
    uint64_t* s_dfull = s_full + 16;                                          // [4] descriptor staged
    uint64_t* s_dempty = s_full + 20;                                         // [4] descriptor released
    ItemDesc* s_desc = reinterpret_cast<ItemDesc*>(smem_raw + L.desc);        // [3]
    unsigned char* s_ring = smem_raw + L.ring;                                // [nring][slot][4 KB]
    const int nring = P.nring;
    const int never = P.never;   // always 0; see DMMA_IF

    if (tid == 0) {
        for (int i = 0; i < nring; i++) {
            mbar_init(smem_u32(s_full + i), 1);
            mbar_init(smem_u32(s_empty + i), kConsumerWarps);
        }
        for (int i = 0; i < kDescSlots; i++) {
            mbar_init(smem_u32(s_dfull + i), 1);
            mbar_init(smem_u32(s_dempty + i), kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // The two CTAs of an SM put their producer warp on different sub-partitions (warp w runs on sub-partition
    // w % 4), so that the SM's 14 consumer warps spread 3/4/4/3: the first CTA to arrive uses warp 7, the second warp 4.
    __shared__ int s_parity;
    if (tid == 0) {
        unsigned int smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        s_parity = (int)(atomicAdd(P.counter + 1 + (smid & 255u), 1u) & 1u);
    }
    fence_proxy_async();
    __syncthreads();
    const int parity = kCtasPerSm == 2 ? s_parity : 0;
    const int producer_warp = parity ? 4 : kConsumerWarps;
    // consumer index (which tile of the item): the plan fills tiles[v + 4 r] for virtual sub-partition v (v = 3 holds
    // one tile fewer); parity 1 swaps sub-partitions 0 and 3
    const int cidx = parity == 0 ? warp : (warp == 0 ? 3 : (warp == 3 ? 0 : (warp == 7 ? 4 : warp)));
    TIMER_DECL

    if (warp == producer_warp) {
        // ================= producer warp =================
        // Descriptor i+1 is fetched (one bulk copy straight into the slot, completion on its own
        // mbarrier) while the stages of item i are being streamed; the queue index is taken one more
        // item ahead so that the atomic's latency is off the critical path as well.
        uint32_t rs = 0, rph = 0;   // ring slot and phase of the next stage to fill
        auto fetch_desc = [&](int i, unsigned int it) {   // lane 0: item index it -> descriptor slot i % 3
            const int ds = i % kDescSlots;
            mbar_wait(smem_u32(s_dempty + ds), (((uint32_t)i / kDescSlots) & 1u) ^ 1u);
            const uint32_t bar = smem_u32(s_dfull + ds);
            if (it < (unsigned int)P.nitems) {
                mbar_arrive_expect_tx(bar, (uint32_t)sizeof(ItemDesc));
                bulk_g2s(smem_u32(&s_desc[ds]), P.descs + it, (uint32_t)sizeof(ItemDesc), bar);
            } else {
                s_desc[ds].valid = 0;
                mbar_arrive(bar);
            }
        };
        unsigned int it_next = 0, it_after = 0;
        if (lane == 0) {
            it_next = atomicAdd(P.counter, 1u);
            fetch_desc(0, it_next);
            it_next = atomicAdd(P.counter, 1u);
        }
        for (int i = 0;; i++) {
            const ItemDesc* cur = &s_desc[i % kDescSlots];
            if (lane == 0) {
                it_after = atomicAdd(P.counter, 1u);                    // index of item i+2, needed one item from now
                mbar_wait(smem_u32(s_dfull + i % kDescSlots), ((uint32_t)i / kDescSlots) & 1u);
                if (cur->valid) fetch_desc(i + 1, it_next);             // in flight while this item streams
                it_next = it_after;
            }
            __syncwarp();
            if (!cur->valid) break;
            const int nslot = cur->item.nslot;
            const unsigned char* psi_bytes = reinterpret_cast<const unsigned char*>(P.psi) +
                                             (size_t)cur->item.reg.psi_chunk0 * kChunkBytes;
            // lane q copies the chunks of slot q; lane 0 also owns the barriers
            const unsigned char* src_lane = psi_bytes + (size_t)(lane < nslot ? cur->item.slot_group[lane] : 0) * P.nstage * kChunkBytes;
            uint32_t todo = cur->item.stage_mask;
            while (todo) {
                const int s = __ffs(todo) - 1;
                todo &= todo - 1;
                const uint32_t act = cur->act[s];
                const uint32_t bar = smem_u32(s_full + rs);
                if (lane == 0) {
                    TIMER_START
                    mbar_wait(smem_u32(s_empty + rs), rph ^ 1u);
                    TIMER_ADD(1)
                    if (act) mbar_arrive_expect_tx(bar, (uint32_t)__popc(act) * kChunkBytes);
                    else mbar_arrive(bar);
                }
                __syncwarp();
                if ((act >> lane) & 1u)
                    bulk_g2s(smem_u32(s_ring + (size_t)rs * kStageBytes) + lane * kChunkBytes,
                             src_lane + (size_t)s * kChunkBytes, kChunkBytes, bar);
                if (++rs == (uint32_t)nring) { rs = 0; rph ^= 1u; }
            }
            TIMER_COUNT(6)
        }
    } else {
        // ================= consumer warps =================
        if constexpr (MODE == 0) {

        const int frow = lane >> 2, fk = lane & 3;
        uint32_t cs = 0, cph = 0;   // ring slot and phase of the next stage to consume
        for (int it = 0;; it++) {
            const int ds = it % kDescSlots;
            TIMER_START
            mbar_wait(smem_u32(s_dfull + ds), ((uint32_t)it / kDescSlots) & 1u);
            TIMER_ADD(0)
            const ItemDesc* cur = &s_desc[ds];
            if (!cur->valid) break;
            const int sa = cur->item.tiles[cidx][0], sb = cur->item.tiles[cidx][1];
            const bool has_tile = sa != 0xFF;
            const bool diag = sa == sb;
            double acc[4][4][2];
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int j = 0; j < 4; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

            uint32_t todo = cur->item.stage_mask;
#ifdef GINT_TIMING
            int nvis = 0;
#endif
            while (todo) {
                const int s = __ffs(todo) - 1;
                todo &= todo - 1;
                TIMER_START
                mbar_wait(smem_u32(s_full + cs), cph);
                TIMER_ADD(3)
#ifdef GINT_TIMING
                if (nvis == 0) { TIMER_ADD(1) } else if (nvis < 4) { TIMER_ADD(2) }
                nvis++;
#endif
                TIMER_START
#ifdef GINT_TIMING
                if (has_tile && !(P.debug & 1)) {
#else
                if (has_tile) {
#endif
                    // activity nibbles of the stage's k-steps, one byte each; k-pair kp = bytes 2 kp, 2 kp + 1, OR-ed and
                    // packed: pair 0 -> bits 0-3, pair 1 -> bits 16-19, pair 2 -> bits 4-7, pair 3 -> bits 20-23
                    uint32_t ma, mb;
                    if (kStageKsteps == 8) {
                        const uint64_t ma8 = *reinterpret_cast<const uint64_t*>(&cur->gmask[sa][s * 8]);
                        const uint64_t mb8 = *reinterpret_cast<const uint64_t*>(&cur->gmask[sb][s * 8]);
                        const uint64_t qa = (ma8 | (ma8 >> 8)) & 0x000F000F000F000Full, qb = (mb8 | (mb8 >> 8)) & 0x000F000F000F000Full;
                        ma = (uint32_t)qa | (uint32_t)(qa >> 28);
                        mb = (uint32_t)qb | (uint32_t)(qb >> 28);
                    } else {
                        const uint32_t ma4 = *reinterpret_cast<const uint32_t*>(&cur->gmask[sa][s * 4]);
                        const uint32_t mb4 = *reinterpret_cast<const uint32_t*>(&cur->gmask[sb][s * 4]);
                        ma = (ma4 | (ma4 >> 8)) & 0x000F000Fu;
                        mb = (mb4 | (mb4 >> 8)) & 0x000F000Fu;
                    }
                    const unsigned char* stage = s_ring + (size_t)cs * kStageBytes;
                    const double2* pa = reinterpret_cast<const double2*>(stage + sa * kChunkBytes) + lane;
                    const double2* pb = reinterpret_cast<const double2*>(stage + sb * kChunkBytes) + lane;
                    // sign bits of V dV at this lane's four points (k-step ks: bit 4 ks + fk of the stage's 16)
                    const uint32_t sg = (kStagePts == 32 ? cur->sign[s] : (cur->sign[s >> 1] >> ((s & 1) * 16))) >> fk;
#pragma unroll 1
                    for (int kp = 0; kp < kStagePairs; kp++) {
#ifdef GINT_TIMING
                        const uint32_t ra = (P.debug & 8) ? 0xFu : (ma >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
                        const uint32_t ca = (P.debug & 8) ? 0xFu : (mb >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
#else
                        const uint32_t ra = (ma >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
                        const uint32_t ca = (mb >> ((kp & 1) * 16 + (kp >> 1) * 4)) & 0xFu;
#endif
                        if (ra == 0u || ca == 0u) continue;
                        // operands of both k-steps; fragments outside the masks may hold stale data and are not used
                        const double2 a0 = pa[(0 * kStagePairs + kp) * 32], a1 = pa[(1 * kStagePairs + kp) * 32], a2 = pa[(2 * kStagePairs + kp) * 32],
                                      a3 = pa[(3 * kStagePairs + kp) * 32];
                        double2 b0 = pb[(0 * kStagePairs + kp) * 32], b1 = pb[(1 * kStagePairs + kp) * 32], b2 = pb[(2 * kStagePairs + kp) * 32],
                                b3 = pb[(3 * kStagePairs + kp) * 32];
                        const uint32_t x0 = ((sg >> (8 * kp)) & 1u) << 31, x1 = ((sg >> (8 * kp + 4)) & 1u) << 31;
#define SIGN_FLIP(v)                                                                 \
    v.x = __hiloint2double(__double2hiint(v.x) ^ x0, __double2loint(v.x)); \
    v.y = __hiloint2double(__double2hiint(v.y) ^ x1, __double2loint(v.y));
                        SIGN_FLIP(b0) SIGN_FLIP(b1) SIGN_FLIP(b2) SIGN_FLIP(b3)
#undef SIGN_FLIP
                        if (!diag) {
                            if ((ra & ca) == 0xFu) {
#define FX(i, j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a##i.x, b##j.x);
#define FY(i, j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a##i.y, b##j.y);
                                FX(0, 0) FX(0, 1) FX(0, 2) FX(0, 3) FX(1, 0) FX(1, 1) FX(1, 2) FX(1, 3)
                                FX(2, 0) FX(2, 1) FX(2, 2) FX(2, 3) FX(3, 0) FX(3, 1) FX(3, 2) FX(3, 3)
                                FY(0, 0) FY(0, 1) FY(0, 2) FY(0, 3) FY(1, 0) FY(1, 1) FY(1, 2) FY(1, 3)
                                FY(2, 0) FY(2, 1) FY(2, 2) FY(2, 3) FY(3, 0) FY(3, 1) FY(3, 2) FY(3, 3)
#undef FX
#undef FY
                            } else if (ra == 0xFu) {
                                kpair_rect_allrows(acc, ca, a0, a1, a2, a3, b0, b1, b2, b3);
                            } else {
                                kpair_rect(acc, ra, ca, a0, a1, a2, a3, b0, b1, b2, b3, never);
                            }
                        } else {
                            kpair_diag(acc, ra, a0, a1, a2, a3, b0, b1, b2, b3, never);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(s_empty + cs));
                if (++cs == (uint32_t)nring) { cs = 0; cph ^= 1u; }
                TIMER_ADD(4)
            }
            TIMER_START

        // ---------------- flush: add the tile into the canonical H blocks ---------------------------
#ifdef GINT_TIMING
        if (has_tile && !(P.debug & 4)) {
#else
        if (has_tile) {
#endif
            const int ga = cur->item.slot_group[sa], gb = cur->item.slot_group[sb];
            const uint32_t* pair = P.pair + cur->item.reg.pair_off;
            const int m = cur->item.reg.nentry;
            // this lane's 8 columns: j = 0..3, h = 0..1 -> column 8 j + 2 fk + h of the column group
            uint32_t ci[4][2];
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const uint2 c2 = *reinterpret_cast<const uint2*>(&cur->rinfo[sb][8 * j + 2 * fk]);
                ci[j][0] = c2.x;
                ci[j][1] = c2.y;
            }
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const int row = ga * kGroupRows + 8 * i + frow;
                const uint32_t ri = cur->rinfo[sa][8 * i + frow];
                const int ea = ri & 0xFFF, mu = (ri >> 12) & 0xFF, nI = ri >> 20;
                // all pair-table look-ups of the row first (independent loads), then the reductions
                uint32_t pr[4][2];
#pragma unroll
                for (int j = 0; j < 4; j++)
#pragma unroll
                    for (int h = 0; h < 2; h++) {
                        const int col = gb * kGroupRows + 8 * j + 2 * fk + h;
                        const bool ok = ri != kNoBlock && ci[j][h] != kNoBlock && row <= col && !(diag && i > j) &&
                                        acc[i][j][h] != 0.0;
                        pr[j][h] = ok ? __ldg(pair + ea * m + (int)(ci[j][h] & 0xFFF)) : kNoBlock;
                    }
#pragma unroll
                for (int j = 0; j < 4; j++)
#pragma unroll
                    for (int h = 0; h < 2; h++) {
                        const uint32_t p2 = pr[j][h];
                        if (p2 == kNoBlock) continue;
                        const int nu = (ci[j][h] >> 12) & 0xFF, nJ = ci[j][h] >> 20;
                        const uint32_t idx = (p2 & kPairTransposed) ? (uint32_t)(nu * nI + mu) : (uint32_t)(mu * nJ + nu);
                        atomicAdd(H + (size_t)(p2 & ~kPairTransposed) + idx, acc[i][j][h]);
                    }
            }
        }
            TIMER_ADD(5)
            TIMER_COUNT(6)
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(s_dempty + ds));   // descriptor (row info, masks) no longer read
        }
        } else {
            rho_consumer(P, Din, H, s_full, s_empty, s_dfull, s_dempty, s_desc, s_ring, nring, never, lane, cidx);
        }
    }
#ifdef GINT_TIMING
    if (lane == 0 && blockIdx.x < 16) {
        long long* out = reinterpret_cast<long long*>(P.counter + 272) + (16 * blockIdx.x + warp) * 8;
        for (int k = 0; k < 8; k++) out[k] = tm_[k];
    }
#endif
}

// H(J,I,-R) = H(I,J,R)^T for every non-canonical block; lower <- upper for (I,I,0).
__global__ void __launch_bounds__(256) gint_mirror_kernel(const MirrorItem* __restrict__ items, int nitems,
                                                          double* __restrict__ H) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= nitems) return;
    const MirrorItem it = items[w];
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
size_t psi_kernel_smem(size_t table_bytes) { return eval_smem(table_bytes).total; }
size_t contract_kernel_smem(int nring) { return contract_smem(nring).total; }

cudaError_t configure_kernels(size_t psi_smem, size_t contract_smem_bytes, bool tab_smem) {
    cudaError_t e = tab_smem ? cudaFuncSetAttribute(gint_psi_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psi_smem)
                             : cudaFuncSetAttribute(gint_psi_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psi_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(gint_contract_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)contract_smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gint_contract_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)contract_smem_bytes);
}

cudaError_t launch_vlocal(const DevicePlan& P, size_t psi_smem, size_t contract_smem_bytes, bool tab_smem, int nsm,
                          size_t h_len, const double* V, double* H, cudaStream_t stream, cudaEvent_t* ev) {
    if (ev) cudaEventRecord(ev[0], stream);
    cudaError_t e = cudaMemsetAsync(H, 0, h_len * sizeof(double), stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int) * 257, stream);   // work-queue head + per-SM arrival counters
    if (e != cudaSuccess) return e;
    if (ev) cudaEventRecord(ev[1], stream);
    if (P.nitems > 0) {
        const int pgrid = P.nwork_regions < 3 * nsm ? P.nwork_regions : 3 * nsm;
        if (tab_smem)
            gint_psi_kernel<true><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
        else
            gint_psi_kernel<false><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[2], stream);
    if (P.nitems > 0) {
        const int grid = P.nitems < kCtasPerSm * nsm ? P.nitems : kCtasPerSm * nsm;
        gint_contract_kernel<0><<<grid, kThreads, contract_smem_bytes, stream>>>(P, nullptr, H);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[3], stream);
    if (P.nmirror > 0) {
        const int wpb = 256 / 32;
        gint_mirror_kernel<<<(P.nmirror + wpb - 1) / wpb, 256, 0, stream>>>(P.mirror, P.nmirror, H);
        e = cudaGetLastError();
    }
    if (ev) cudaEventRecord(ev[4], stream);
    return e;
}

cudaError_t launch_psi(const DevicePlan& P, size_t psi_smem, bool tab_smem, int nsm, const double* V, cudaStream_t stream) {
    if (P.nitems <= 0) return cudaSuccess;
    const int pgrid = P.nwork_regions < 3 * nsm ? P.nwork_regions : 3 * nsm;
    if (tab_smem)
        gint_psi_kernel<true><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
    else
        gint_psi_kernel<false><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
    return cudaGetLastError();
}

// gint_rho on the tensor pipe: rho <- 0, queue head <- 0, contraction kernel in MODE 1 (phi must be in the scratch)
cudaError_t launch_rho_dmma(const DevicePlan& P, size_t contract_smem_bytes, int nsm, const double* D, double* rho,
                            cudaStream_t stream) {
    const size_t npts = (size_t)P.ngrid[0] * P.ngrid[1] * P.ngrid[2];
    cudaError_t e = cudaMemsetAsync(rho, 0, npts * sizeof(double), stream);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int) * 257, stream);
    if (e != cudaSuccess || P.nitems <= 0) return e;
    const int grid = P.nitems < kCtasPerSm * nsm ? P.nitems : kCtasPerSm * nsm;
    gint_contract_kernel<1><<<grid, kThreads, contract_smem_bytes, stream>>>(P, D, rho);
    return cudaGetLastError();
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
