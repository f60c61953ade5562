// gint_kernels.cu -- sm_100a kernels of gint_vlocal (and gint_rho, which shares them).
//
//   H_mu,nu(R) = sum_g phi_mu(r_g - tau_I) V(r_g) phi_nu(r_g - tau_J - R) dV   (Eq. 45)
//
// Five kernels per gint_vlocal call (per batch of regions for the two in the middle, see launch_vlocal):
//
//   gint_vrange_kernel / gint_hinit_kernel   range of V, then H <- c S with S the grid overlap (Eq. 45 with
//       V = 1, computed once at setup) and c = max V (or min V, whichever is smaller in magnitude): the rest of
//       the call integrates the one-signed potential u = |V - c| >= 0,  H = c S -/+ sum_g phi u phi dV,  so that
//       the weight can be split evenly over the two operands of a SYMMETRIC product (no per-point sign).
//   gint_psi_kernel     psi = phi sqrt(u dV) for every (atom image, mesh point) pair listed by
//       the plan, evaluated exactly once -- Eq. 1: 4-point Lagrange radial table x real Y_lm, one
//       lane per mesh point -- and stored to a scratch buffer as chunks [k-step][row pair][point][parity] of
//       one (row group, 32-point stage).  The V dV weighting of Eq. 45 is thereby folded into the operand:
//       C = psi psi^T.
//   gint_contract_kernel<0>  (gint_vlocal) output-stationary contraction (the paper's per-BigGrid dense
//       contraction).  One persistent CTA per SM pulls work items from a global
//       queue; a work item is a set of up to 15 32x32 tiles (one per consumer warp) of the upper
//       triangle of a region's C (small left-over tile sets of several regions share an item).  A producer warp
//       stages the item descriptor and streams the row groups the tiles need through a ring of 8 KB chunk buffers in
//       shared memory (a 32-point stage takes one buffer per active row group) with cp.async.bulk + mbarrier, running
//       ahead across item boundaries; the 15 consumer warps keep their tile in registers and issue
//       mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4; tcgen05 has no FP64 kind).  (fragment, k-step) pairs that hold no
//       in-sphere point are skipped by warp-uniform control flow decided on the host (a predicated-off DMMA still
//       costs its 16 pipe cycles): per (warp, stage) a program of runs of k-steps with one fragment pattern, one
//       indexed jump per run into a software-pipelined loop for the pattern (gint_kstep_dispatch.inc).  After the
//       last stage the warp adds its tile into the canonical H blocks with red.global.add.f64 (once per item, not
//       once per BigGrid).
//   gint_contract_kernel<1>  (gint_rho, Eq. 44): same items, stages and producer;
//       see rho_consumer.
//   gint_mirror_kernel  writes every non-canonical block as the transpose of its partner,
//       H(J,I,-R) = H(I,J,R)^T, and symmetrises the (I,I,0) blocks.
#include <cuda_runtime.h>

#include <cstdint>

#include "gint_device.hpp"
#include "gint_kstep_dispatch.inc"

namespace gint {

namespace {

constexpr int kConsumerWarps = kTilesPerItem;          // 15
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kThreads = kConsumerThreads + 32;        // + 1 producer warp
constexpr int kKstepDoubles = kGroupRows * kKstepPts;  // 128: one k-step of a chunk, [row 32][point 4]

__device__ __forceinline__ void dmma8x8x4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// Operands of one k-step (4 mesh points) of a 32x32 tile: fragment i of the row group and of the column
// group.  In DMMA.8x8x4 lane l holds A[l/4][l%4] and B[l%4][l/4]; a chunk stores element (row r, point k)
// of k-step ks at ks*128 + (r/2)*8 + k*2 + r%2, so lane l = 4 q + k reads double number
// ks*128 + 32 i + (q/2)*8 + k*2 + q%2 of its chunk: the lanes of a fragment read a permutation of 32 consecutive
// doubles (conflict-free LDS.64).  pa / pb already include the lane's offset (frag_lane_offset).
struct Frag8 {
    double a0, a1, a2, a3, b0, b1, b2, b3;
};
__device__ __forceinline__ void load_kstep(Frag8& o, const double* __restrict__ pa, const double* __restrict__ pb, uint32_t pos) {
    const uint32_t off = pos * (kKstepDoubles / 4);   // pos = 4 * k-step
    o.a0 = pa[off];
    o.a1 = pa[off + 32];
    o.a2 = pa[off + 64];
    o.a3 = pa[off + 96];
    o.b0 = pb[off];
    o.b1 = pb[off + 32];
    o.b2 = pb[off + 64];
    o.b3 = pb[off + 96];
}
__device__ __forceinline__ int frag_lane_offset(int lane) { return ((lane >> 3) << 3) + ((lane & 3) << 1) + ((lane >> 2) & 1); }
__device__ __forceinline__ double flip_sign(double v, uint32_t x) {   // x = 0 or 0x80000000
    return __hiloint2double(__double2hiint(v) ^ (int)x, __double2loint(v));
}

// DMMAs of one k-step (4 mesh points) of a tile, for the fragment pairs whose rows AND columns hold an in-sphere
// point there (host-built 4-bit masks ra, ca).  A predicated-off DMMA still holds the FP64 tensor pipe for its 16
// cycles (measured), so inactive fragment pairs must be skipped by real, warp-uniform control flow; the cheapest
// form is ONE indexed jump (PTX brx.idx -> SASS BRX through a table in the constant bank) on the key ra | ca << 4
// into straight-line code for exactly that pattern: no per-row tests, no predication, every accumulator at a
// fixed register.  nvcc lowers a C++ switch over the patterns to a compare tree, so the jump and its 225 targets are
// one inline-PTX statement generated by gen_kstep_dispatch.py (gint_kstep_dispatch.inc).
#define KACC(i, j) "+d"(acc[i][j][0]), "+d"(acc[i][j][1])
#define KACC_ROW(i) KACC(i, 0), KACC(i, 1), KACC(i, 2), KACC(i, 3)
#define KSTEP_OPERANDS                                                                                           \
    : KACC_ROW(0), KACC_ROW(1), KACC_ROW(2), KACC_ROW(3)                                                         \
    : "d"(o.a0), "d"(o.a1), "d"(o.a2), "d"(o.a3), "d"(o.b0), "d"(o.b1), "d"(o.b2), "d"(o.b3), "r"(key)
// off-diagonal tile: key = ra | ca << 4
__device__ __forceinline__ void kstep_rect(double (&acc)[4][4][2], const Frag8& o, uint32_t key) {
    asm volatile(GINT_KSTEP_RECT_ASM KSTEP_OPERANDS);
}
// diagonal tile (row group == column group, ra == ca): fragment pairs i <= j with both active; key = ra
__device__ __forceinline__ void kstep_diag(double (&acc)[4][4][2], const Frag8& o, uint32_t key) {
    asm volatile(GINT_KSTEP_DIAG_ASM KSTEP_OPERANDS);
}
// A RUN of n consecutive k-steps with one pattern (the activity of a fragment along a stage is an interval, so
// patterns persist: 3.7 k-steps per run on the Si workloads): one jump per run into a software-pipelined loop that
// loads the next k-step's operands before the DMMAs of the current one are issued -- a single warp keeps the tensor
// pipe busy by itself.  pa / pb: shared-memory byte addresses of this lane's element of fragment 0 of the first
// k-step (k-steps are 1 KB apart, fragments 256 B).
#define KRUN_OPERANDS                                                                                            \
    : KACC_ROW(0), KACC_ROW(1), KACC_ROW(2), KACC_ROW(3)                                                         \
    : "r"(pa), "r"(pb), "r"(n), "r"(key)
// off-diagonal tile with all four row fragments active; key = column mask ca
__device__ __forceinline__ void run_rect(double (&acc)[4][4][2], uint32_t pa, uint32_t pb, uint32_t n, uint32_t key) {
    asm volatile(GINT_RUN_RECT_ASM KRUN_OPERANDS);
}
// diagonal tile (B = A, pairs i <= j); key = fragment mask ra
__device__ __forceinline__ void run_diag(double (&acc)[4][4][2], uint32_t pa, uint32_t n, uint32_t key) {
    const uint32_t pb = pa;
    asm volatile(GINT_RUN_DIAG_ASM KRUN_OPERANDS);
}
#undef KRUN_OPERANDS
#undef KACC
#undef KACC_ROW
#undef KSTEP_OPERANDS
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

// psi = phi sqrt(|V dV|) of one entry on the 32 points of a stage (lane = point), Eq. 1, stored to the
// region's scratch: element (row R, point p = 4 ks + k of stage s) sits at
//   chunk(R >> 5, s) + ks * 128 + ((R & 31) >> 1) * 8 + k * 2 + (R & 1)     (chunk(g, s) = (g * nstage + s) * 1024 doubles),
// i.e. [k-step][row pair][point][row parity]: a DMMA operand fragment of one k-step is a permutation of 32 consecutive
// doubles (one per lane, conflict-free LDS.64), and a lane stores two consecutive rows with one 16-byte store.
struct SpeciesDev {   // staged in shared memory by the psi kernel
    int32_t tab_off, ntab, nradp, norb;
    int32_t l[8];
    double rc2, inv_dr;
};
__device__ __forceinline__ void eval_task(const SpeciesDev& sp, const double* __restrict__ tab, double relx, double rely, double relz,
                                          int row0, int gstride, int stage, int lane, const double* __restrict__ s_off,
                                          const double* __restrict__ s_sqrtw, double* __restrict__ psi_stage) {
    const int nradp = sp.nradp;
    const int p = stage * kStagePts + lane;
    const double dx = relx + s_off[p];
    const double dy = rely + s_off[kMaxRegionPoints + p];
    const double dz = relz + s_off[2 * kMaxRegionPoints + p];
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const bool inside = r2 < sp.rc2;
    double rinv = 0.0, lnz = 0.0;   // lnz: 1 if the l>0 components survive (r >= 1e-12)
    if (r2 >= 1e-24) {
        const double y0 = rsqrt_seed(r2);              // relative error ~2^-22
        const double e = fma(-(r2 * y0), y0, 1.0);     // 1 - r2 y0^2
        rinv = fma(e * y0, fma(0.375, e, 0.5), y0);    // y0 (1 + e/2 + 3 e^2/8): cubic convergence
        lnz = 1.0;
    }
    const double r = r2 * rinv;
    const double x = dx * rinv, y = dy * rinv, z = dz * rinv;
    const double s = r * sp.inv_dr;
    int k = __double2int_rd(s);
    const double t = s - (double)k;
    k = inside ? min(k, sp.ntab) : sp.ntab;            // outside: the four zero nodes after the table
    const double t1 = 1.0 - t, t2 = 2.0 - t, t3 = 3.0 - t;
    const double a23 = t2 * t3, b01 = t * t1;
    const double sq = s_sqrtw[p];
    const double L0 = (t1 * a23) * (sq * (1.0 / 6.0));
    const double L1 = (t * a23) * (sq * 0.5);
    const double L2 = (b01 * t3) * (sq * -0.5);
    const double L3 = (b01 * t2) * (sq * (1.0 / 6.0));
    const double* Tk = tab + sp.tab_off + k * nradp;
    // store addressing: lane part + row part; rows go out in pairs (even row, odd row) = 16 bytes
    double* out = psi_stage + (lane >> 2) * kKstepDoubles + (lane & 3) * 2;
    int R = row0;
    double pending = 0.0;
    auto put = [&](double v) {
        double* dst = out + (R >> 5) * gstride + ((R & 31) >> 1) * 8;
        if (R & 1) {
            if (R == row0) dst[1] = v;                                         // entry starts on an odd row
            else *reinterpret_cast<double2*>(dst) = make_double2(pending, v);
        } else {
            pending = v;
        }
        R++;
    };
    auto emit = [&](int l, double fv) {
        if (l == 0) {
            put(fv);
        } else if (l == 1) {
            put(fv * y);
            put(fv * z);
            put(fv * x);
        } else if (l == 2) {
            // table carries 1/2 sqrt(15/pi); ratios: 1/4 sqrt(5/pi) / that = 1/(2 sqrt 3), 1/4 sqrt(15/pi) / that = 1/2
            put(fv * (x * y));
            put(fv * (y * z));
            put(fv * (fma(3.0 * z, z, -lnz) * 0.28867513459481288));
            put(fv * (x * z));
            put(fv * (fma(x, x, -(y * y)) * 0.5));
        } else {
            // l = 3, m = -3..3; table carries 1/2 sqrt(105/pi); ratios 1/(2 sqrt 6), 1/(2 sqrt 10), 1/(2 sqrt 15), 1/2
            const double x2 = x * x, y2 = y * y, q = fma(5.0 * z, z, -lnz);
            put(fv * (0.20412414523193151 * y * fma(3.0, x2, -y2)));
            put(fv * (x * y * z));
            put(fv * (0.15811388300841897 * y * q));
            put(fv * (0.12909944487358055 * z * fma(5.0 * z, z, -3.0 * lnz)));
            put(fv * (0.15811388300841897 * x * q));
            put(fv * (0.5 * z * (x2 - y2)));
            put(fv * (0.20412414523193151 * x * fma(-3.0, y2, x2)));
        }
    };
    for (int f = 0; f < nradp; f += 2) {
        const double2 T0 = *reinterpret_cast<const double2*>(Tk + f);
        const double2 T1 = *reinterpret_cast<const double2*>(Tk + nradp + f);
        const double2 T2 = *reinterpret_cast<const double2*>(Tk + 2 * nradp + f);
        const double2 T3 = *reinterpret_cast<const double2*>(Tk + 3 * nradp + f);
        const int l0 = sp.l[f];
        const int l1 = (f + 1 < 8) ? sp.l[f + 1] : -1;
        emit(l0, fma(T0.x, L0, fma(T1.x, L1, fma(T2.x, L2, T3.x * L3))));
        if (l1 >= 0) emit(l1, fma(T0.y, L0, fma(T1.y, L1, fma(T2.y, L2, T3.y * L3))));
    }
    if (R & 1) out[((R - 1) >> 5) * gstride + (((R - 1) & 31) >> 1) * 8] = pending;   // last row was an even one
}

}  // namespace
// ---- kernel 1: psi = phi sqrt(|V dV|) of every region, evaluated once ---------------------------
// One CTA per region (with work): stage sqrt(u dV), u = |V - c| (see gint_hinit_kernel), of the region's points, then
// the warps walk the region's (atom image, run of stages) tasks.  Plenty of warps per SM (3 CTAs of 8
// warps) hide the table and entry latencies; the output is 8.5 GB at si512_dzp.
constexpr int kEvalThreads = 256;
constexpr int kEvalCtasPerSm = 2;

struct EvalSmem {
    uint32_t off, xyz, sqrtw, spec, tab, total;
};
GINT_HD inline EvalSmem eval_smem(size_t table_bytes, int nspecies) {
    EvalSmem L;
    uint32_t o = 0;
    L.off = o;   o += 3 * kMaxRegionPoints * 8;
    L.xyz = o;   o += kMaxRegionPoints * 4;
    L.sqrtw = o; o += 2 * kMaxRegionPoints * 8;   // two regions (double buffer)
    L.spec = o;  o += smem_align((size_t)nspecies * sizeof(SpeciesDev));
    L.tab = o;   o += smem_align(table_bytes);
    L.total = o;
    return L;
}

template <bool TAB_SMEM>
__global__ void __launch_bounds__(kEvalThreads, kEvalCtasPerSm)
gint_psi_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ V) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const EvalSmem L = eval_smem(TAB_SMEM ? (size_t)P.tab_doubles * sizeof(double) : 0, P.nspecies);
    double* s_off = reinterpret_cast<double*>(smem_raw + L.off);
    uchar4* s_xyz = reinterpret_cast<uchar4*>(smem_raw + L.xyz);
    double* s_sqrtw2 = reinterpret_cast<double*>(smem_raw + L.sqrtw);
    double* s_tab = reinterpret_cast<double*>(smem_raw + L.tab);
    SpeciesDev* s_spec = reinterpret_cast<SpeciesDev*>(smem_raw + L.spec);
    if (TAB_SMEM) {
        for (int i = tid; i < P.tab_doubles; i += kEvalThreads) s_tab[i] = __ldg(P.tab + i);
    }
    for (int i = tid; i < P.nspecies; i += kEvalThreads) {
        const int32_t* meta = P.sp_meta + 12 * i;
        SpeciesDev sd;
        sd.tab_off = meta[0]; sd.ntab = meta[1]; sd.nradp = meta[2]; sd.norb = meta[3];
        for (int k = 0; k < 8; k++) sd.l[k] = meta[4 + k];
        sd.rc2 = P.sp_real[2 * i]; sd.inv_dr = P.sp_real[2 * i + 1];
        s_spec[i] = sd;
    }
    const double* tab = TAB_SMEM ? s_tab : P.tab;
    const int npt = P.nstage * kStagePts;
    for (int p = tid; p < npt; p += kEvalThreads) {
        const uchar4 c = reinterpret_cast<const uchar4*>(P.slot_xyz)[p];
        for (int k = 0; k < 3; k++)
            s_off[k * kMaxRegionPoints + p] = c.x * P.estep[k] + c.y * P.estep[3 + k] + c.z * P.estep[6 + k];
        s_xyz[p] = c;
    }
    const double vshift = V ? P.shift->c : 0.0;
    // sqrt(u dV) of a region's points, two points per thread; the values of the NEXT region are fetched (work list ->
    // region origin -> V: three dependent global loads) while the tasks of the current one run, into the other buffer
    auto fetch_w = [&](int r, double (&w)[kMaxRegionPoints / kEvalThreads]) {
        const Region* reg = P.regions + __ldg(P.work_regions + r);
        const int ox = __ldg(&reg->origin[0]), oy = __ldg(&reg->origin[1]), oz = __ldg(&reg->origin[2]);
#pragma unroll
        for (int k = 0; k < kMaxRegionPoints / kEvalThreads; k++) {
            const int p = tid + k * kEvalThreads;
            w[k] = 0.0;
            if (p < npt) {
                const uchar4 c = s_xyz[p];
                const int g1 = ox + c.x, g2 = oy + c.y, g3 = oz + c.z;
                if (c.w && g1 < P.ngrid[0] && g2 < P.ngrid[1] && g3 < P.ngrid[2])   // V == nullptr: plain phi (gint_rho)
                    w[k] = V ? (__ldg(V + ((size_t)g1 * P.ngrid[1] + g2) * P.ngrid[2] + g3) - vshift) * P.dV : 1.0;
            }
        }
    };
    auto store_w = [&](double* dst, const double (&w)[kMaxRegionPoints / kEvalThreads]) {
#pragma unroll
        for (int k = 0; k < kMaxRegionPoints / kEvalThreads; k++) {
            const int p = tid + k * kEvalThreads;
            if (p < npt) dst[p] = sqrt(fabs(w[k]));
        }
    };
    __syncthreads();   // s_xyz, tables and species staged
    double wnext[kMaxRegionPoints / kEvalThreads];
    int buf = 0;
    if ((int)blockIdx.x < P.nwork_regions) {
        fetch_w(blockIdx.x, wnext);
        store_w(s_sqrtw2, wnext);
    }
    __syncthreads();
    for (int r = blockIdx.x; r < P.nwork_regions; r += gridDim.x) {
        const double* s_sqrtw = s_sqrtw2 + buf * kMaxRegionPoints;
        const bool more = r + (int)gridDim.x < P.nwork_regions;
        if (more) fetch_w(r + gridDim.x, wnext);
        const Region* reg = P.regions + __ldg(P.work_regions + r);
        const int ntask = __ldg(&reg->ntask);
        const uint32_t* tasks = P.etasks + __ldg(&reg->task_off);
        const Entry* entries = P.entries + __ldg(&reg->entry0);
        double* psi_region = P.psi + (size_t)__ldg(&reg->psi_chunk0) * kChunkDoubles;
        const int gstride = P.nstage * kChunkDoubles;
        // the entry of a task (position, species, first row, activity of the run's 8 stages: byte s of the 64 k-step
        // bits starting at stage s0) is fetched one task ahead: two dependent global loads hidden behind an evaluation
        struct TaskRegs { double relx, rely, relz; int rp, row0, s0, norb; uint2 km; };
        auto fetch_task = [&](int t, TaskRegs& tr) {
            const uint32_t tk = __ldg(tasks + t);
            const Entry* en = entries + (tk & 0xFFFFu);
            tr.s0 = (int)(tk >> 16) * 8;
            tr.relx = __ldg(&en->rel[0]); tr.rely = __ldg(&en->rel[1]); tr.relz = __ldg(&en->rel[2]);
            tr.rp = __ldg(&en->Rpack); tr.row0 = __ldg(&en->row0); tr.norb = __ldg(&en->norb);
            tr.km = __ldg(reinterpret_cast<const uint2*>(&en->kmask[tr.s0 >> 2]));
        };
        TaskRegs nxt;
        if (warp < ntask) fetch_task(warp, nxt);
        for (int t = warp; t < ntask; t += kEvalThreads / 32) {
            const TaskRegs cur = nxt;
            if (t + kEvalThreads / 32 < ntask) fetch_task(t + kEvalThreads / 32, nxt);
            const double relx = cur.relx, rely = cur.rely, relz = cur.relz;
            const int spi = (cur.rp >> 24) & 0x7F, row0 = cur.row0, s0 = cur.s0;
            const uint2 km = cur.km;
            const SpeciesDev& sp = s_spec[spi];
            for (int q = 0; q < 8 && s0 + q < P.nstage; q++) {
                const int stage = s0 + q;
                if ((((q < 4 ? km.x : km.y) >> (8 * (q & 3))) & 0xFFu) == 0u) {
                    // No point of the stage inside the sphere.  With one batch the rows stay zero from the memset at
                    // setup; when batches share the scratch they hold another region's values and are zeroed here,
                    // in the chunks that will be read (row group active in the stage).
                    if (P.multibatch) {
                        const uint8_t* gm = P.gmask + __ldg(&reg->gmask_off) + (size_t)stage * kStageKsteps;
                        double* out = psi_region + (size_t)stage * kChunkDoubles + (lane >> 2) * kKstepDoubles + (lane & 3) * 2;
                        for (int R = row0; R < row0 + cur.norb; R++) {
                            if (*reinterpret_cast<const unsigned long long*>(gm + (size_t)(R >> 5) * P.nks_pad) != 0ull)
                                out[(R >> 5) * gstride + ((R & 31) >> 1) * 8 + (R & 1)] = 0.0;
                        }
                    }
                    continue;
                }
                eval_task(sp, tab, relx, rely, relz, row0, gstride, stage, lane, s_off, s_sqrtw,
                          psi_region + (size_t)stage * kChunkDoubles);
            }
        }
        if (more) store_w(s_sqrtw2 + (buf ^ 1) * kMaxRegionPoints, wnext);
        buf ^= 1;
        __syncthreads();   // next region's weights visible; this region's no longer read
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
    L.ring = o;  o += (uint32_t)nring * kChunkBytes;
    L.total = o;
    return L;
}

// bit 4 ks set iff nibble ks of m is non-zero
__device__ __forceinline__ uint32_t nonzero_nibbles(uint32_t m) { return (m | (m >> 1) | (m >> 2) | (m >> 3)) & 0x11111111u; }

// ---- gint_rho on the tensor pipe (MODE 1 of the contraction kernel) --------------------------------
//   rho(p) = sum over tiles (ga <= gb) of  Phi_ga(p)^T E Phi_gb(p),   E = D[ga][gb] + D[gb][ga]^T  (ga < gb),
//                                                                      E = D[ga][ga]               (ga = gb),
// D[.][.] being the region's density matrix gathered from the blocks (entry a, entry b) -> (I_a, I_b, R_b - R_a)
// (Eq. 44; no symmetry of D is assumed).  The warp holds E as 4 x 8 A fragments
// (rows 8 i + lane/4, columns 4 kc + lane%4) in registers for the whole item.  Per k-pair (8 mesh points) it
// forms T = E Phi_gb as 4 accumulator fragments (rows x 8 points) with the B operand read from the stage
// (rows of gb are the K dimension, the 8 points the N dimension), multiplies by Phi_ga in the accumulator
// layout, reduces over the rows by shuffles and adds the 8 point values into rho with red.global.add.f64.
#define RHO_GUARD(cond, body)          \
    if (cond) {                        \
        do { body } while (never);     \
    }
__device__ __forceinline__ void rho_consumer(const DevicePlan& P, const double* __restrict__ D, double* __restrict__ rho,
                                             uint64_t* s_full, uint64_t* s_empty, uint64_t* s_dfull, uint64_t* s_dempty,
                                             const ItemDesc* s_desc, const unsigned char* s_ring, int nring, int never,
                                             int lane, int cidx) {
    const int frow = lane >> 2, fk = lane & 3;
    uint32_t cseq = 0, cpos = 0;   // as in the gint_vlocal consumer
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
            const uint32_t* pdir = P.pair_direct + cur->slot[sa].pair_off;
            const int m = cur->slot[sa].nentry;
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
        const SlotInfo& reg = cur->slot[has_tile ? sa : 0];
        const int ox = reg.origin[0], oy = reg.origin[1], oz = reg.origin[2];
        uint32_t todo = cur->item.stage_mask;
        while (todo) {
            const int s = __ffs(todo) - 1;
            todo &= todo - 1;
            uint32_t ma = 0, mb = 0;   // per k-pair kp: nibble 2 kp = OR of the activity of its two k-steps
            if (has_tile) {
                ma = cur->gm32[sa][s];
                mb = cur->gm32[sb][s];
                ma |= ma >> 4;
                mb |= mb >> 4;
            }
            const uint32_t act = cur->act[s];
            mbar_wait(smem_u32(s_full + (cseq & 7u)), (cseq >> 3) & 1u);
            if (has_tile) {
                uint32_t ca = cpos + (uint32_t)__popc(act & ((1u << sa) - 1u)), cb = cpos + (uint32_t)__popc(act & ((1u << sb) - 1u));
                if (ca >= (uint32_t)nring) ca -= (uint32_t)nring;
                if (cb >= (uint32_t)nring) cb -= (uint32_t)nring;
                const double* chA = reinterpret_cast<const double*>(s_ring + (size_t)ca * kChunkBytes);
                const double* chB = reinterpret_cast<const double*>(s_ring + (size_t)cb * kChunkBytes);
#pragma unroll 1
                for (int kp = 0; kp < kStageKsteps / 2; kp++) {
                    const uint32_t ra = (ma >> (8 * kp)) & 0xFu;
                    const uint32_t ca = (mb >> (8 * kp)) & 0xFu;
                    if (ra == 0u || ca == 0u) continue;
                    double C[4][2];
#pragma unroll
                    for (int i = 0; i < 4; i++) C[i][0] = C[i][1] = 0.0;
                    // B operand of k-step kc = 2 j + h2: Phi_gb[row 8 j + 4 h2 + lane%4][point lane/4 of the k-pair];
                    // point q of the k-pair is point q % 4 of k-step 2 kp + q / 4
                    const double* bsrc = chB + (2 * kp + (frow >> 2)) * kKstepDoubles + (fk >> 1) * 8 + (frow & 3) * 2 + (fk & 1);
                    if ((ra & ca) == 0xFu) {
#pragma unroll
                        for (int kc = 0; kc < 8; kc++) {
                            const double b = bsrc[kc * 16];
#pragma unroll
                            for (int i = 0; i < 4; i++) dmma8x8x4(C[i][0], C[i][1], A[i][kc], b);
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 4; j++) {
                            // blocks of 8 DMMAs on 4 accumulators (all four row fragments: guarding single row
                            // fragments costs more in lost instruction-level parallelism than the skipped DMMAs save)
                            RHO_GUARD(ca & (1u << j), {
                                const double b0 = bsrc[j * 32];
                                const double b1 = bsrc[j * 32 + 16];
#pragma unroll
                                for (int i = 0; i < 4; i++) dmma8x8x4(C[i][0], C[i][1], A[i][2 * j], b0);
#pragma unroll
                                for (int i = 0; i < 4; i++) dmma8x8x4(C[i][0], C[i][1], A[i][2 * j + 1], b1);
                            })
                        }
                    }
                    // C[i][h] = T[row 8 i + lane/4][point 2 (lane%4) + h]: times Phi_ga there, summed over the rows
                    double p0 = 0.0, p1 = 0.0;
                    const double* asrc = chA + (2 * kp + (fk >> 1)) * kKstepDoubles + (frow >> 1) * 8 + 4 * (fk & 1) + (frow & 1);
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        if ((ra >> i) & 1u) {
                            p0 = fma(asrc[i * 32], C[i][0], p0);
                            p1 = fma(asrc[i * 32 + 2], C[i][1], p1);
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
            if (lane == 0) mbar_arrive(smem_u32(s_empty + (cseq & 7u)));
            cseq++;
            cpos += (uint32_t)__popc(act);
            if (cpos >= (uint32_t)nring) cpos -= (uint32_t)nring;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(s_dempty + ds));
    }
}
#undef RHO_GUARD

// MODE 0: gint_vlocal (H -/+= psi psi^T, Eq. 45 with the one-signed potential).  MODE 1: gint_rho (Eq. 44): the same items, stages and
// producer; a consumer warp keeps its 32x32 tile of the region's density matrix in registers as the A operand,
// forms T = E Phi_b on the tensor pipe per 8 points and dots it with Phi_a (rho_consumer above).
template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
gint_contract_kernel(const __grid_constant__ DevicePlan P, const double* __restrict__ Din, double* __restrict__ H) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const ContractSmem L = contract_smem(P.nring);
    uint64_t* s_full = reinterpret_cast<uint64_t*>(smem_raw + L.bar);         // [8] stage filled (tx bytes)
    uint64_t* s_empty = s_full + 8;                                           // [8] stage released by the 15 consumer warps
    uint64_t* s_dfull = s_full + 16;                                          // [4] descriptor staged
    uint64_t* s_dempty = s_full + 20;                                         // [4] descriptor released
    ItemDesc* s_desc = reinterpret_cast<ItemDesc*>(smem_raw + L.desc);        // [kDescSlots]
    unsigned char* s_ring = smem_raw + L.ring;                                // [nring] chunk buffers of 8 KB
    const int nring = P.nring;
    const int never = P.never;   // always 0; see KROW

    if (tid == 0) {
        for (int i = 0; i < kRingMaxStages; i++) {
            mbar_init(smem_u32(s_full + i), 1);
            mbar_init(smem_u32(s_empty + i), kConsumerWarps);
        }
        for (int i = 0; i < kDescSlots; i++) {
            mbar_init(smem_u32(s_dfull + i), 1);
            mbar_init(smem_u32(s_dempty + i), kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    __syncthreads();
    // consumer warp w runs on SM sub-partition w % 4 and takes tile w of the item (the plan balances the four
    // sub-partitions' DMMA counts; sub-partition 3 also hosts the producer warp and gets one tile fewer)
    const int cidx = warp;

    if (warp == kConsumerWarps) {
        // ================= producer warp =================
        // Descriptor i+1 is fetched (one bulk copy straight into the slot, completion on its own
        // mbarrier) while the stages of item i are being streamed; the queue index is taken one more
        // item ahead so that the atomic's latency is off the critical path as well.
        // The ring is a circle of nring 8 KB chunk buffers; a stage takes as many consecutive buffers as it has active
        // chunks (5.9 on average, not 8), so more stages are in flight and a warp that is ahead waits less often.
        // Stage number seq uses the barrier pair seq % 8.  All lanes keep the same bookkeeping.
        uint32_t seq = 0, tail = 0, head = 0, inflight = 0, cnt_word = 0;   // cnt_word: 4 bits per barrier pair = chunks held
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
            // lane q copies the chunks of slot q; lane 0 also owns the barriers
            const unsigned char* src_lane = reinterpret_cast<const unsigned char*>(P.psi) +
                                            (size_t)(lane < nslot ? cur->slot[lane].chunk0 : 0) * kChunkBytes;
            uint32_t todo = cur->item.stage_mask;
            while (todo) {
                const int s = __ffs(todo) - 1;
                todo &= todo - 1;
                const uint32_t act = cur->act[s];
                const uint32_t c = (uint32_t)__popc(act);
                while (inflight + c > (uint32_t)nring || seq - tail >= (uint32_t)kRingMaxStages) {   // oldest stage released?
                    mbar_wait(smem_u32(s_empty + (tail & 7u)), (tail >> 3) & 1u);
                    inflight -= (cnt_word >> (4u * (tail & 7u))) & 15u;
                    tail++;
                }
                const uint32_t slot = seq & 7u, bar = smem_u32(s_full + slot);
                if (lane == 0) {
                    if (act) mbar_arrive_expect_tx(bar, c * kChunkBytes);
                    else mbar_arrive(bar);
                }
                __syncwarp();
                if ((act >> lane) & 1u) {
                    uint32_t pos = head + (uint32_t)__popc(act & ((1u << lane) - 1u));
                    if (pos >= (uint32_t)nring) pos -= (uint32_t)nring;
                    bulk_g2s(smem_u32(s_ring) + pos * kChunkBytes, src_lane + (size_t)s * kChunkBytes, kChunkBytes, bar);
                }
                cnt_word = (cnt_word & ~(15u << (4u * slot))) | (c << (4u * slot));
                head += c;
                if (head >= (uint32_t)nring) head -= (uint32_t)nring;
                inflight += c;
                seq++;
            }
        }
    } else {
        // ================= consumer warps =================
        if constexpr (MODE == 0) {
            const int frow = lane >> 2, fk = lane & 3;
            const int lane_off = frag_lane_offset(lane);
            const uint32_t ring_u32 = smem_u32(s_ring);

            uint32_t cseq = 0, cpos = 0;   // number of the next stage to consume and its first chunk buffer in the ring
            for (int it = 0;; it++) {
                const int ds = it % kDescSlots;
                mbar_wait(smem_u32(s_dfull + ds), ((uint32_t)it / kDescSlots) & 1u);
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
                while (todo) {
                    const int s = __ffs(todo) - 1;
                    todo &= todo - 1;
                    // this warp's program for the stage: up to 8 runs of k-steps (host-built, see pack_run), 0-terminated
                    uint2 pg = make_uint2(0u, 0u), pg2 = make_uint2(0u, 0u);
                    if (has_tile) {
                        const uint4 w4 = *reinterpret_cast<const uint4*>(&cur->prog[cidx][s][0]);
                        pg = make_uint2(w4.x, w4.y);
                        pg2 = make_uint2(w4.z, w4.w);
                    }
                    const uint32_t act = cur->act[s];
                    mbar_wait(smem_u32(s_full + (cseq & 7u)), (cseq >> 3) & 1u);
                    if (pg.x) {
                        // the stage's active chunks sit in consecutive ring buffers from cpos on, in slot order
                        uint32_t ca = cpos + (uint32_t)__popc(act & ((1u << sa) - 1u)), cb = cpos + (uint32_t)__popc(act & ((1u << sb) - 1u));
                        if (ca >= (uint32_t)nring) ca -= (uint32_t)nring;
                        if (cb >= (uint32_t)nring) cb -= (uint32_t)nring;
                        const uint32_t pa = ring_u32 + ca * kChunkBytes + lane_off * 8, pb = ring_u32 + cb * kChunkBytes + lane_off * 8;
                        do {
                            const uint32_t run = pg.x;
                            const uint32_t off = (run << 2) & 0x1C00u;             // first k-step x 1 KB
                            const uint32_t n = ((run >> 11) & 7u) + 1u;
                            if (diag) {
                                run_diag(acc, pa + off, n, (run >> 4) & 0xFu);
                            } else if ((run & 0xF0u) == 0xF0u) {
                                run_rect(acc, pa + off, pb + off, n, run & 0xFu);
                            } else {   // rare (2.5 % of the DMMAs): k-step by k-step
                                const double* ga = reinterpret_cast<const double*>(s_ring + (size_t)ca * kChunkBytes) + lane_off;
                                const double* gb = reinterpret_cast<const double*>(s_ring + (size_t)cb * kChunkBytes) + lane_off;
#pragma unroll 1
                                for (uint32_t q = 0; q < n; q++) {
                                    Frag8 o;
                                    load_kstep(o, ga, gb, ((run >> 6) & 0x1Cu) + 4 * q);
                                    kstep_rect(acc, o, ((run >> 4) & 0xFu) | ((run & 0xFu) << 4));
                                }
                            }
                            // next run word (16 bits each)
                            pg.x = (pg.x >> 16) | (pg.y << 16);
                            pg.y = (pg.y >> 16) | (pg2.x << 16);
                            pg2.x = (pg2.x >> 16) | (pg2.y << 16);
                            pg2.y >>= 16;
                        } while (pg.x & 0xFFFFu);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(smem_u32(s_empty + (cseq & 7u)));
                    cseq++;
                    cpos += (uint32_t)__popc(act);
                    if (cpos >= (uint32_t)nring) cpos -= (uint32_t)nring;
                }

                // ---------------- flush: add the tile into the canonical H blocks ---------------------------
                if (has_tile) {
                    const PairWord* pair = P.pair + cur->slot[sa].pair_off;
                    const int m = cur->slot[sa].nentry;
                    const uint32_t negbit = P.shift->neg << 31;   // H = c S - C (c = max V) or c S + C (c = min V)
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
                        const uint32_t ri = cur->rinfo[sa][8 * i + frow];
                        if (ri == kNoBlock) continue;
                        const PairWord* prow = pair + (ri & 0xFFFu) * m;
                        const uint32_t mu = (ri >> 12) & 0xFFu;
                        // all pair-table look-ups of the row first (independent loads), then the reductions
                        uint2 pw[4][2];
#pragma unroll
                        for (int j = 0; j < 4; j++)
#pragma unroll
                            for (int h = 0; h < 2; h++) {
                                // diagonal tile: fragments i > j were never computed (zero), i == j needs row <= column
                                // zero test on the bits: an FP64 compare would take a slot of the pipe the DMMAs run on
                                const bool nz = (((uint32_t)__double2hiint(acc[i][j][h]) << 1) | (uint32_t)__double2loint(acc[i][j][h])) != 0u;
                                const bool ok = ci[j][h] != kNoBlock && nz && !(diag && i == j && frow > 2 * fk + h);
                                pw[j][h] = ok ? __ldg(reinterpret_cast<const uint2*>(prow + (ci[j][h] & 0xFFFu)))
                                              : make_uint2(kNoBlock, 0u);
                            }
#pragma unroll
                        for (int j = 0; j < 4; j++)
#pragma unroll
                            for (int h = 0; h < 2; h++) {
                                if (pw[j][h].x == kNoBlock) continue;
                                const uint32_t nu = (ci[j][h] >> 12) & 0xFFu;
                                const uint32_t idx = mu * (pw[j][h].y & 0xFFFFu) + nu * (pw[j][h].y >> 16);
                                atomicAdd(H + (size_t)pw[j][h].x + idx, flip_sign(acc[i][j][h], negbit));
                            }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(s_dempty + ds));   // descriptor (row info, masks) no longer read
            }
        } else {
            rho_consumer(P, Din, H, s_full, s_empty, s_dfull, s_dempty, s_desc, s_ring, nring, never, lane, cidx);
        }
    }
}

// ---- one-signed potential: H = c S -/+ sum_g phi |V - c| phi dV ---------------------------------------------------
// gint_vrange_kernel: per-block (min, max) of V.  gint_hinit_kernel: every block reduces the partials to the range
// of V, picks the shift c -- max V (then u = c - V >= 0 and H = c S - C) or min V (u = V - c, H = c S + C),
// whichever is smaller in magnitude, so that |c S| <= max|V| |S| and nothing is lost to cancellation -- block 0
// publishes it for the psi and contraction kernels, and all blocks write H <- c S.
constexpr int kRangeBlocks = 296, kRangeThreads = 256;

__device__ __forceinline__ void block_minmax(double& lo, double& hi, double* s_red /* [2 * 32] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { s_red[warp] = lo; s_red[32 + warp] = hi; }
    __syncthreads();
    if (warp == 0) {
        lo = lane < nw ? s_red[lane] : s_red[0];
        hi = lane < nw ? s_red[32 + lane] : s_red[32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) { s_red[0] = lo; s_red[32] = hi; }
    }
    __syncthreads();
    lo = s_red[0];
    hi = s_red[32];
}

__global__ void __launch_bounds__(kRangeThreads) gint_vrange_kernel(const double* __restrict__ V, size_t n, double* __restrict__ part) {
    __shared__ double s_red[64];
    double lo = V[0], hi = lo;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double v = __ldg(V + i);
        lo = fmin(lo, v);
        hi = fmax(hi, v);
    }
    block_minmax(lo, hi, s_red);
    if (threadIdx.x == 0) { part[2 * blockIdx.x] = lo; part[2 * blockIdx.x + 1] = hi; }
}

__global__ void __launch_bounds__(kRangeThreads) gint_hinit_kernel(const double* __restrict__ part, int npart,
                                                                   const double* __restrict__ S, double* __restrict__ H, size_t h_len,
                                                                   ShiftDev* __restrict__ shift) {
    __shared__ double s_red[64];
    double lo = part[0], hi = part[1];
    for (int i = threadIdx.x; i < npart; i += blockDim.x) {
        lo = fmin(lo, part[2 * i]);
        hi = fmax(hi, part[2 * i + 1]);
    }
    block_minmax(lo, hi, s_red);
    const bool neg = fabs(hi) <= fabs(lo);   // c = max V, u = c - V, H = c S - C
    const double c = neg ? hi : lo;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        shift->c = c;
        shift->neg = neg ? 1u : 0u;
    }
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < h_len; i += (size_t)gridDim.x * blockDim.x)
        H[i] = c == 0.0 ? 0.0 : c * __ldg(S + i);
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
size_t psi_kernel_smem(size_t table_bytes, int nspecies) { return eval_smem(table_bytes, nspecies).total; }
size_t contract_kernel_smem(int nring) { return contract_smem(nring).total; }

cudaError_t configure_kernels(size_t psi_smem, size_t contract_smem_bytes, bool tab_smem) {
    cudaError_t e = tab_smem ? cudaFuncSetAttribute(gint_psi_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psi_smem)
                             : cudaFuncSetAttribute(gint_psi_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psi_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(gint_contract_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)contract_smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gint_contract_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)contract_smem_bytes);
}

// the parameter block of one batch: its slice of the work-region list and of the item queue
DevicePlan batch_plan(const DevicePlan& P, const BatchRange& B) {
    DevicePlan Q = P;
    Q.descs = P.descs + B.item0;
    Q.nitems = B.nitems;
    Q.work_regions = P.work_regions + B.wr0;
    Q.nwork_regions = B.nwr;
    return Q;
}

cudaError_t launch_psi(const DevicePlan& P, size_t psi_smem, bool tab_smem, int nsm, const double* V, cudaStream_t stream) {
    if (P.nitems <= 0) return cudaSuccess;
    const int pgrid = P.nwork_regions < kEvalCtasPerSm * nsm ? P.nwork_regions : kEvalCtasPerSm * nsm;
    if (tab_smem)
        gint_psi_kernel<true><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
    else
        gint_psi_kernel<false><<<pgrid, kEvalThreads, psi_smem, stream>>>(P, V);
    return cudaGetLastError();
}

// raw = true: no shift (c = 0, H <- sum_g phi V phi dV for a non-negative V): used once at setup to build S.
cudaError_t launch_vlocal(const DevicePlan& P, size_t psi_smem, size_t contract_smem_bytes, bool tab_smem, int nsm,
                          const BatchRange* batches, int nbatch, size_t h_len, const double* V, double* H, bool raw,
                          cudaStream_t stream, cudaEvent_t* ev) {
    if (ev) cudaEventRecord(ev[0], stream);
    cudaError_t e;
    if (raw) {
        if ((e = cudaMemsetAsync(P.shift, 0, sizeof(ShiftDev), stream)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(H, 0, h_len * sizeof(double), stream)) != cudaSuccess) return e;
    } else {
        const size_t npts = (size_t)P.ngrid[0] * P.ngrid[1] * P.ngrid[2];
        gint_vrange_kernel<<<kRangeBlocks, kRangeThreads, 0, stream>>>(V, npts, P.vpart);
        gint_hinit_kernel<<<4 * nsm, kRangeThreads, 0, stream>>>(P.vpart, kRangeBlocks, P.S, H, h_len, P.shift);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[1], stream);
    for (int b = 0; b < nbatch; b++) {
        const DevicePlan Q = batch_plan(P, batches[b]);
        if (Q.nitems <= 0) continue;
        if ((e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int) * 4, stream)) != cudaSuccess) return e;   // work-queue head
        if ((e = launch_psi(Q, psi_smem, tab_smem, nsm, V, stream)) != cudaSuccess) return e;
        if (ev && b == nbatch - 1) cudaEventRecord(ev[2], stream);
        const int grid = Q.nitems < nsm ? Q.nitems : nsm;
        gint_contract_kernel<0><<<grid, kThreads, contract_smem_bytes, stream>>>(Q, nullptr, H);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    if (ev && (nbatch == 0 || batches[nbatch - 1].nitems <= 0)) cudaEventRecord(ev[2], stream);
    if (ev) cudaEventRecord(ev[3], stream);
    e = cudaSuccess;
    if (P.nmirror > 0) {
        const int wpb = 256 / 32;
        gint_mirror_kernel<<<(P.nmirror + wpb - 1) / wpb, 256, 0, stream>>>(P.mirror, P.nmirror, H);
        e = cudaGetLastError();
    }
    if (ev) cudaEventRecord(ev[4], stream);
    return e;
}

// gint_rho on the tensor pipe: rho <- 0; per batch: phi (psi kernel with unit weights), queue head <- 0, contraction
// kernel in MODE 1
cudaError_t launch_rho(const DevicePlan& P, size_t psi_smem, size_t contract_smem_bytes, bool tab_smem, int nsm,
                       const BatchRange* batches, int nbatch, const double* D, double* rho, cudaStream_t stream) {
    const size_t npts = (size_t)P.ngrid[0] * P.ngrid[1] * P.ngrid[2];
    cudaError_t e = cudaMemsetAsync(rho, 0, npts * sizeof(double), stream);
    if (e != cudaSuccess) return e;
    for (int b = 0; b < nbatch; b++) {
        const DevicePlan Q = batch_plan(P, batches[b]);
        if (Q.nitems <= 0) continue;
        if ((e = cudaMemsetAsync(P.counter, 0, sizeof(unsigned int) * 4, stream)) != cudaSuccess) return e;
        if ((e = launch_psi(Q, psi_smem, tab_smem, nsm, nullptr, stream)) != cudaSuccess) return e;
        const int grid = Q.nitems < nsm ? Q.nitems : nsm;
        gint_contract_kernel<1><<<grid, kThreads, contract_smem_bytes, stream>>>(Q, D, rho);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
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
