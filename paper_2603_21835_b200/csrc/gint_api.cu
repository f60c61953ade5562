// gint_api.cu -- extern "C" boundary of libgint_b200.so (declared in include/gint.h).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/gint.h"
#include "gint_device.hpp"
#include "gint_plan.hpp"


struct gint_ctx {
    gint::Plan plan;
    gint::DevicePlan dev{};
    int device = -1;
    int nsm = 0;
    std::vector<void*> allocs;
    gint::FoldPlan fold{};
    double2* fold_static_phase = nullptr;   // gint_fold_k_static: device address of the library's fixed phase array
    std::vector<int64_t> first_orb;   // [natom+1]
    size_t psi_smem = 0, contract_smem = 0;
    bool profiling = false;
    bool have_events = false;
    cudaEvent_t ev[5];
    std::vector<gint::BatchRange> batches;   // regions that share the psi scratch, one after the other
    std::vector<int32_t> tg0;                // gint_fvl: first T-kernel task of each batch (+ end)
    gint::FvlPlan fvl{};           // built at the first gint_fvl call
    bool have_fvl = false;
    size_t force_smem = 0;
    gint::SnapPlan snap{};         // gint_snap_setup
    bool have_snap = false;
    int snap_fr = 2, snap_fc = 2;
    std::vector<void*> snap_allocs;
    std::vector<int32_t> snap_iat, snap_jat, snap_R;
    std::vector<int64_t> snap_off;
    double* V_scratch = nullptr;   // gint_vlocal_host only
    double* H_scratch = nullptr;
};

namespace {

thread_local std::string g_last_error;

int fail(int code, const std::string& msg) {
    g_last_error = msg;
    return code;
}
int fail_cuda(cudaError_t e, const char* where) {
    g_last_error = std::string(where) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? GINT_ENOMEM : GINT_ECUDA;
}

// Every device entry point runs on the context's device, whatever device is current in the calling thread, and
// leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
    }
    ~DeviceGuard() {
        int now = -1;
        if (prev >= 0 && cudaGetDevice(&now) == cudaSuccess && now != prev) cudaSetDevice(prev);
    }
};

template <typename T>
cudaError_t upload(gint_ctx* ctx, const std::vector<T>& host, const T** dev_out) {
    void* p = nullptr;
    const size_t bytes = host.size() * sizeof(T);
    cudaError_t e = cudaMalloc(&p, bytes ? bytes : 16);
    if (e != cudaSuccess) return e;
    ctx->allocs.push_back(p);
    if (bytes) e = cudaMemcpy(p, host.data(), bytes, cudaMemcpyHostToDevice);
    *dev_out = reinterpret_cast<const T*>(p);
    return e;
}

void release(gint_ctx* ctx) {
    if (ctx->device >= 0) {
        DeviceGuard guard(ctx->device);
        for (void* p : ctx->allocs) cudaFree(p);
        for (void* p : ctx->snap_allocs) cudaFree(p);
        if (ctx->have_events)
            for (int i = 0; i < 5; i++) cudaEventDestroy(ctx->ev[i]);
        if (ctx->V_scratch) cudaFree(ctx->V_scratch);
        if (ctx->H_scratch) cudaFree(ctx->H_scratch);
    }
    delete ctx;
}

// Device side of a context: upload the plan, allocate the scratch buffers, build the grid overlap S.  On failure the
// caller releases the context (everything allocated so far is in ctx->allocs).
int device_init(gint_ctx* ctx) {
    const int natom = (int)ctx->plan.atom_species.size();
    DeviceGuard guard(ctx->device);
    cudaError_t e = guard.err;
    if (e != cudaSuccess) return fail_cuda(e, "cudaSetDevice");
    const int cuda_device = ctx->device;
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, cuda_device);
    if (e != cudaSuccess) { return fail_cuda(e, "cudaGetDeviceProperties"); }
    ctx->nsm = prop.multiProcessorCount;
    if (ctx->plan.smem_bytes > (size_t)prop.sharedMemPerBlockOptin) {
        return fail(GINT_EUNSUPPORTED, "device offers too little shared memory per block");
    }
    gint::Plan& P = ctx->plan;
    gint::DevicePlan& D = ctx->dev;
#define UP(vec, ptr)                                                   \
    if ((e = upload(ctx, vec, ptr)) != cudaSuccess) {                  \
        return fail_cuda(e, "upload " #vec);                           \
    }
    UP(P.descs, &D.descs)
    UP(P.regions, &D.regions)
    UP(P.entries, &D.entries)
    UP(P.etasks, &D.etasks)
    UP(P.pair, &D.pair)
    UP(P.pair_direct, &D.pair_direct)
    UP(P.gmask, &D.gmask)
    UP(P.slot_xyz, &D.slot_xyz)
    UP(P.mirror, &D.mirror)
    UP(P.tab_packed, &D.tab)
    UP(P.sp_meta, &D.sp_meta)
    UP(P.sp_real, &D.sp_real)
    {   // block table for gint_fold_k
        std::vector<int32_t> run_start, first32(ctx->first_orb.begin(), ctx->first_orb.end());
        for (size_t b = 0; b < P.blk_i.size(); b++)
            if (b == 0 || P.blk_i[b] != P.blk_i[b - 1] || P.blk_j[b] != P.blk_j[b - 1]) run_start.push_back((int32_t)b);
        ctx->fold.nrun = (int32_t)run_start.size();
        run_start.push_back((int32_t)P.blk_i.size());
        ctx->fold.norb_tot = (int32_t)ctx->first_orb.back();
        UP(P.blk_i, &ctx->fold.blk_i)
        UP(P.blk_j, &ctx->fold.blk_j)
        UP(P.blk_R, &ctx->fold.blk_R)
        UP(P.blk_off, &ctx->fold.blk_off)
        UP(run_start, &ctx->fold.run_start)
        UP(first32, &ctx->fold.first)
        std::vector<int32_t> row_run0((size_t)natom + 1, 0), col_atom;
        for (int r = 0; r < ctx->fold.nrun; r++) row_run0[(size_t)P.blk_i[(size_t)run_start[(size_t)r]] + 1]++;
        for (int a = 0; a < natom; a++) {
            row_run0[(size_t)a + 1] += row_run0[(size_t)a];
            col_atom.insert(col_atom.end(), (size_t)(first32[(size_t)a + 1] - first32[(size_t)a]), a);
        }
        UP(row_run0, &ctx->fold.row_run0)
        UP(col_atom, &ctx->fold.col_atom)
        void* ph = nullptr;
        if ((e = cudaMalloc(&ph, (P.blk_i.size() + 1) * sizeof(double2))) != cudaSuccess) return fail_cuda(e, "cudaMalloc fold phases");
        ctx->allocs.push_back(ph);
        ctx->fold.phase = reinterpret_cast<double2*>(ph);
        ctx->fold.nblk = (int32_t)P.blk_i.size();
        ctx->fold.natom = natom;
        if ((e = gint::fold_static_scratch(ctx->device, &ctx->fold_static_phase)) != cudaSuccess)
            return fail_cuda(e, "cudaGetSymbolAddress fold phases");
    }
#undef UP
    void* ctr = nullptr;   // work-queue head, shift of the potential, partial (min, max) of V
    if ((e = cudaMalloc(&ctr, 128 + 2 * 512 * sizeof(double))) != cudaSuccess) { return fail_cuda(e, "cudaMalloc counter"); }
    ctx->allocs.push_back(ctr);
    D.counter = reinterpret_cast<unsigned int*>(ctr);
    D.shift = reinterpret_cast<gint::ShiftDev*>(reinterpret_cast<unsigned char*>(ctr) + 64);
    D.vpart = reinterpret_cast<double*>(reinterpret_cast<unsigned char*>(ctr) + 128);
    {
        std::vector<int32_t> work;
        for (size_t r = 0; r < P.regions.size(); r++)
            if (P.regions[r].ntile > 0) work.push_back((int32_t)r);
        D.nwork_regions = (int32_t)work.size();
        if ((e = upload(ctx, work, &D.work_regions)) != cudaSuccess) { return fail_cuda(e, "upload work_regions"); }
    }
    // psi scratch: zero-filled once; rows and slices that no evaluation task writes stay zero for good
    void* psi = nullptr;
    const size_t psi_bytes = (size_t)P.psi_chunks * gint::kChunkBytes;
    if ((e = cudaMalloc(&psi, psi_bytes ? psi_bytes : 16)) != cudaSuccess) { return fail_cuda(e, "cudaMalloc psi scratch"); }
    ctx->allocs.push_back(psi);
    if (psi_bytes && (e = cudaMemset(psi, 0, psi_bytes)) != cudaSuccess) { return fail_cuda(e, "cudaMemset psi scratch"); }
    D.psi = reinterpret_cast<double*>(psi);
    std::memcpy(D.estep, P.estep, sizeof(D.estep));
    D.dV = P.dV;
    for (int d = 0; d < 3; d++) D.ngrid[d] = P.ngrid[d];
    D.nks_pad = P.nks_pad;
    D.nslice = P.nslice;
    D.nstage = P.nstage;
    D.nregions = (int32_t)P.regions.size();
    D.nring = P.nring;
    D.multibatch = P.batches.size() > 1 ? 1 : 0;
    ctx->batches.clear();
    for (const gint::Plan::Batch& B : P.batches) ctx->batches.push_back(gint::BatchRange{B.item0, B.nitems, B.wr0, B.nwr});
    D.never = 0;
    D.nitems = (int32_t)P.descs.size();
    D.nmirror = (int32_t)P.mirror.size();
    D.tab_doubles = (int32_t)P.tab_packed.size();
    D.nspecies = (int32_t)P.species.size();
    ctx->psi_smem = gint::psi_kernel_smem(P.tables_in_smem ? P.tab_packed.size() * sizeof(double) : 0, (int)P.species.size());
    ctx->contract_smem = gint::contract_kernel_smem(P.nring);
    if ((e = gint::configure_kernels(ctx->psi_smem, ctx->contract_smem, P.tables_in_smem)) != cudaSuccess) {
        return fail_cuda(e, "cudaFuncSetAttribute");
    }
    {   // S = grid overlap blocks (Eq. 45 with V = 1): the per-call shift of the potential needs them (gint_hinit_kernel)
        const size_t nH = (size_t)P.blk_off.back(), nV = (size_t)P.ngrid[0] * P.ngrid[1] * P.ngrid[2];
        void *Sd = nullptr, *ones = nullptr;
        if ((e = cudaMalloc(&Sd, (nH ? nH : 1) * sizeof(double))) != cudaSuccess) { return fail_cuda(e, "cudaMalloc S"); }
        ctx->allocs.push_back(Sd);
        D.S = reinterpret_cast<const double*>(Sd);
        if ((e = cudaMalloc(&ones, nV * sizeof(double))) != cudaSuccess) { return fail_cuda(e, "cudaMalloc V=1"); }
        std::vector<double> one(nV, 1.0);
        e = cudaMemcpy(ones, one.data(), nV * sizeof(double), cudaMemcpyHostToDevice);
        if (e == cudaSuccess)
            e = gint::launch_vlocal(D, ctx->psi_smem, ctx->contract_smem, P.tables_in_smem, ctx->nsm, ctx->batches.data(),
                                    (int)ctx->batches.size(), nH, reinterpret_cast<const double*>(ones),
                                    reinterpret_cast<double*>(Sd), true, nullptr, nullptr);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        cudaFree(ones);
        if (e != cudaSuccess) { return fail_cuda(e, "grid overlap S"); }
    }
    return GINT_OK;
}

// frees what device_init allocated (the context keeps its events and host-call scratch)
void device_release_arrays(gint_ctx* ctx) {
    DeviceGuard guard(ctx->device);
    for (void* p : ctx->allocs) cudaFree(p);
    ctx->allocs.clear();
    ctx->have_fvl = false;
    ctx->fvl = gint::FvlPlan{};
    ctx->fold = gint::FoldPlan{};
    ctx->dev = gint::DevicePlan{};
    if (ctx->H_scratch) { cudaFree(ctx->H_scratch); ctx->H_scratch = nullptr; }
}

void snap_release(gint_ctx* ctx) {
    if (ctx->device >= 0 && !ctx->snap_allocs.empty()) {
        DeviceGuard guard(ctx->device);
        cudaDeviceSynchronize();   // a gint_snap_psibeta in flight still reads these tables
        for (void* p : ctx->snap_allocs) cudaFree(p);
    }
    ctx->snap_allocs.clear();
    ctx->snap = gint::SnapPlan{};
    ctx->have_snap = false;
    ctx->snap_iat.clear(); ctx->snap_jat.clear(); ctx->snap_R.clear(); ctx->snap_off.clear();
}

template <typename T>
cudaError_t snap_upload(gint_ctx* ctx, const std::vector<T>& host, const T** dev_out) {
    void* p = nullptr;
    const size_t bytes = host.size() * sizeof(T);
    cudaError_t e = cudaMalloc(&p, bytes ? bytes : 16);
    if (e != cudaSuccess) return e;
    ctx->snap_allocs.push_back(p);
    if (bytes) e = cudaMemcpy(p, host.data(), bytes, cudaMemcpyHostToDevice);
    *dev_out = reinterpret_cast<const T*>(p);
    return e;
}

}  // namespace

extern "C" {

int gint_setup(gint_ctx** out, const double* lattice, const int32_t* ngrid, int32_t nspecies,
               const gint_species* species, int32_t natom, const int32_t* atom_species, const double* atom_pos,
               int32_t cuda_device, const gint_options* opt) {
    if (!out) return fail(GINT_EINVAL, "out is null");
    *out = nullptr;
    if (!species || nspecies <= 0) return fail(GINT_EINVAL, "no species");
    gint_ctx* ctx = new (std::nothrow) gint_ctx;
    if (!ctx) return fail(GINT_ENOMEM, "host allocation failed");
    try {
        std::vector<gint::SpeciesHost> sp((size_t)nspecies);
        for (int s = 0; s < nspecies; s++) {
            const gint_species& in = species[s];
            if (!in.l || !in.table || in.nrad <= 0 || in.ntab <= 0 || in.nrad > 64) {
                delete ctx;
                return fail(GINT_EINVAL, "bad species descriptor");
            }
            sp[s].rcut = in.rcut;
            sp[s].dr = in.dr;
            sp[s].ntab = in.ntab;
            sp[s].nrad = in.nrad;
            sp[s].l.assign(in.l, in.l + in.nrad);
            sp[s].table.assign(in.table, in.table + (size_t)in.nrad * in.ntab);
        }
        std::string err;
        const int32_t* bc = opt ? opt->bcell : nullptr;
        const int rc = gint::build_plan(ctx->plan, lattice, ngrid, nspecies, sp.data(), natom, atom_species, atom_pos,
                                        bc, opt ? opt->rank : 0, opt ? opt->nranks : 1, opt ? opt->scratch_max_bytes : 0, err);
        if (rc != GINT_OK) {
            delete ctx;
            return fail(rc, err);
        }
    } catch (const std::bad_alloc&) {
        delete ctx;
        return fail(GINT_ENOMEM, "host allocation failed");
    }
    {
        const gint::Plan& PP = ctx->plan;
        ctx->first_orb.assign(1, 0);
        for (int a = 0; a < natom; a++) ctx->first_orb.push_back(ctx->first_orb.back() + PP.species[PP.atom_species[a]].norb);
    }
    if (cuda_device < 0) {   // host-only context
        *out = ctx;
        return GINT_OK;
    }
    ctx->device = cuda_device;
    const int rc = device_init(ctx);
    if (rc != GINT_OK) {
        release(ctx);
        return rc;
    }
    *out = ctx;
    return GINT_OK;
}

int gint_update_positions(gint_ctx* ctx, const double* atom_pos) {
    if (!ctx || !atom_pos) return fail(GINT_EINVAL, "null argument");
    const gint::Plan& old = ctx->plan;
    const int natom = (int)old.atom_species.size();
    gint_ctx* fresh = new (std::nothrow) gint_ctx;
    if (!fresh) return fail(GINT_ENOMEM, "host allocation failed");
    try {
        std::string err;
        std::vector<int32_t> asp(old.atom_species.begin(), old.atom_species.end());
        const int32_t ng[3] = {old.ngrid[0], old.ngrid[1], old.ngrid[2]};
        const int32_t bc[3] = {old.bcell[0], old.bcell[1], old.bcell[2]};
        const int rc = gint::build_plan(fresh->plan, old.lattice, ng, (int)old.species.size(), old.species.data(), natom,
                                        asp.data(), atom_pos, bc, old.rank, old.nranks, old.scratch_max_bytes, err);
        if (rc != GINT_OK) {
            delete fresh;
            return fail(rc, err);   // the context is unchanged
        }
    } catch (const std::bad_alloc&) {
        delete fresh;
        return fail(GINT_ENOMEM, "host allocation failed");
    }
    std::swap(ctx->plan, fresh->plan);
    delete fresh;
    if (ctx->device < 0) return GINT_OK;
    {
        DeviceGuard guard(ctx->device);
        if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
        cudaDeviceSynchronize();   // calls in flight still read the old tables
    }
    device_release_arrays(ctx);
    snap_release(ctx);   // pair list of the old geometry: gint_snap_setup has to be called again
    return device_init(ctx);
}

int gint_num_blocks(const gint_ctx* ctx, int64_t* nblocks, int64_t* h_len) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    if (nblocks) *nblocks = (int64_t)ctx->plan.blk_i.size();
    if (h_len) *h_len = ctx->plan.blk_off.back();
    return GINT_OK;
}

int gint_get_blocks(const gint_ctx* ctx, int32_t* iat, int32_t* jat, int32_t* R, int64_t* offset) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    const gint::Plan& P = ctx->plan;
    const size_t n = P.blk_i.size();
    if (iat && n) std::memcpy(iat, P.blk_i.data(), n * sizeof(int32_t));
    if (jat && n) std::memcpy(jat, P.blk_j.data(), n * sizeof(int32_t));
    if (R && n) std::memcpy(R, P.blk_R.data(), 3 * n * sizeof(int32_t));
    if (offset) std::memcpy(offset, P.blk_off.data(), (n + 1) * sizeof(int64_t));
    return GINT_OK;
}

int gint_vlocal(gint_ctx* ctx, const double* V_dev, double* H_dev, void* stream) {
    if (!ctx || !V_dev || !H_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaError_t e = gint::launch_vlocal(ctx->dev, ctx->psi_smem, ctx->contract_smem, ctx->plan.tables_in_smem, ctx->nsm,
                                        ctx->batches.data(), (int)ctx->batches.size(), (size_t)ctx->plan.blk_off.back(),
                                        V_dev, H_dev, false,
                                        reinterpret_cast<cudaStream_t>(stream), ctx->profiling ? ctx->ev : nullptr);
    if (e != cudaSuccess) return fail_cuda(e, "gint_vlocal launch");
    return GINT_OK;
}

int gint_rho(gint_ctx* ctx, const double* D_dev, double* rho_dev, void* stream) {
    if (!ctx || !D_dev || !rho_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    cudaError_t e = gint::launch_rho(ctx->dev, ctx->psi_smem, ctx->contract_smem, ctx->plan.tables_in_smem, ctx->nsm,
                                     ctx->batches.data(), (int)ctx->batches.size(), D_dev, rho_dev, st);
    if (e != cudaSuccess) return fail_cuda(e, "gint_rho launch");
    return GINT_OK;
}

// scratch buffers and tables of gint_fvl, allocated when it is first called (E: 8 (32 ngroup)^2 bytes per region,
// T: as large as the psi scratch)
static int fvl_init(gint_ctx* ctx) {
    const gint::Plan& P = ctx->plan;
    gint::FvlPlan& F = ctx->fvl;
    std::vector<int64_t> e0(P.regions.size(), 0);
    std::vector<int4> tasks;
    int64_t echunks = 0, ecur = 0;   // E scratch: as large as its largest batch needs
    ctx->tg0.assign(1, 0);
    for (size_t r = 0; r < P.regions.size(); r++) {
        const gint::Region& R = P.regions[r];
        if (r > 0 && P.region_batch[r] != P.region_batch[r - 1]) {
            ecur = 0;
            ctx->tg0.push_back((int32_t)tasks.size());
        }
        if (R.ntile <= 0) continue;
        e0[r] = ecur;
        ecur += (int64_t)R.ngroup * R.ngroup;
        echunks = std::max(echunks, ecur);
        for (int rq = 0; rq * 4 < R.ngroup; rq++)
            for (int sq = 0; sq * 4 < P.nstage; sq++) tasks.push_back(make_int4((int)r, rq, sq, 0));
    }
    while (ctx->tg0.size() < P.batches.size() + 1) ctx->tg0.push_back((int32_t)tasks.size());
    cudaError_t e;
    F.gmask = ctx->dev.gmask;
    if ((e = upload(ctx, P.rowinfo, &F.rowinfo)) != cudaSuccess) return fail_cuda(e, "upload rowinfo");
    if ((e = upload(ctx, e0, &F.e_chunk0)) != cudaSuccess) return fail_cuda(e, "upload e_chunk0");
    if ((e = upload(ctx, tasks, &F.tg_tasks)) != cudaSuccess) return fail_cuda(e, "upload tgemm tasks");
    void *es = nullptr, *ts = nullptr;
    if ((e = cudaMalloc(&es, echunks ? (size_t)echunks * gint::kChunkBytes : 16)) != cudaSuccess) return fail_cuda(e, "cudaMalloc E scratch");
    ctx->allocs.push_back(es);
    if ((e = cudaMalloc(&ts, P.psi_chunks ? (size_t)P.psi_chunks * gint::kChunkBytes : 16)) != cudaSuccess) return fail_cuda(e, "cudaMalloc T scratch");
    ctx->allocs.push_back(ts);
    F.escratch = reinterpret_cast<double*>(es);
    F.tscratch = reinterpret_cast<double*>(ts);
    F.ntg = (int32_t)tasks.size();
    F.nks_pad = P.nks_pad;
    ctx->force_smem = gint::force_kernel_smem(P.tables_in_smem ? P.tab_packed.size() * sizeof(double) : 0, (int)P.species.size());
    if ((e = gint::configure_fvl(ctx->force_smem, P.tables_in_smem)) != cudaSuccess) return fail_cuda(e, "cudaFuncSetAttribute (fvl)");
    ctx->have_fvl = true;
    return GINT_OK;
}

int gint_fvl(gint_ctx* ctx, const double* V_dev, const double* D_dev, double* F_dev, void* stream) {
    if (!ctx || !V_dev || !D_dev || !F_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    if (!ctx->have_fvl) {
        const int rc = fvl_init(ctx);
        if (rc != GINT_OK) return rc;
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    cudaError_t e = gint::launch_fvl(ctx->dev, ctx->fvl, ctx->psi_smem, ctx->force_smem, ctx->plan.tables_in_smem, ctx->nsm,
                                     (int)ctx->plan.atom_species.size(), ctx->batches.data(), ctx->tg0.data(),
                                     (int)ctx->batches.size(), V_dev, D_dev, F_dev, st);
    if (e != cudaSuccess) return fail_cuda(e, "gint_fvl launch");
    return GINT_OK;
}

int gint_num_orbitals(const gint_ctx* ctx, int64_t* norb_tot, int64_t* first) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    if (norb_tot) *norb_tot = ctx->first_orb.back();
    if (first) std::memcpy(first, ctx->first_orb.data(), ctx->first_orb.size() * sizeof(int64_t));
    return GINT_OK;
}

int gint_fold_k(gint_ctx* ctx, const double* H_dev, const double* kfrac, double* Hk_dev, void* stream) {
    if (!ctx || !H_dev || !kfrac || !Hk_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaError_t e = gint::launch_fold(ctx->fold, H_dev, kfrac, Hk_dev, reinterpret_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "gint_fold_k launch");
    return GINT_OK;
}

int64_t gint_fold_k_static_max_blocks(void) { return gint::kFoldStaticMaxBlocks; }

int gint_fold_k_static(gint_ctx* ctx, const double* H_dev, const double* kfrac, double* Hk_dev, void* stream) {
    if (!ctx || !H_dev || !kfrac || !Hk_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    if (ctx->fold.nblk > gint::kFoldStaticMaxBlocks)
        return fail(GINT_EUNSUPPORTED, "gint_fold_k_static: " + std::to_string(ctx->fold.nblk) + " blocks exceed the fixed scratch of " +
                                           std::to_string(gint::kFoldStaticMaxBlocks) + " blocks; use gint_fold_k");
    if (!ctx->fold_static_phase) return fail(GINT_ECUDA, "gint_fold_k_static: the fixed scratch was not resolved at set-up");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaError_t e = gint::launch_fold_static(ctx->fold, ctx->fold_static_phase, H_dev, kfrac, Hk_dev,
                                             reinterpret_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "gint_fold_k_static launch");
    return GINT_OK;
}

int gint_snap_setup(gint_ctx* ctx, const gint_species* proj, int32_t nrad_pts, const double* rad_x, const double* rad_w,
                    int32_t nang, const double* ang_xyz, const double* ang_w) {
    if (!ctx || !proj || !rad_x || !rad_w || !ang_xyz || !ang_w) return fail(GINT_EINVAL, "null argument");
    if (nrad_pts <= 0 || nang <= 0) return fail(GINT_EINVAL, "empty quadrature table");
    const gint::Plan& P = ctx->plan;
    const int nsp = (int)P.species.size(), natom = (int)P.atom_species.size();
    try {
        std::vector<gint::SnapSpecies> orb((size_t)nsp), prj((size_t)nsp);
        std::vector<double> tab;
        int max_n = 0, max_m = 0;
        for (int s = 0; s < nsp; s++) {
            const gint::SpeciesHost& h = P.species[(size_t)s];
            gint::SnapSpecies& o = orb[(size_t)s];
            std::memset(&o, 0, sizeof(o));
            o.tab_off = (int32_t)tab.size(); o.ntab = h.ntab; o.nrad = h.nrad; o.ncomp = h.norb;
            for (int f = 0; f < h.nrad; f++) o.l[f] = h.l[(size_t)f];
            o.rcut = h.rcut; o.inv_dr = 1.0 / h.dr;
            tab.insert(tab.end(), h.table.begin(), h.table.end());
            max_n = std::max(max_n, h.norb);
            const gint_species& q = proj[s];
            gint::SnapSpecies& b = prj[(size_t)s];
            std::memset(&b, 0, sizeof(b));
            if (q.nrad < 0 || q.nrad > 8) return fail(GINT_EUNSUPPORTED, "more than 8 projector radial functions per species");
            if (q.nrad == 0) continue;   // this species hosts no projectors
            if (!q.l || !q.table || !(q.rcut > 0) || !(q.dr > 0)) return fail(GINT_EINVAL, "bad projector species");
            if ((double)q.ntab * q.dr < q.rcut + 3.0 * q.dr - 1e-9) return fail(GINT_EINVAL, "projector table too short for rcut + 3 dr");
            b.tab_off = (int32_t)tab.size(); b.ntab = q.ntab; b.nrad = q.nrad;
            for (int f = 0; f < q.nrad; f++) {
                if (q.l[f] < 0 || q.l[f] > 3) return fail(GINT_EUNSUPPORTED, "projector l > 3");
                b.l[f] = q.l[f];
                b.ncomp += 2 * q.l[f] + 1;
            }
            b.rcut = q.rcut; b.inv_dr = 1.0 / q.dr;
            tab.insert(tab.end(), q.table, q.table + (size_t)q.nrad * q.ntab);
            max_m = std::max(max_m, b.ncomp);
        }
        if (max_n > 32) return fail(GINT_EUNSUPPORTED, "gint_snap: more than 32 orbitals per atom");
        if (max_m > 16) return fail(GINT_EUNSUPPORTED, "gint_snap: more than 16 projector components per atom");
        // pair list: every (I, J, R) with |tau_J + R - tau_I| < rb_I + rc_J, in (I, J, R1, R2, R3) order
        const double* a = P.lattice;
        const double c0[3] = {a[4] * a[8] - a[5] * a[7], a[5] * a[6] - a[3] * a[8], a[3] * a[7] - a[4] * a[6]};   // a2 x a3
        const double c1[3] = {a[7] * a[2] - a[8] * a[1], a[8] * a[0] - a[6] * a[2], a[6] * a[1] - a[7] * a[0]};   // a3 x a1
        const double c2[3] = {a[1] * a[5] - a[2] * a[4], a[2] * a[3] - a[0] * a[5], a[0] * a[4] - a[1] * a[3]};   // a1 x a2
        const double vol = a[0] * c0[0] + a[1] * c0[1] + a[2] * c0[2];
        const double* cr[3] = {c0, c1, c2};
        double height[3];
        for (int k = 0; k < 3; k++) height[k] = std::fabs(vol) / std::sqrt(cr[k][0] * cr[k][0] + cr[k][1] * cr[k][1] + cr[k][2] * cr[k][2]);
        std::vector<gint::SnapPair> pairs;
        snap_release(ctx);
        int64_t off = 0;
        for (int I = 0; I < natom; I++) {
            const gint::SnapSpecies& b = prj[(size_t)P.atom_species[(size_t)I]];
            if (b.nrad == 0) continue;
            if (P.nranks > 1 && I % P.nranks != P.rank) continue;   // sharded context: projector atoms dealt out by index
            const double* tI = &P.atom_pos[3 * (size_t)I];
            for (int J = 0; J < natom; J++) {
                const gint::SnapSpecies& o = orb[(size_t)P.atom_species[(size_t)J]];
                const double* tJ = &P.atom_pos[3 * (size_t)J];
                const double cut = b.rcut + o.rcut;
                const double dx = tJ[0] - tI[0], dy = tJ[1] - tI[1], dz = tJ[2] - tI[2];
                int lo[3], hi[3];
                for (int k = 0; k < 3; k++) {   // fractional coordinate of tau_J - tau_I along a_k, plus the reach of the cutoff
                    const double f = (dx * cr[k][0] + dy * cr[k][1] + dz * cr[k][2]) / vol;
                    lo[k] = (int)std::floor(-f - cut / height[k]) - 1;
                    hi[k] = (int)std::ceil(-f + cut / height[k]) + 1;
                }
                for (int r1 = lo[0]; r1 <= hi[0]; r1++)
                    for (int r2 = lo[1]; r2 <= hi[1]; r2++)
                        for (int r3 = lo[2]; r3 <= hi[2]; r3++) {
                            const double ex = dx + r1 * a[0] + r2 * a[3] + r3 * a[6];
                            const double ey = dy + r1 * a[1] + r2 * a[4] + r3 * a[7];
                            const double ez = dz + r1 * a[2] + r2 * a[5] + r3 * a[8];
                            if (!(ex * ex + ey * ey + ez * ez < cut * cut)) continue;
                            gint::SnapPair pr;
                            pr.d[0] = -ex; pr.d[1] = -ey; pr.d[2] = -ez;
                            pr.tauI[0] = tI[0]; pr.tauI[1] = tI[1]; pr.tauI[2] = tI[2];
                            pr.off = off;
                            pr.spI = P.atom_species[(size_t)I]; pr.spJ = P.atom_species[(size_t)J];
                            pairs.push_back(pr);
                            ctx->snap_iat.push_back(I); ctx->snap_jat.push_back(J);
                            ctx->snap_R.push_back(r1); ctx->snap_R.push_back(r2); ctx->snap_R.push_back(r3);
                            ctx->snap_off.push_back(off);
                            off += (int64_t)o.ncomp * b.ncomp;
                        }
            }
        }
        ctx->snap_off.push_back(off);
        if (pairs.size() > 0x7FFFFFFFull) return fail(GINT_EUNSUPPORTED, "gint_snap: too many pairs");
        ctx->snap_fr = std::max(1, (std::max(max_n, max_m) + 7) / 8);   // projector values pass through the orbital columns
        ctx->snap_fc = std::max(1, (2 * max_m + 7) / 8);
        if (ctx->device < 0) {   // host-only context: the pair list can be queried, gint_snap_psibeta returns GINT_ENODEVICE
            ctx->have_snap = true;
            return GINT_OK;
        }
        DeviceGuard guard(ctx->device);
        if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
        cudaError_t e;
        gint::SnapPlan& S = ctx->snap;
        const std::vector<double> rx(rad_x, rad_x + nrad_pts), rw(rad_w, rad_w + nrad_pts), an(ang_xyz, ang_xyz + 3 * (size_t)nang),
            aw(ang_w, ang_w + nang);
        if ((e = snap_upload(ctx, orb, &S.orb)) != cudaSuccess || (e = snap_upload(ctx, prj, &S.proj)) != cudaSuccess ||
            (e = snap_upload(ctx, tab, &S.tab)) != cudaSuccess || (e = snap_upload(ctx, pairs, &S.pairs)) != cudaSuccess ||
            (e = snap_upload(ctx, rx, &S.rad_x)) != cudaSuccess || (e = snap_upload(ctx, rw, &S.rad_w)) != cudaSuccess ||
            (e = snap_upload(ctx, an, &S.ang_xyz)) != cudaSuccess || (e = snap_upload(ctx, aw, &S.ang_w)) != cudaSuccess) {
            snap_release(ctx);
            return fail_cuda(e, "gint_snap_setup upload");
        }
        std::vector<int32_t> groups;   // consecutive pairs of one projector atom share a CTA
        for (size_t b0 = 0; b0 < pairs.size();) {
            size_t n = 1;
            while (n < (size_t)gint::kSnapGroupPairs && b0 + n < pairs.size() && ctx->snap_iat[b0 + n] == ctx->snap_iat[b0]) n++;
            groups.push_back((int32_t)b0);
            groups.push_back((int32_t)n);
            b0 += n;
        }
        if ((e = snap_upload(ctx, groups, &S.groups)) != cudaSuccess) {
            snap_release(ctx);
            return fail_cuda(e, "gint_snap_setup upload");
        }
        S.ngroup = (int32_t)(groups.size() / 2);
        S.npair = (int32_t)pairs.size(); S.nrad = nrad_pts; S.nang = nang;
        ctx->have_snap = true;
    } catch (const std::bad_alloc&) {
        snap_release(ctx);
        return fail(GINT_ENOMEM, "host allocation failed");
    }
    return GINT_OK;
}

int gint_snap_num_pairs(const gint_ctx* ctx, int64_t* npair, int64_t* s_len) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    if (!ctx->have_snap) return fail(GINT_EINVAL, "gint_snap_setup has not been called (or the positions changed since)");
    if (npair) *npair = (int64_t)ctx->snap_iat.size();
    if (s_len) *s_len = ctx->snap_off.back();
    return GINT_OK;
}

int gint_snap_get_pairs(const gint_ctx* ctx, int32_t* iat, int32_t* jat, int32_t* R, int64_t* offset) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    if (!ctx->have_snap) return fail(GINT_EINVAL, "gint_snap_setup has not been called (or the positions changed since)");
    const size_t n = ctx->snap_iat.size();
    if (iat && n) std::memcpy(iat, ctx->snap_iat.data(), n * sizeof(int32_t));
    if (jat && n) std::memcpy(jat, ctx->snap_jat.data(), n * sizeof(int32_t));
    if (R && n) std::memcpy(R, ctx->snap_R.data(), 3 * n * sizeof(int32_t));
    if (offset) std::memcpy(offset, ctx->snap_off.data(), (n + 1) * sizeof(int64_t));
    return GINT_OK;
}

int gint_snap_psibeta(gint_ctx* ctx, const double* A, double* S_dev, void* stream) {
    if (!ctx || !A || !S_dev) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    if (!ctx->have_snap) return fail(GINT_EINVAL, "gint_snap_setup has not been called (or the positions changed since)");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaError_t e = gint::launch_snap(ctx->snap, ctx->snap_fr, ctx->snap_fc, A, S_dev, reinterpret_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "gint_snap_psibeta launch");
    return GINT_OK;
}

int gint_vlocal_host(gint_ctx* ctx, const double* V_host, double* H_host) {
    if (!ctx || !V_host || !H_host) return fail(GINT_EINVAL, "null argument");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    cudaError_t e = guard.err;
    if (e != cudaSuccess) return fail_cuda(e, "cudaSetDevice");
    const size_t nV = (size_t)ctx->plan.ngrid[0] * ctx->plan.ngrid[1] * ctx->plan.ngrid[2];
    const size_t nH = (size_t)ctx->plan.blk_off.back();
    if (!ctx->V_scratch && (e = cudaMalloc(&ctx->V_scratch, nV * sizeof(double))) != cudaSuccess)
        return fail_cuda(e, "cudaMalloc V");
    if (!ctx->H_scratch && (e = cudaMalloc(&ctx->H_scratch, (nH ? nH : 1) * sizeof(double))) != cudaSuccess)
        return fail_cuda(e, "cudaMalloc H");
    if ((e = cudaMemcpyAsync(ctx->V_scratch, V_host, nV * sizeof(double), cudaMemcpyHostToDevice, 0)) != cudaSuccess)
        return fail_cuda(e, "H2D V");
    const int rc = gint_vlocal(ctx, ctx->V_scratch, ctx->H_scratch, nullptr);
    if (rc != GINT_OK) return rc;
    if ((e = cudaMemcpyAsync(H_host, ctx->H_scratch, nH * sizeof(double), cudaMemcpyDeviceToHost, 0)) != cudaSuccess)
        return fail_cuda(e, "D2H H");
    if ((e = cudaStreamSynchronize(0)) != cudaSuccess) return fail_cuda(e, "synchronize");
    return GINT_OK;
}

int gint_set_profiling(gint_ctx* ctx, int32_t on) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    if (ctx->device < 0) return fail(GINT_ENODEVICE, "host-only context");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    if (on && !ctx->have_events) {
        for (int i = 0; i < 5; i++) {
            cudaError_t e = cudaEventCreate(&ctx->ev[i]);
            if (e != cudaSuccess) return fail_cuda(e, "cudaEventCreate");
        }
        ctx->have_events = true;
    }
    ctx->profiling = on != 0;
    return GINT_OK;
}

int gint_get_kernel_ms(gint_ctx* ctx, double* ms) {
    if (!ctx || !ms) return fail(GINT_EINVAL, "null argument");
    if (!ctx->profiling || !ctx->have_events) return fail(GINT_EINVAL, "profiling is off");
    DeviceGuard guard(ctx->device);
    if (guard.err != cudaSuccess) return fail_cuda(guard.err, "cudaSetDevice");
    cudaError_t e = cudaEventSynchronize(ctx->ev[4]);
    if (e != cudaSuccess) return fail_cuda(e, "cudaEventSynchronize");
    float a = 0, b = 0, c = 0, d = 0;
    cudaEventElapsedTime(&a, ctx->ev[2], ctx->ev[3]);
    cudaEventElapsedTime(&b, ctx->ev[3], ctx->ev[4]);
    cudaEventElapsedTime(&c, ctx->ev[0], ctx->ev[4]);
    cudaEventElapsedTime(&d, ctx->ev[1], ctx->ev[2]);
    ms[0] = a;
    ms[1] = b;
    ms[2] = c;
    ms[3] = d;
    return GINT_OK;
}

int gint_get_stats(const gint_ctx* ctx, double* stats, int32_t n) {
    if (!ctx || !stats) return fail(GINT_EINVAL, "null argument");
    const int m = n < 32 ? n : 32;
    for (int i = 0; i < m; i++) stats[i] = ctx->plan.stats[i];
    return m;
}

int gint_get_cell_lists(const gint_ctx* ctx, int64_t* ncell, int64_t* nentry, int64_t* cell_start,
                        int32_t* entry_atom, int32_t* entry_R) {
    if (!ctx) return fail(GINT_EINVAL, "ctx is null");
    const gint::Plan& P = ctx->plan;
    if (ncell) *ncell = (int64_t)P.cell_start.size() - 1;
    if (nentry) *nentry = (int64_t)P.cell_atom.size();
    if (cell_start) std::memcpy(cell_start, P.cell_start.data(), P.cell_start.size() * sizeof(int64_t));
    if (entry_atom && !P.cell_atom.empty()) std::memcpy(entry_atom, P.cell_atom.data(), P.cell_atom.size() * sizeof(int32_t));
    if (entry_R && !P.cell_R.empty()) std::memcpy(entry_R, P.cell_R.data(), P.cell_R.size() * sizeof(int32_t));
    return GINT_OK;
}

int gint_measure_fp64_peak(int32_t cuda_device, double seconds, double* tflops) {
    if (!tflops || cuda_device < 0) return fail(GINT_EINVAL, "bad argument");
    DeviceGuard guard(cuda_device);
    cudaError_t e = guard.err;
    if (e != cudaSuccess) return fail_cuda(e, "cudaSetDevice");
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, cuda_device)) != cudaSuccess) return fail_cuda(e, "cudaGetDeviceProperties");
    if ((e = gint::measure_dmma_peak(seconds, prop.multiProcessorCount, tflops)) != cudaSuccess)
        return fail_cuda(e, "dmma peak kernel");
    return GINT_OK;
}

int gint_destroy(gint_ctx* ctx) {
    if (!ctx) return GINT_OK;
    release(ctx);
    return GINT_OK;
}

const char* gint_strerror(int code) {
    switch (code) {
        case GINT_OK: return "ok";
        case GINT_EINVAL: return "invalid argument";
        case GINT_EUNSUPPORTED: return "unsupported input";
        case GINT_ENOMEM: return "out of memory";
        case GINT_ECUDA: return "CUDA error";
        case GINT_ENODEVICE: return "context has no device";
        default: return "unknown error";
    }
}

const char* gint_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
