#!/usr/bin/env python
"""bench.py -- gint_vlocal H build on the 512-atom Si-like DZP workload (BASELINE.json configs[3]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload si512_dzp] [--impl reference]

A "step" is one gint_vlocal call = the whole hot path (psi kernel: V staging, phi
evaluation, V*dV weighting; contraction kernel: DMMA contraction + accumulation into
H blocks; mirror kernel) over the whole mesh.  Prints ONE JSON line (rank 0).

  value            FP64 TFLOP/s = F_sym / time, F_sym = sum_g n(g)(n(g)+1) useful flops
                   (the kernel exploits H(R) = H(-R)^T), inputs resident in HBM
  ms_per_step      ms per gint_vlocal call (CUDA events, L2 flushed between calls)
  e2e              same metric through gint_vlocal_host: pinned HOST V in, HOST H out,
                   both copies inside the timed region
  roofline         the dominant kernel (gint_contract_kernel<0>, the contraction of gint_vlocal) alone: achieved
                   TFLOP/s (F_sym / its event-timed duration) over the FP64 tensor (DMMA.8x8x4)
                   peak measured live; the psi kernel's HBM figures ride along
  cpu_baseline     the CPU oracle, as it stands, on a bounded sample of the same workload

N > 1 (torchrun): the big cells are sharded over ranks (strided slabs along a1), every
rank integrates its share and the partial H buffers are summed with one NCCL
all-reduce -- the path's only exchange step; scaling is strong.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "gint_vlocal FP64 TFLOP/s (useful flops F_sym per H build; ms/call in ms_per_step, % of roofline in roofline.frac)"
UNIT = "TFLOP/s"



def ncu_traffic(workload):
    """DRAM traffic of the contraction kernel per launch (dram__bytes_read.sum + dram__bytes_write.sum of the latest
    ncu --set full capture), read from profiles/ncu_traffic.csv at run time; None if no capture is recorded."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        with open(p) as f:
            for line in f.read().splitlines()[1:]:
                cols = line.split(",")
                if cols[0] == workload:
                    return float(cols[2]) + float(cols[3])
    except (OSError, ValueError, IndexError):
        pass
    return None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def useful_flops(w):
    """F_pt = sum_g 2 n(g)^2 and F_sym = sum_g n(g)(n(g)+1), n(g) = orbitals non-zero at mesh point g (all atom
    images counted), counted here with a k-d tree over the atom images -- no library call, so
    that the oracle arm (--impl reference) runs with the product .so absent."""
    from scipy.spatial import cKDTree
    n1, n2, n3 = (int(x) for x in w.ngrid)
    f = np.stack(np.meshgrid(np.arange(n1) / n1, np.arange(n2) / n2, np.arange(n3) / n3, indexing="ij"), axis=-1)
    pts = f.reshape(-1, 3) @ w.lattice
    inv = np.linalg.inv(w.lattice)
    norb = np.zeros(pts.shape[0], dtype=np.int64)
    for s_id, sp in enumerate(w.species):
        atoms = w.atom_pos[np.asarray(w.atom_species) == s_id]
        if atoms.shape[0] == 0:
            continue
        reach = np.ceil(sp.rcut * np.linalg.norm(inv, axis=0)).astype(int) + 1      # images that can reach the cell
        fa = atoms @ inv
        lo, hi = np.floor(fa.min(0)).astype(int), np.floor(fa.max(0)).astype(int)
        sh = np.array([[a, b, c] for a in range(-hi[0] - reach[0], -lo[0] + reach[0] + 1)
                       for b in range(-hi[1] - reach[1], -lo[1] + reach[1] + 1)
                       for c in range(-hi[2] - reach[2], -lo[2] + reach[2] + 1)])
        img = (atoms[None, :, :] + (sh @ w.lattice)[:, None, :]).reshape(-1, 3)
        c = img @ inv                                                               # keep images near the cell only
        pad = sp.rcut * np.linalg.norm(inv, axis=0) + 1e-9
        img = img[np.all((c > -pad) & (c < 1.0 + pad), axis=1)]
        cnt = cKDTree(img).query_ball_point(pts, sp.rcut * (1.0 - 1e-15), return_length=True, workers=-1)
        norb += sp.norb * np.asarray(cnt, dtype=np.int64)
    nn = norb.astype(np.float64)
    return float(np.sum(2.0 * nn * nn)), float(np.sum(nn * (nn + 1.0)))


def oracle_sample(w, natoms_sample, nthreads=0):
    """Time the CPU oracle on all blocks of the first `natoms_sample` row atoms."""
    import oracle
    bi, bj, bR, off = oracle.enumerate_blocks(w.lattice, w.species, w.atom_species, w.atom_pos)
    sel = np.nonzero(bi < natoms_sample)[0]
    t = time.perf_counter()
    _, _, used = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V,
                               blocks=(bi[sel], bj[sel], bR[sel]), nthreads=nthreads, return_threads=True)
    return time.perf_counter() - t, int(used), len(sel), len(bi)


def run_reference(args, w, stats_fpt):
    """--impl reference: the oracle as it stands on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    frac_atoms = max(1, min(w.natom, args.ref_atoms or 32))
    times = []
    used = nblk = ntot = 0
    for i in range(args.warmup + args.steps):
        dt, used, nblk, ntot = oracle_sample(w, frac_atoms)
        if i >= args.warmup:
            times.append(dt)
    sec = float(np.mean(times))
    flops = stats_fpt * frac_atoms / w.natom      # the oracle computes both (I,J,R) and (J,I,-R): F_pt accounting
    val = flops / sec * 1e-12
    sample = "all %d blocks of the first %d of %d row atoms (%d of %d blocks), flops = F_pt*%d/%d" % (
        nblk, frac_atoms, w.natom, nblk, ntot, frac_atoms, w.natom)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "natom": w.natom, "norb": w.norb_total, "ngrid": [int(x) for x in w.ngrid],
                   "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample,
                         "ms_per_call_extrapolated": sec * 1e3 * w.natom / frac_atoms},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="si512_dzp")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-atoms", type=int, default=0,
                    help="row atoms in the oracle sample (default: 256 for the cpu_baseline leg, 32 per step for --impl reference)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from paper_2603_21835_b200 import workloads
    w = workloads.make(args.workload)

    if args.impl == "reference":
        # the oracle arm loads oracle/ and the seeded input generator only: no product library, no CUDA
        run_reference(args, w, useful_flops(w)[0])
        return

    import torch
    from paper_2603_21835_b200 import gint_setup, gint_measure_fp64_peak
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the gint_vlocal hot path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    t0 = time.perf_counter()
    ctx = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=local_rank,
                     rank=rank, nranks=world)
    setup_s = time.perf_counter() - t0
    st = ctx.gint_get_stats()
    # useful flops of the WHOLE job (all ranks): from an unsharded host-only plan when sharded
    if world > 1:
        st_all = gint_setup(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, cuda_device=-1).gint_get_stats()
    else:
        st_all = st
    F_sym, F_pt = st_all["F_sym"], st_all["F_pt"]

    V = torch.from_numpy(w.V).to(dev)
    H = torch.empty(ctx.h_len, dtype=torch.float64, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # 256 MB > 126 MB L2
    ctx.gint_set_profiling(True)

    def step():
        ctx.gint_vlocal(V, H)
        if world > 1:
            dist.all_reduce(H)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    peak_live = gint_measure_fp64_peak(local_rank, 0.3)

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (outside the event pair)
        ev[i][0].record()
        step()
        ev[i][1].record()
        kern_ms.append(ctx.gint_get_kernel_ms())     # syncs on this call's events
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(step_ms.sum())
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step = total_ms / args.steps
    value = F_sym / (ms_per_step * 1e-3) * 1e-12

    # ---- end to end through the C ABI with host buffers --------------------------------
    Vh = torch.from_numpy(w.V).pin_memory()
    Hh = torch.empty(ctx.h_len, dtype=torch.float64).pin_memory()
    Vh_np, Hh_np = Vh.numpy(), Hh.numpy()
    for _ in range(2):
        ctx.gint_vlocal_host(Vh_np, Hh_np)
    e2e_t = []
    nrep = max(3, min(args.steps, 10))
    for _ in range(nrep):
        flush.zero_()
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ctx.gint_vlocal_host(Vh_np, Hh_np)        # H2D V + kernels + D2H H + sync, all inside
        e2e_t.append(time.perf_counter() - t1)
    e2e_ms = float(np.mean(e2e_t)) * 1e3
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    # sharded: every rank's e2e call covers its share of the flops; whole job = F_sym per max time
    e2e_val = F_sym / (e2e_ms * 1e-3) * 1e-12

    # ---- next step of the workflow, outside the headline: H(k) = sum_R exp(i k.R) H(R) (Eq. 5) -------------
    fold = rho_info = fvl_info = snap_info = None
    if world == 1:
        ntot = ctx.gint_num_orbitals()[0]
        Hk = torch.empty((ntot, ntot), dtype=torch.complex128, device=dev)
        for _ in range(2):
            ctx.gint_fold_k(H, (0.25, 0.5, -0.125), Hk)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        f0.record()
        for _ in range(10):
            ctx.gint_fold_k(H, (0.25, 0.5, -0.125), Hk)
        f1.record()
        torch.cuda.synchronize()
        fold_ms = f0.elapsed_time(f1) / 10
        fold_bytes = 8.0 * ctx.h_len + 16.0 * ntot * ntot
        fold = {"ms_per_call": fold_ms, "algorithmic_bytes": fold_bytes, "achieved_gbs": fold_bytes / (fold_ms * 1e-3) * 1e-9,
                "norb_tot": ntot, "note": "gint_fold_k: H blocks read once, dense complex H(k) written once (single pass, zeros included)"}
        del Hk
        # charge density (Eq. 44), first cut
        Dm = torch.randn(ctx.h_len, dtype=torch.float64, device=dev)
        rho = ctx.gint_rho(Dm)
        torch.cuda.synchronize()
        f0.record()
        for _ in range(2):
            ctx.gint_rho(Dm, rho)
        f1.record()
        torch.cuda.synchronize()
        rho_ms = f0.elapsed_time(f1) / 2
        rho_info = {"ms_per_call": rho_ms, "useful_flops": F_sym, "achieved_tflops": F_sym / (rho_ms * 1e-3) * 1e-12,
                    "note": "gint_rho (Eq. 44) on the tensor pipe: tiles ga <= gb with E = D + D^T folded at gather time, "
                            "so F_sym accounting as for gint_vlocal; the time includes its psi kernel"}
        # local Pulay force (Eq. 46)
        Fv = ctx.gint_fvl(V, Dm)
        torch.cuda.synchronize()
        f0.record()
        for _ in range(2):
            ctx.gint_fvl(V, Dm, Fv)
        f1.record()
        torch.cuda.synchronize()
        fvl_ms = f0.elapsed_time(f1) / 2
        fvl_info = {"ms_per_call": fvl_ms, "useful_flops": F_pt, "achieved_tflops": F_pt / (fvl_ms * 1e-3) * 1e-12,
                    "note": "gint_fvl (Eq. 46): psi kernel + E = D + D^T gather + T = E Phi (DMMA) + force kernel; T needs every "
                            "(row, column) pair, so F_pt accounting"}
        del Dm, rho, Fv
        # velocity-gauge nonlocal overlaps on the atom-centred quadrature grid (Eq. 47)
        proj = [workloads.projector_species() for _ in w.species]
        rx, rw = workloads.radial_quadrature(140)
        an, aw = workloads.angular_quadrature(110)
        t1 = time.perf_counter()
        ctx.gint_snap_setup(proj, rx, rw, an, aw)
        snap_setup_s = time.perf_counter() - t1
        sp_iat, sp_jat, sp_R, sp_off = ctx.gint_snap_get_pairs()
        Sv = ctx.gint_snap_psibeta((0.08, -0.11, 0.05))
        torch.cuda.synchronize()
        f0.record()
        for _ in range(3):
            ctx.gint_snap_psibeta((0.08, -0.11, 0.05), Sv)
        f1.record()
        torch.cuda.synchronize()
        snap_ms = f0.elapsed_time(f1) / 3
        npts = len(rx) * len(aw)
        snap_flops = 4.0 * float(sp_off[-1]) * npts      # one complex += real x complex per (orbital, projector, point)
        snap_info = {"ms_per_call": snap_ms, "pairs": int(len(sp_iat)), "points_per_pair": int(npts),
                     "point_evaluations_per_s": len(sp_iat) * npts / (snap_ms * 1e-3),
                     "contraction_flops": snap_flops, "contraction_tflops": snap_flops / (snap_ms * 1e-3) * 1e-12,
                     "setup_s": snap_setup_s,
                     "note": "gint_snap_psibeta (Eq. 47): 140 x 110 quadrature points around every projector atom, all "
                             "(I, J, R) pairs in one launch; bound by the per-point evaluation of orbitals and projectors "
                             "(FP64 ALU), the sum over points runs on the tensor pipe"}
        del Sv

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, peaks_src = measured_peaks()
    peak_rule = peaks["bf16_tflops"] * (40.0 / 2250.0)      # bf16 measured x nominal FP64-tensor/bf16 ratio (B200 HGX: 40 / 2250)
    peak = max(peak_live, peak_rule)
    main_ms = float(np.mean([k[0] for k in kern_ms]))
    mirror_ms = float(np.mean([k[1] for k in kern_ms]))
    psi_ms = float(np.mean([k[3] for k in kern_ms]))
    psi_bytes = 8.0 * st["evaluated_pairs"] * (w.norb_total / w.natom) + 8.0 * float(np.prod(w.ngrid))
    F_rank = st["F_sym"]
    achieved = F_rank / (main_ms * 1e-3) * 1e-12
    hbm_bytes = 8.0 * float(np.prod(w.ngrid)) + 8.0 * ctx.h_len
    roofline = {
        "bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
        "traffic": ncu_traffic(w.name),
        "kernel": "gint_contract_kernel<0>", "kernel_ms": main_ms, "mirror_kernel_ms": mirror_ms,
        "kernel_share_of_step": main_ms / ms_per_step,
        "psi_kernel": {"kernel": "gint_psi_kernel", "kernel_ms": psi_ms, "share_of_step": psi_ms / ms_per_step,
                       "bound": "hbm", "implementation_bytes": psi_bytes,
                       "achieved_gbs": psi_bytes / (psi_ms * 1e-3) * 1e-9, "peak_gbs": peaks["hbm_gbs"],
                       "frac": psi_bytes / (psi_ms * 1e-3) * 1e-9 / peaks["hbm_gbs"],
                       "note": "writes psi = phi sqrt(|V dV|) once per listed (atom image, point) pair: "
                               "8 B x orbitals x evaluated pairs, plus V read once"},
        "flops_per_launch": F_rank, "flops_accounting": "F_sym = sum_g n(g)(n(g)+1) (symmetry exploited); F_pt = %.4e" % F_pt,
        "executed_tensor_flops": st["executed_flops"],
        "peak_source": "live DMMA.8x8x4 register-resident microbenchmark (gint_measure_fp64_peak) %.2f; "
                       "rule (MEASURED_PEAKS bf16 %s x 40/2250) %.2f; larger one used" % (peak_live, peaks_src, peak_rule),
        "hbm_algorithmic_bytes": hbm_bytes,
        "hbm_time_floor_ms": hbm_bytes / (peaks["hbm_gbs"] * 1e9) * 1e3,
        "whole_call_frac": value / peak,
    }
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "ms_median": float(np.median(step_ms)), "ms_min": float(step_ms.min()),
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "natom": w.natom, "norb": w.norb_total, "ngrid": [int(x) for x in w.ngrid],
                   "nblocks": ctx.nblocks, "h_doubles": ctx.h_len,
                   "bcell": [int(st["bcell1"]), int(st["bcell2"]), int(st["bcell3"])],
                   "psi_scratch_bytes": st["psi_scratch_bytes"],
                   "l2": "flushed between timed iterations (256 MB write)", "parallelism": "cells sharded x%d" % world,
                   "input_sha256": w.sha256()[:16], "setup_s": setup_s, "wall_s_timed_region": wall},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_call": e2e_ms,
                "h2d_bytes_per_step": int(8 * np.prod(w.ngrid)), "d2h_bytes_per_step": int(8 * ctx.h_len),
                "api": "gint_vlocal_host (pinned host V in, host H out)"},
        "gpu_launches": int(args.steps * st["kernels_per_call"]),
        "roofline": roofline,
    }
    if fold is not None:
        fold["peak_gbs"] = peaks["hbm_gbs"]
        fold["frac"] = fold["achieved_gbs"] / peaks["hbm_gbs"]
        out["fold_k"] = fold
        rho_info["peak_tflops"] = peak
        rho_info["frac"] = rho_info["achieved_tflops"] / peak
        out["rho"] = rho_info
        fvl_info["peak_tflops"] = peak
        fvl_info["frac"] = fvl_info["achieved_tflops"] / peak
        out["fvl"] = fvl_info
        out["snap_psibeta"] = snap_info
    if not args.no_cpu_baseline and world == 1:
        na = min(w.natom, args.ref_atoms or 256)
        dt, used, nblk, ntot = oracle_sample(w, na)
        cval = F_pt * na / w.natom / dt * 1e-12
        out["cpu_baseline"] = {
            "value": cval, "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": "all %d blocks of the first %d of %d row atoms, %.1f s; flops = F_pt*%d/%d (oracle computes both "
                      "(I,J,R) and (J,I,-R))" % (nblk, na, w.natom, dt, na, w.natom),
            "ms_per_call_extrapolated": dt * 1e3 * w.natom / na}
        if snap_info is not None:
            # the same oracle-beside-it for gint_snap_psibeta: the first 256 pairs, one at a time (NumPy, one core)
            import oracle
            nsamp = min(256, len(sp_iat))
            sub_n = (sp_off[1:] - sp_off[:-1])[:nsamp]
            sub = (sp_iat[:nsamp], sp_jat[:nsamp], sp_R[:nsamp], np.concatenate([[0], np.cumsum(sub_n)]).astype(np.int64))
            t1 = time.perf_counter()
            oracle.snap_psibeta(w.lattice, w.species, proj, w.atom_species, w.atom_pos, (0.08, -0.11, 0.05), rx, rw, an, aw, pairs=sub)
            dts = time.perf_counter() - t1
            snap_info["cpu_oracle"] = {"pairs": int(nsamp), "seconds": dts, "cores": 1, "kind": "oracle",
                                       "ms_per_call_extrapolated": dts * 1e3 * len(sp_iat) / nsamp}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
