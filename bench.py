#!/usr/bin/env python
"""bench.py -- seconds per 50-aperture DAO plan on the 9-field prostate phantom (BASELINE.json
configs[1]), plus the SpMV / SpMV^T HBM roofline fractions, on N GPUs of one node.

A "step" is one whole plan: 50 column-generation iterations of the hot path (intensities -> dose
SpMV + objective/gradient -> transposed SpMV -> pricing -> aperture column -> master solve) and the
final dose evaluation, through the C ABI (`dao_run`).  N > 1 runs N independent replicas (the
path does not shard at these sizes: DESIGN.md "Multi-GPU"), one process per GPU under torchrun.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg1] [--impl reference]

Prints ONE JSON line (rank 0).  `--impl reference` times the fp64 CPU oracle instead: one full plan of the
same workload on one host core (minutes; --ref-apertures times a prefix and says so).
"""
from __future__ import annotations

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

METRIC = "50-aperture DAO plan time"
N_APERTURES = 50          # BASELINE.json configs[1]; --apertures overrides it for the other configs (configs[4]: 100)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) >= 9:
                for n, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------
def algorithmic_bytes(ph, sell_elems=None):
    """what each kernel class must move per launch (padding / re-reads excluded)."""
    V, N, nnz, R = ph.n_vox, ph.n_bl, ph.nnz, ph.n_rows
    return {
        "spmv": 8 * nnz + 4 * (V + 1) + 4 * N + 4 * V + V + 4 * V,      # + sid + fused g
        "spmv_t": 8 * nnz + 4 * (N + 1) + 4 * V + 4 * N,
        "price": 4 * N + 4 * (R + 1) + 12 * R,
        "column": 8 * nnz + 4 * (V + 1) + 4 * N + 4 * V,
    }


T_PROCESS_START = time.perf_counter()   # the default run bounds its optional parts against this
TRAFFIC_CSV = os.path.join("profiles", "r02b_traffic.csv")   # one `ncu --set full` capture per kernel; see profiles/r02b_traffic.md


def ncu_traffic(kernel: str):
    """DRAM bytes (read + write) of ONE captured launch of `kernel`, with what identifies that launch (pool size K,
    passes over A), from TRAFFIC_CSV; None when the capture is not committed."""
    import csv
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None
    try:
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel:
                    return {"dram_bytes": int(row["dram_bytes_per_launch"]), "K": int(row.get("K") or 0),
                            "passes": int(row.get("passes") or 0), "pg_iterations": int(row.get("pg_iterations") or 0)}
    except Exception:
        pass
    return None


def measure_l2_bandwidth(torch, l2_bytes: int, reps: int = 400):
    """A denominator for the L2-resident regime of the master ("below that, L2 bandwidth -- say so"):
    read + write GB/s of a device-to-device copy whose source and destination together take a third of the L2, repeated
    back to back so that every pass after the first hits the L2.  torch's copy kernel is the measuring tool here, like
    the copy behind MEASURED_PEAKS.json; it is not on the product path and not counted in gpu_launches."""
    n = max(1 << 20, (l2_bytes // 6) // 4096 * 4096)
    src = torch.empty(n, dtype=torch.uint8, device="cuda").random_(0, 255)
    dst = torch.empty_like(src)
    for _ in range(20):
        dst.copy_(src)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        dst.copy_(src)
    e1.record()
    torch.cuda.synchronize()
    s = e0.elapsed_time(e1) * 1e-3
    return {"GBps": 2.0 * n * reps / s * 1e-9, "bytes_per_buffer": int(n), "reps": reps,
            "how": "torch device-to-device copy, source + destination = L2/3, back to back (read + write bytes / time)"}


def master_alg_bytes(method: int, V: int, K: int, n_iter: int, n_passes: int) -> float:
    """Algorithmic bytes of one master solve.  Methods 0/1: per projected-gradient
    iteration 2*4*V*K (two passes over A) + (n_ls + 3)*8*V with n_ls = the repeated gradient passes per iteration.
    Method 2: every pass reads A once (4*V*K), reads sid (V) and writes the fp64 dose (8*V)."""
    if method >= 2:      # 3: the same pass with the Hessian on tcgen05; sid and thresholds ride in the tile (2 meta rows)
        return float(n_passes) * (4.0 * V * K + 9.0 * V)
    n_ls = max(0, n_passes - (2 * n_iter + 1))
    return n_iter * (2.0 * 4.0 * V * K + 3.0 * 8.0 * V) + n_ls * (4.0 * V * K + 8.0 * V)


def reduce_max(x: float, world: int, device: str = "cuda") -> float:
    """Max over ranks of a per-rank device time (torch.distributed all-reduce; NCCL on the GPU box,
    gloo in the CPU tests).  The multi-rank path has no data-path collective: ranks are replicas."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_seconds_per_plan(elapsed_max: float, steps: int, world: int) -> float:
    """Whole-job metric: `world` replicas each finish `steps` plans in `elapsed_max` seconds."""
    return elapsed_max / (steps * world)


def time_oracle(ph, n_ap):
    """Seconds the oracle, as it stands (one host core), takes for the first n_ap column-generation iterations."""
    from oracle import dao_oracle as orc
    orc.build()
    t0 = time.perf_counter()
    plan = orc.run(ph, n_ap)
    return time.perf_counter() - t0, plan


def cpu_baseline_of(ph, args):
    """The reported CPU baseline: ONE full plan of the oracle (about 140 s for cfg1 on one core), not an extrapolation;
    --ref-apertures < apertures times a prefix instead and says so."""
    n_ap = min(args.ref_apertures or N_APERTURES, N_APERTURES)
    dt, plan = time_oracle(ph, n_ap)
    full = n_ap == N_APERTURES
    return {"value": dt if full else dt * N_APERTURES / n_ap, "unit": "s", "cores": 1, "kind": "oracle",
            "objective": plan.objective,
            "sample": (f"one full {N_APERTURES}-aperture plan of {ph.name} (measured, {dt:.1f} s, not extrapolated)" if full else
                       f"first {n_ap} of {N_APERTURES} column-generation iterations ({dt:.1f} s) scaled by {N_APERTURES}/{n_ap}: "
                       "an UNDER-estimate, later iterations carry larger master problems")}


def run_reference(args, rank, world):
    """The reference arm: the oracle, as it stands, on the host cores.  One full plan per step; because a plan
    takes minutes, --steps / --warmup above 1 / 0 are ignored (said in `sample`)."""
    if rank != 0:
        return
    from paper_1003_5402_b200.inputs import phantom
    ph = phantom.make(args.config, 0)
    cpu = cpu_baseline_of(ph, args)
    cpu["sample"] += "; --steps/--warmup ignored: 1 timed plan, no warm-up"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": "s", "n_gpus": args.gpus,
        "steps": 1, "warmup": 0, "ms_per_step": 1e3 * cpu["value"],
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(ph, args), "cpu_baseline": cpu,
        "e2e": {"value": cpu["value"], "unit": "s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def workload_config(ph, args):
    return {"workload": f"{args.config}: {ph.name}, seed 0, {ph.n_beams} beams, V={ph.n_vox} voxels, N={ph.n_bl} beamlets, "
                        f"nnz={ph.nnz}, {ph.n_rows} leaf rows, {N_APERTURES} apertures",
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU",
            "l2": "inputs larger than L2 (D and D^T are 8*nnz bytes each; no flush needed)"}


def pinned_phantom(ph, torch):
    """Same phantom with its big arrays in pinned host memory (for the e2e leg)."""
    import copy
    q = copy.copy(ph)
    keep = []
    for name in ("row_ptr", "col_idx", "val", "vox_struct"):
        t = torch.from_numpy(np.ascontiguousarray(getattr(ph, name))).pin_memory()
        keep.append(t)
        setattr(q, name, t.numpy())
    q._pinned = keep
    return q


SWEEP_MATRICES = ["sweep_1m", "sweep_3m", "cfg1_literal", "cfg4_literal", "cfg2", "cfg1", "sweep_100m", "cfg4", "sweep_200m"]


def run_sweep(args):
    """BASELINE.json configs[3]: isolated SpMV / SpMV^T on pencil-beam matrices of 1M-200M non-zeros and the
    pricing kernels on 1k-100k leaf rows, GB/s against the measured HBM peak, each checked against the oracle
    (full vectors).  Prints a markdown table; every timing is per launch with CUDA events on the launching
    stream, cold = a 512 MB buffer is rewritten between launches (L2 flushed), warm = back to back."""
    import torch
    from oracle import dao_oracle as orc
    from paper_1003_5402_b200 import build, dao
    from paper_1003_5402_b200.inputs import phantom
    build.build()
    orc.build()
    peak, peak_src = load_peaks()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, reps, cold):
        ts = []
        for _ in range(3):
            fn()
        for _ in range(reps):
            if cold:
                flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        return float(np.median(ts))

    print(f"HBM peak {peak:.0f} GB/s, {peak_src}; bytes = SURVEY 8(d) algorithmic bytes; median of {args.sweep_reps} launches\n")
    print("| matrix | V | N | V:N | nnz | 8 nnz (MB) | SpMV cold us | GB/s | frac | SpMV warm GB/s | SpMV^T cold us | GB/s | frac | SpMV^T warm GB/s | max err z, w vs oracle |")
    print("|---|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---|")
    names = args.sweep_only.split(",") if args.sweep_only else SWEEP_MATRICES
    for name in names:
        ph = phantom.make(name, 0)
        rng = np.random.default_rng(1)
        x = rng.random(ph.n_bl).astype(np.float32)
        g = rng.standard_normal(ph.n_vox).astype(np.float32)
        xd, gd = torch.from_numpy(x).cuda(), torch.from_numpy(g).cuda()
        with dao.Dao(ph, k_max=1) as d:
            zd = torch.empty(ph.n_vox, dtype=torch.float32, device="cuda")
            wd = torch.empty(ph.n_bl, dtype=torch.float32, device="cuda")
            res = {}
            for cold in (True, False):
                res["spmv", cold] = timed(lambda: d.spmv(xd, zd), args.sweep_reps, cold)
                res["spmvt", cold] = timed(lambda: d.spmv_t(gd, wd), args.sweep_reps, cold)
            z, w = zd.cpu().numpy(), wd.cpu().numpy()
        zo = orc.dose(ph.row_ptr, ph.col_idx, ph.val, x.astype(np.float64))
        wo = orc.beamlet_gradient(ph.row_ptr, ph.col_idx, ph.val, g.astype(np.float64), ph.n_bl)
        ez, ew = np.abs(z - zo).max() / np.abs(zo).max(), np.abs(w - wo).max() / np.abs(wo).max()
        b_spmv = 8 * ph.nnz + 4 * (ph.n_vox + 1) + 4 * ph.n_bl + 4 * ph.n_vox
        b_t = 8 * ph.nnz + 4 * (ph.n_bl + 1) + 4 * ph.n_vox + 4 * ph.n_bl
        c1, w1, c2, w2 = res["spmv", True], res["spmv", False], res["spmvt", True], res["spmvt", False]
        print(f"| {name} ({ph.name}) | {ph.n_vox} | {ph.n_bl} | {ph.n_vox / ph.n_bl:.0f} | {ph.nnz} | {8e-6 * ph.nnz:.0f} | "
              f"{1e6 * c1:.1f} | {1e-9 * b_spmv / c1:.0f} | {1e-9 * b_spmv / c1 / peak:.2f} | {1e-9 * b_spmv / w1:.0f} | "
              f"{1e6 * c2:.1f} | {1e-9 * b_t / c2:.0f} | {1e-9 * b_t / c2 / peak:.2f} | {1e-9 * b_t / w2:.0f} | {ez:.1e}, {ew:.1e} |", flush=True)
        del ph, zo, wo
    print("\n| leaf rows R | beamlets per row | N | pricing cold us | GB/s (4N + 4(R+1) + 20R bytes) | frac | warm us | rows bit-exact vs oracle | best beam |")
    print("|---:|---:|---:|---:|---:|---:|---:|---|---|")
    ph = phantom.make("cfg1_literal", 0)
    with dao.Dao(ph, k_max=1) as d:
        for n_rows in (1000, 10000, 100000):
            for row_len in (20, 40, 80):
                w, brp, rbp = phantom.pricing_rows(n_rows, row_len, rows_per_beam=40, seed=n_rows % 3)
                wd, rd, bd = (torch.from_numpy(a).cuda() for a in (w, rbp, brp))
                tc = timed(lambda: d.price_from_w(wd, rd, bd), args.sweep_reps, True)
                tw = timed(lambda: d.price_from_w(wd, rd, bd), args.sweep_reps, False)
                le, ri, vs, bp, best = (t.cpu().numpy() for t in d.price_from_w(wd, rd, bd))
                pr = orc.price(w.astype(np.float64), brp, rbp)
                same = int(((le == pr.left) & (ri == pr.right)).sum())
                nbytes = 4 * w.size + 4 * (n_rows + 1) + 20 * n_rows
                print(f"| {n_rows} | {row_len} | {w.size} | {1e6 * tc:.1f} | {1e-9 * nbytes / tc:.0f} | {1e-9 * nbytes / tc / peak:.3f} | "
                      f"{1e6 * tw:.1f} | {same}/{n_rows} | {'same' if int(best[0]) == pr.best_beam else 'differs'} |", flush=True)


def run_widened(args):
    """Measurements of the SURVEY 8(f) rows built beyond the paper's experiments, on the bench workload: the FMO
    workload (8f-2), the re-optimisation mode (8f-1) and the alternative MLC rules (8f-4).  Markdown table."""
    import torch
    from paper_1003_5402_b200 import build, dao
    from paper_1003_5402_b200.inputs import phantom
    build.build()
    peak, peak_src = load_peaks()
    ph = phantom.make(args.config, 0)
    print(f"workload {args.config}: {ph.name}, V={ph.n_vox}, N={ph.n_bl}, nnz={ph.nnz}; HBM peak {peak:.0f} GB/s ({peak_src})\n")
    print("| row | what | result |")
    print("|---|---|---|")
    with dao.Dao(ph, k_max=N_APERTURES) as d:
        d.fmo_solve(max_iter=50)
        f = d.fmo_solve(max_iter=1000, tol=1e-9)
        per_it = f.seconds / max(1, f.n_iter)
        moved = 3 * 8 * ph.nnz                      # dose SpMV + SpMV^T + dz SpMV per iteration
        print(f"| 8f-2 FMO | {f.n_iter} projected-gradient iterations from x = 0 | {f.seconds:.3f} s, {1e6 * per_it:.0f} us per iteration "
              f"(3 SpMV-class passes = {moved / per_it * 1e-9:.0f} GB/s, {moved / per_it * 1e-9 / peak:.2f} of peak), F = {f.objective:.6g}, "
              f"{f.n_ls_evals} line-search evaluations |")
    modes = [("consecutive (the paper's experiments)", dao.MLC_CONSECUTIVE), ("8f-4 jaws-only", dao.MLC_JAWS_ONLY),
             ("8f-4 interdigitation", dao.MLC_INTERDIGITATION), ("8f-4 connectedness", dao.MLC_CONNECTED)]
    for name, code in modes:
        with dao.Dao(ph, k_max=N_APERTURES, mlc_mode=code) as d:
            d.run(N_APERTURES); d.reset()
            i = d.run(N_APERTURES)
        n = max(1, i.n_iterations)
        print(f"| {name} | {i.n_apertures}-aperture plan | {i.seconds_total:.4f} s, pricing {1e6 * i.seconds_price / n:.1f} us per iteration, "
              f"master {1e6 * i.seconds_master / n:.0f} us, F = {i.objective:.6g}, {i.n_pg_iter_total} projected-gradient iterations |")
    pr = phantom.make(args.config + "_reopt", 0)
    with dao.Dao(pr, k_max=N_APERTURES) as d:
        d.run(N_APERTURES); d.reset()
        i = d.run(N_APERTURES)
    n = max(1, i.n_iterations)
    print(f"| 8f-1 re-optimisation (per-voxel T_j) | {i.n_apertures}-aperture plan | {i.seconds_total:.4f} s, dose SpMV {1e6 * i.seconds_spmv / n:.1f} us, "
          f"master {1e6 * i.seconds_master / n:.0f} us per iteration, F = {i.objective:.6g}, {i.n_pg_iter_total} projected-gradient iterations |")


def main():
    global N_APERTURES, METRIC
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg1")
    ap.add_argument("--impl", default="dao", choices=["dao", "reference"])
    ap.add_argument("--apertures", type=int, default=N_APERTURES, help="apertures per plan (50; configs[4] asks for 100)")
    ap.add_argument("--ref-apertures", type=int, default=0,
                    help="apertures of the oracle run behind cpu_baseline / --impl reference (0 = the full plan; fewer = a scaled prefix)")
    ap.add_argument("--master-method", type=int, default=2, help="dao_options.master_method (2 = projected Newton, exact Hessian on the fp64 tensor cores; 3 = the same with the Hessian on tcgen05 in split TF32; 1 = conjugated gradient projection)")
    ap.add_argument("--split-steps", type=int, default=2, help="plans of the separate per-kernel-class timing pass")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the plan times of paper_p1 / configs[2] / configs[4] and of master_method = 3 that the default run appends")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[3] kernel sweep (markdown table)")
    ap.add_argument("--widened", action="store_true", help="measure the SURVEY 8(f) rows (FMO, re-optimisation, MLC modes)")
    ap.add_argument("--sweep-reps", type=int, default=15)
    ap.add_argument("--sweep-only", default="", help="comma-separated subset of the sweep matrices")
    args = ap.parse_args()
    N_APERTURES = args.apertures
    METRIC = f"{N_APERTURES}-aperture DAO plan time"
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.sweep:
        if rank == 0:
            run_sweep(args)
        return
    if args.widened:
        if rank == 0:
            run_widened(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_1003_5402_b200 import build, dao
    from paper_1003_5402_b200.inputs import phantom

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    build.build()
    ph = phantom.make(args.config, 0)
    peak, peak_src = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K plans through dao_run, NO event timers inside the library ----
    opts = dict(k_max=N_APERTURES, master_method=args.master_method)
    d = dao.Dao(ph, timers=0, **opts)
    dims = d.dims()
    method = int(d.dims().master_method)          # the method in effect (capacity fallbacks applied)
    infos = []
    for _ in range(args.warmup):
        d.reset()
        d.run(N_APERTURES)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        d.reset()
        infos.append(d.run(N_APERTURES))
    ev1.record()
    barrier()
    clocks = sampler.stop()
    elapsed = ev0.elapsed_time(ev1) * 1e-3
    elapsed = reduce_max(elapsed, world)
    sec_per_plan = job_seconds_per_plan(elapsed, args.steps, world)   # N replicas produce N plans per step
    last = infos[-1]
    n_it = sum(i.n_iterations for i in infos)
    launches = sum(i.n_kernel_launches for i in infos)
    timed_plan = d.get_plan()
    d.close()

    # ---- per-kernel-class split: a separate pass with the library's CUDA-event timers on (same kernels, same plan;
    #      the events cost a few us per iteration, which is why they are not in the timed region) ----
    dt_ = dao.Dao(ph, timers=1, **opts)
    dt_.run(N_APERTURES)
    tinfos = []
    for _ in range(max(1, args.split_steps)):
        dt_.reset()
        tinfos.append(dt_.run(N_APERTURES))
    hist = dt_.get_vector(dao.VEC_HISTORY)[:tinfos[-1].n_apertures]
    # the timed pass (timers = 0: speculative dose SpMV behind the state copy) and this pass (timers = 1, the branch the
    # parity tests run against the oracle) must have produced the SAME plan, bit for bit -- a stale-dose or ordering bug
    # in the untimed branch would show here
    split_plan = dt_.get_plan()
    assert (tinfos[-1].objective == last.objective and tinfos[-1].n_apertures == last.n_apertures and
            tinfos[-1].n_iterations == last.n_iterations and tinfos[-1].n_passes_total == last.n_passes_total), \
        ("timed (timers=0) and split (timers=1) passes disagree", last.objective, tinfos[-1].objective)
    for f in ("beams", "intensity", "ap_row_ptr", "left", "right"):
        assert np.array_equal(getattr(timed_plan, f), getattr(split_plan, f)), f"timers=0 / timers=1 plans differ in {f}"
    it_sec = dt_.get_vector(dao.VEC_ITER_SECONDS).reshape(-1, 6)[:tinfos[-1].n_apertures]   # one row per aperture added: pairs with hist
    dt_.close()
    n_it_t = sum(i.n_iterations for i in tinfos)
    ab = algorithmic_bytes(ph)
    classes = {"intensity": "seconds_intensity", "spmv": "seconds_spmv", "spmv_t": "seconds_spmv_t",
               "price": "seconds_price", "column": "seconds_column", "master": "seconds_master"}
    tot = {k: sum(getattr(i, f) for i in tinfos) for k, f in classes.items()}
    tsum = sum(tot.values())
    kernels = {}
    for k in classes:
        avg = tot[k] / max(1, n_it_t)
        kernels[k] = {"avg_us": 1e6 * avg, "share": tot[k] / tsum if tsum > 0 else None}
        if k in ab and avg > 0:
            gbs = ab[k] / avg * 1e-9
            kernels[k].update({"alg_bytes": ab[k], "GBps": gbs, "frac_of_hbm_peak": gbs / peak})

    # ---- the master: algorithmic bytes per solve from the per-iteration history, split by where A lives ----
    V = ph.n_vox
    l2_bytes = int(torch.cuda.get_device_properties(local_rank).L2_cache_size)
    vpad = (V + 127) // 128 * 128
    solves = []
    for h, sec in zip(hist, it_sec):
        K = int(h["k"])
        solves.append({"K": K, "bytes": master_alg_bytes(method, V, K, int(h["n_pg_iter"]), int(h["n_passes"])),
                       "s": float(sec[5]), "passes": int(h["n_passes"]), "iters": int(h["n_pg_iter"]),
                       "regime": "hbm" if 4.0 * vpad * K >= 0.8 * l2_bytes else "l2"})
    master_bytes_plan = sum(x["bytes"] for x in solves)
    master_s_plan = sum(x["s"] for x in solves)
    regimes = {}
    for r in ("l2", "hbm"):
        sel = [x for x in solves if x["regime"] == r]
        if sel:
            bsum, ssum = sum(x["bytes"] for x in sel), sum(x["s"] for x in sel)
            regimes[r] = {"solves": len(sel), "K_range": [min(x["K"] for x in sel), max(x["K"] for x in sel)],
                          "alg_bytes": bsum, "seconds": ssum, "achieved_GBps": bsum / ssum * 1e-9 if ssum > 0 else None,
                          "share_of_master_time": ssum / master_s_plan if master_s_plan > 0 else None}
    l2_bw = measure_l2_bandwidth(torch, l2_bytes) if "l2" in regimes else None
    if "l2" in regimes:
        regimes["l2"].update({"peak": l2_bw["GBps"], "frac": regimes["l2"]["achieved_GBps"] / l2_bw["GBps"],
                              "peak_source": l2_bw,
                              "note": "4*V*K fits the L2: the peak is an L2-resident copy bandwidth measured in this run"})
    if "hbm" in regimes:
        regimes["hbm"].update({"peak": peak, "frac": regimes["hbm"]["achieved_GBps"] / peak})
    kernels["master"].update({
        "method": method, "iterations_per_plan": sum(x["iters"] for x in solves), "passes_over_A_per_plan": sum(x["passes"] for x in solves),
        "alg_bytes_per_plan": master_bytes_plan, "GBps": master_bytes_plan / master_s_plan * 1e-9 if master_s_plan > 0 else None,
        "regimes": regimes})
    plan_bytes = N_APERTURES * (ab["spmv"] + ab["spmv_t"] + ab["price"] + ab["column"]) + master_bytes_plan

    master_kernel = "k_master_newton" if method >= 2 else "k_master"
    master_model = ("per pass over A: 4*V*K (A read once) + V (sid) + 8*V (fp64 dose written); a solve makes `passes` passes"
                    if method >= 2 else
                    "SURVEY 8(d): per projected-gradient iteration 2*4*V*K + (n_ls+3)*8*V, n_ls = repeated gradient passes")

    def traffic_of(kernel, alg_of_launch):
        """ncu DRAM bytes of ONE captured launch next to the algorithmic bytes of that same launch."""
        t = ncu_traffic(kernel)
        if t is None:
            return None, None
        return t["dram_bytes"], {"source": TRAFFIC_CSV, "launch": {k: v for k, v in t.items() if k != "dram_bytes" and v},
                                 "alg_bytes_of_that_launch": alg_of_launch(t),
                                 "dram_over_alg": t["dram_bytes"] / alg_of_launch(t) if alg_of_launch(t) else None}

    def class_roofline(key, kernel_name, label):
        k = kernels[key]
        tr, trd = traffic_of(kernel_name, lambda t: ab[key])
        return {"kernel": label, "bound": "hbm", "achieved": k.get("GBps"), "peak": peak, "unit": "GB/s",
                "frac": k.get("frac_of_hbm_peak"), "frac_of_nominal_8000": (k.get("GBps") or 0.0) / 8000.0,
                "traffic": tr, "traffic_detail": trd, "alg_bytes_per_launch": ab[key],
                "avg_launch_us": k["avg_us"], "share_of_step": k["share"], "peak_source": peak_src}

    roofline_kernels = {
        "spmv": class_roofline("spmv", "k_spmv_ring<0>", "k_spmv_ring<0> (dose SpMV + fused objective/gradient)"),
        "spmv_t": class_roofline("spmv_t", "k_spmvt", "k_spmvt + k_spmvt_finish (w = D^T pi)"),
        "column": class_roofline("column", "k_spmv_ring<2>", "k_spmv_ring<2> (aperture column a_K = D 1_A)"),
        "sell_padding": dims.sell_elems / max(1, ph.nnz)}
    # the master's roofline object: the HBM regime when the plan has one (A streams from DRAM), else the L2 regime
    hb = regimes.get("hbm")
    head = hb or regimes.get("l2") or {}
    mtr, mtrd = traffic_of(master_kernel + ("@method3" if method == 3 else ""), lambda t: master_alg_bytes(method, V, t["K"], t["pg_iterations"], t["passes"]))
    n_head = max(1, head.get("solves", 1))
    master_roofline = {
        "kernel": f"{master_kernel} (restricted master problem over the dense block A, method {method})",
        "bound": "hbm" if hb else "l2", "achieved": head.get("achieved_GBps"), "peak": peak if hb else None, "unit": "GB/s",
        "frac": hb["frac"] if hb else None, "traffic": mtr, "traffic_detail": mtrd, "peak_source": peak_src,
        "alg_bytes_per_launch": head.get("alg_bytes", 0.0) / n_head, "avg_launch_us": 1e6 * head.get("seconds", 0.0) / n_head,
        "alg_bytes_model": master_model, "share_of_step": kernels["master"]["share"],
        # the same quotient over ALL launches of the plan (every pool size, L2-resident solves included) against the HBM
        # peak: `frac` above describes the HBM-regime solves only
        "frac_all_launches": (master_bytes_plan / master_s_plan * 1e-9 / peak) if master_s_plan > 0 else None,
        "achieved_all_launches": (master_bytes_plan / master_s_plan * 1e-9) if master_s_plan > 0 else None,
        "alg_bytes_per_launch_all": master_bytes_plan / max(1, len(solves)),
        "avg_launch_us_all": 1e6 * master_s_plan / max(1, len(solves)),
        # `traffic` is the ncu DRAM count of ONE captured launch; these are the algorithmic bytes of that same launch
        "traffic_launch_alg_bytes": (mtrd or {}).get("alg_bytes_of_that_launch"),
        "traffic_over_alg_same_launch": (mtrd or {}).get("dram_over_alg"),
        "traffic_source": TRAFFIC_CSV + " (committed ncu capture of an earlier build of this kernel; re-capture after kernel changes)",
        "regime": (f"solves with 4*V_pad*K >= 0.8 x L2 ({l2_bytes >> 20} MB): K = {hb['K_range'][0]}..{hb['K_range'][1]}, "
                   f"{100 * hb['share_of_master_time']:.0f} % of the master's time; the other solves are L2-resident (see regimes)"
                   if hb else "every solve is L2-resident: no HBM figure, no measured L2 peak"),
        "regimes": regimes}
    shares = {k: (kernels[k]["share"] or 0.0) for k in kernels}
    dominant = max(shares, key=shares.get)
    roofline = master_roofline if dominant == "master" else roofline_kernels[dominant]
    roofline["dominant_class"] = dominant

    # ---- e2e: host (pinned) buffers -> dao_create -> dao_run -> dao_get_plan, wall clock ----
    e2e = None
    if args.e2e_steps > 0:
        php = pinned_phantom(ph, torch)
        h2d = int(php.row_ptr.nbytes + php.col_idx.nbytes + php.val.nbytes + php.vox_struct.nbytes)
        d2h = 0
        ts = []
        for i in range(args.e2e_steps + 1):
            barrier()
            t0 = time.perf_counter()
            with dao.Dao(php, timers=0, **opts) as d2:
                inf = d2.run(N_APERTURES)
                plan = d2.get_plan()
                d2h = int(plan.beams.nbytes + plan.intensity.nbytes + plan.ap_row_ptr.nbytes + plan.left.nbytes +
                          plan.right.nbytes + (inf.n_iterations + 3) * 128)
            torch.cuda.synchronize()
            if i > 0:
                ts.append(time.perf_counter() - t0)
        e = float(np.mean(ts))
        e = reduce_max(e, world)
        e2e = {"value": e / world, "unit": "s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "includes": f"dao_create from pinned host CSR (H2D + sliced-ELL + transpose build), dao_run({N_APERTURES}), dao_get_plan"}

    # ---- the other BASELINE.json configs and master_method = 3, plan time only (rank 0, N = 1; bounded) ----
    others = None
    if rank == 0 and world == 1 and args.config == "cfg1" and not args.no_other_configs:
        others = {}

        def plan_time(ph_o, n_ap, split=False, **o):
            with dao.Dao(ph_o, timers=0, k_max=n_ap, **o) as d3:
                for _ in range(3):
                    d3.reset()
                    inf3 = d3.run(n_ap)
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(3):
                    d3.reset()
                    inf3 = d3.run(n_ap)
                e1.record()
                torch.cuda.synchronize()
                res = {"seconds_per_plan": e0.elapsed_time(e1) * 1e-3 / 3, "apertures": int(inf3.n_apertures),
                       "objective": inf3.objective, "master_passes_over_A": int(inf3.n_passes_total),
                       "master_method": int(d3.dims().master_method), "n_vox": int(ph_o.n_vox), "n_bl": int(ph_o.n_bl),
                       "nnz": int(ph_o.nnz)}
            if split:
                # BASELINE.json configs[4]: "per-iteration time split across SpMV, gradient, pricing and master solve"
                # (the gradient is fused into the dose SpMV's epilogue): one more plan with the library's event timers on
                with dao.Dao(ph_o, timers=1, k_max=n_ap, **o) as d4:
                    d4.run(n_ap); d4.reset()
                    i4 = d4.run(n_ap)
                cls = {"intensity": i4.seconds_intensity, "spmv_dose_objective_gradient": i4.seconds_spmv,
                       "spmv_t": i4.seconds_spmv_t, "pricing": i4.seconds_price, "column": i4.seconds_column,
                       "master": i4.seconds_master}
                tot4 = sum(cls.values())
                res["per_iteration_split_us"] = {k: 1e6 * v / max(1, i4.n_iterations) for k, v in cls.items()}
                res["split_share"] = {k: v / tot4 for k, v in cls.items()} if tot4 > 0 else None
                res["split_same_plan"] = bool(i4.objective == res["objective"])
            return res

        others["cfg1_master_method_3"] = plan_time(ph, N_APERTURES, master_method=3)
        # the gradient projection PAPER.md:134 names (conjugated directions on the free face), same plan, same optimum
        others["cfg1_master_method_1"] = plan_time(ph, N_APERTURES, master_method=1)
        for name, n_ap in (("paper_p1", 50), ("cfg2", 50), ("cfg4", 100)):
            if time.perf_counter() - T_PROCESS_START > (90.0 if name == "cfg4" else 150.0):
                others[name] = {"skipped": "time budget of the default run (the whole run must end within minutes)"}
                continue
            others[name] = plan_time(phantom.make(name, 0), n_ap, master_method=args.master_method, split=(name == "cfg4"))

    # ---- CPU baseline: the oracle as it stands, one full plan, rank 0, N = 1 only ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_of(ph, args)

    if rank == 0:
        out = {"metric": METRIC, "value": sec_per_plan, "unit": "s", "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": 1e3 * elapsed / args.steps, "higher_is_better": False,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32 storage, f64 accumulate", "data": "synthetic",
               "config": workload_config(ph, args), "clocks": clocks, "e2e": e2e,
               "gpu_launches": int(launches), "roofline": roofline, "roofline_kernels": roofline_kernels,
               "roofline_master": master_roofline, "cpu_baseline": cpu, "kernels": kernels, "other_configs": others,
               "plan": {"objective": last.objective, "apertures": last.n_apertures, "cg_iterations_per_s": n_it / elapsed,
                        "master_iterations": int(last.n_pg_iter_total), "master_passes_over_A": int(last.n_passes_total),
                        "master_hit_max_iter": int(last.n_hit_max_iter), "converged": int(last.converged),
                        "duplicates": int(last.n_duplicates), "kernel_launches_per_plan": int(last.n_kernel_launches),
                        "bytes_moved_roofline_s": plan_bytes / (peak * 1e9),
                        "frac_of_bytes_moved_roofline": plan_bytes / (peak * 1e9) / (elapsed / args.steps),
                        "bytes_model": "sum over iterations of the SURVEY 8(d) bytes of the three SpMV-class kernels and pricing + the "
                                       "master's algorithmic bytes (roofline_master.alg_bytes_model), all over the measured HBM peak",
                        "master_tol": d.opt.master_tol, "master_max_iter": d.opt.master_max_iter,
                        "master_method": method},
               "timers": "value / ms_per_step: dao_run with timers = 0; kernels / roofline*: a separate pass with the library's "
                         "CUDA-event timers on",
               "paper_context": "0.7-2.5 s per 50-aperture plan on a Tesla C1060 for ~20x smaller clinical cases (PAPER.md:202)"}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
