#!/usr/bin/env python
"""bench.py -- throughput of the QLP BLS hot path (S0..S4) on synthetic TESS-shaped light curves.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C] [--stars S]

One "step" = one pass of the whole hot path (grid -> prep -> fold+box-scan -> S/N + peaks -> peak statistics) over one
batch.  Default workload = the north-star configuration, BASELINE.json configs[4] ("config 5": the 200,000-star
production-shaped ragged batch; PAPER.md:7 abstract, Table 1 at :67-71 are whole-sector multi-sector figures): its
first 4,000 stars per GPU (a cost-representative prefix: every star has its own seed, the prefix holds 40 of the
top-1 % heaviest stars), so that a default run ends within a few minutes.  `--config 5 --stars 200000 --chunk 20000`
searches the whole batch in chunks; `--config 2 --stars 1000` is the small single-sector case.  ONE JSON line (rank 0).

  value        : point x frequency BLS evaluations per second, whole job, inputs resident in HBM
  e2e          : the same metric through qlp_bls_search_host with pinned HOST buffers (H2D + D2H inside)
  e2e_vet      : the same through qlp_bls_vet_host (search + trapezoid fit + noise / detection row)
  roofline     : fold+box-scan launches, CUDA-event timed inside the timed region, against the shared-memory-atomic
                 issue ceiling derived in DESIGN.md ("bound": "alu"), with the per-tile-class split
  cpu_baseline : oracle/ (the unoptimised checker, not a tuned CPU BLS) timed on this box's host cores on a bounded,
                 cost-stratified sample (N=1, rank 0 only)

`--gpus N` without a torchrun environment re-launches itself under `python -m torch.distributed.run` with N ranks
(one per GPU).  Stars are dealt to ranks by cost N_pts x n_freq (longest-processing-time greedy after a device grid
pass); the per-star peak table is gathered with one NCCL all-gather per step.
`--impl reference` times the oracle (the only reference that exists for this paper) on the host.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bls_point_frequency_evals_per_s"
UNIT = "evals/s"
DEFAULT_CONFIG, DEFAULT_STARS = 5, 4000
DTYPE = "f64 phase / int32 fixed-point accumulators / f32 box scan"
# per evaluation the fold needs 2 shared-memory integer atomic lanes and 3 FP64
# lanes (the exact bin takes three FP64 instructions); measured ceilings on B200 (profiles/ubench_r1.txt):
# ATOMS.ADD lanes/clk/SM and FP64 lanes/clk/SM.  The binding one is the atomic path.
ATOMS_LANES_PER_CLK_SM = 31.6
FP64_LANES_PER_CLK_SM = 62.3
N_SM = 148
# dram__bytes_read.sum + dram__bytes_write.sum over the foldscan launches of ONE step of a named workload, from an
# `ncu --set full` capture kept under profiles/ (not measured in this run: a run under ncu is never a bench value).
NCU_TRAFFIC = {
    (5, 4000): (7.837e9, "profiles/r2_launches.md (ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum over the "
                         "nine foldscan launches of one step of this workload)"),
    (2, 1000): (719.3e6, "profiles/r1_foldscan_ncu.txt (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum "
                         "over the foldscan launches of one step)"),
}
CLASS_COLS = [128, 128, 64, 32, 16, 8, 4, 2, 1]
CLASS_NBCAP = [94, 208, 420, 840, 1680, 3360, 6720, 13440, 24576]


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def fold_peak_evals_per_s(sm_mhz: float) -> float:
    per_clk_sm = min(ATOMS_LANES_PER_CLK_SM / 2.0, FP64_LANES_PER_CLK_SM / 3.0)
    return N_SM * sm_mhz * 1e6 * per_clk_sm


def fold_issue_bound_evals_per_s(sm_mhz: float) -> float:
    """Tighter bound: an FP64 instruction costs its scheduler 2 issue cycles and nothing issues in its shadow
    (profiles/ubench_r1.txt), so 32 evaluations cost >= 3*2 + 2 (address) + 2 (ATOMS) + 0.25 (LDS) cycles."""
    return N_SM * sm_mhz * 1e6 * 4 * 32 / 10.25


def scan_roofline(total_bins: int, n_widths: int, fold_s: float, scan_share: float, sm_mhz: float):
    cand = float(total_bins) * n_widths
    t = fold_s * scan_share
    # 8 instructions per candidate, one of them a MUFU.RCP (16 lanes/clk/SM): both give 16 candidates/clk/SM
    bound = N_SM * sm_mhz * 1e6 * 16.0
    ach = cand / t if t > 0 else 0.0
    return {"achieved": ach / 1e9, "peak": bound / 1e9, "unit": "Gcandidates/s", "frac": ach / bound,
            "candidates_per_step": cand}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------- workload
def shard_star_ids(n_stars_per_gpu: int, rank: int) -> np.ndarray:
    """The contiguous slice of star ids a rank starts from (ids [r*n, (r+1)*n)): the slice whose costs it measures
    before the cost-balanced deal (stars are independent; no data-path collective)."""
    return np.arange(rank * n_stars_per_gpu, (rank + 1) * n_stars_per_gpu, dtype=np.int64)


def make_workload(config: int, n_stars: int, rank: int):
    """Seeded synthetic batch of the contiguous slice of rank `rank`."""
    from paper_2302_01293_b200 import synth
    return synth.make_batch(config, star_ids=shard_star_ids(n_stars, rank))


def _gen_block(job):
    from paper_2302_01293_b200 import synth
    config, ids = job
    b = synth.make_batch(config, star_ids=np.asarray(ids, dtype=np.int64))
    return b.row_ptr, b.t, b.y, b.dy, b.rho, b.rstar, b.truth


def _times_block(job):
    from paper_2302_01293_b200 import synth
    config, ids = job
    ts, rho = [], []
    for sid in ids:
        t, r = synth.star_times(config, int(sid))
        ts.append(t); rho.append(r)
    return ts, rho


def make_workload_ids(config: int, ids, pool, block: int = 250):
    """The stars `ids` of a config, generated by the worker pool in blocks (every star has its own seed,
    paper_2302_01293_b200.synth), packed into one CSR batch in the order of `ids`."""
    from paper_2302_01293_b200 import synth
    ids = np.asarray(ids, dtype=np.int64)
    jobs = [(config, ids[a:a + block]) for a in range(0, ids.size, block)]
    parts = pool.map(_gen_block, jobs) if pool is not None else [_gen_block(j) for j in jobs]
    if not parts:
        return synth.make_batch(config, star_ids=ids)
    sizes = np.concatenate([np.diff(p[0]) for p in parts])
    row_ptr = np.zeros(sizes.size + 1, dtype=np.int64)
    np.cumsum(sizes, out=row_ptr[1:])
    cat = lambda k: np.concatenate([p[k] for p in parts])
    return synth.Batch(config, 0, ids, row_ptr, cat(1), cat(2), cat(3), cat(4), cat(5), cat(6))


def make_workload_parallel(config: int, lo: int, hi: int, pool, block: int = 250):
    """Stars [lo, hi) of a config (see make_workload_ids)."""
    return make_workload_ids(config, np.arange(lo, hi, dtype=np.int64), pool, block)


def make_times_ids(config: int, ids, pool, block: int = 500):
    """Timestamps and densities only (no flux) of the stars `ids`: the input of the cost pass -> (row_ptr, t, rho)."""
    ids = np.asarray(ids, dtype=np.int64)
    jobs = [(config, ids[a:a + block]) for a in range(0, ids.size, block)]
    parts = pool.map(_times_block, jobs) if pool is not None else [_times_block(j) for j in jobs]
    ts = [t for p in parts for t in p[0]]
    rho = np.array([r for p in parts for r in p[1]], dtype=np.float64)
    row_ptr = np.zeros(len(ts) + 1, dtype=np.int64)
    np.cumsum([t.size for t in ts], out=row_ptr[1:])
    return row_ptr, (np.concatenate(ts) if ts else np.zeros(0)), rho


# ---------------------------------------------------------------------------------------------- the oracle, timed
GRID_NOTE = "comparison grid O1.10 (PAPER.md:13): P <= 56 d, <= 80,000 frequencies per star"
GRID_KW = {}   # --comparison-grid: the O1.10 caps, given to both the CUDA context and the oracle config
ORACLE_KIND = "oracle"
ORACLE_NOTE = ("the unoptimised FP64 checker of oracle/ as it stands (triple-loop box scan, 128-bit bin index, malloc per "
               "star): a reported baseline, not a tuned CPU BLS; a GPU/CPU ratio formed from it says nothing about "
               "kernel quality")


class OracleSample:
    """A bounded, cost-stratified sample of a workload for timing the oracle as it stands: whole
    path (grid + SR + S/N + peaks, OpenMP over stars) on stars at evenly spaced cost ranks that one thread finishes
    within the budget, plus -- where the workload has one -- the star with the most frequencies (> 10^5) on a sample
    of its frequencies (fold + box scan only, OpenMP over frequencies)."""

    def __init__(self, batch, budget_s: float, threads: int):
        from oracle import oracle as orc
        from paper_2302_01293_b200 import synth
        orc.build()
        self.orc, self.threads = orc, threads
        self.cfg = orc.default_config(**GRID_KW)
        S = batch.n_stars
        npts = np.diff(batch.row_ptr).astype(np.float64)
        nf = np.zeros(S)
        grids = []
        for s in range(S):
            g = orc.grid(self.cfg, batch.star(s)[0], float(batch.rho[s]))
            grids.append(g)
            nf[s] = float(g["n_freq"])
        cost = npts * nf
        # calibration on `threads` stars of median cost
        med = np.argsort(cost, kind="stable")[S // 2: S // 2 + threads]
        sub = synth.from_arrays([batch.star(int(s)) for s in med], rho=batch.rho[med])
        t0 = time.perf_counter()
        orc.batch(self.cfg, sub.row_ptr, sub.t, sub.y, sub.dy, sub.rho, K=3, want_snr=True, threads=threads)
        dt = max(time.perf_counter() - t0, 1e-3)
        rate = max(cost[med].sum() / dt, 1.0)                 # evals/s, all threads
        per_thread = rate / max(min(threads, med.size), 1)
        ok = np.nonzero((cost > 0) & (cost <= 0.5 * budget_s * per_thread))[0]
        ok = ok[np.argsort(cost[ok], kind="stable")]
        if ok.size == 0:   # a budget below one star per thread: the cheapest stars, one per thread
            ok = np.argsort(np.where(cost > 0, cost, np.inf), kind="stable")[:max(1, min(threads, int((cost > 0).sum())))]
        want = 0.7 * budget_s * rate
        n_light = int(max(min(ok.size, threads), min(ok.size, want / max(cost[ok].mean(), 1.0)))) if ok.size else 0
        pick = np.unique(ok[np.linspace(0, ok.size - 1, n_light).round().astype(np.int64)]) if n_light else ok[:0]
        self.light = synth.from_arrays([batch.star(int(s)) for s in pick], rho=batch.rho[pick])
        self.light_evals = float(cost[pick].sum())
        self.heavy = None
        big = int(np.argmax(nf))
        if nf[big] > 1e5 and cost[big] > 0.5 * budget_s * per_thread:
            nk = int(min(nf[big], max(64, 0.3 * budget_s * rate / npts[big])))
            ks = np.unique(np.linspace(0, nf[big] - 1, nk).round().astype(np.int64))
            self.heavy = (grids[big], batch.star(big), ks)
            self.heavy_evals = float(npts[big] * ks.size)
        self.desc = (f"{pick.size} stars at evenly spaced cost ranks of the workload (whole path: grid+SR+S/N+peaks)"
                     + (f" + {self.heavy[2].size} evenly spaced frequencies of its longest-grid star "
                        f"({int(nf[big])} frequencies, {int(npts[big])} points; fold+box scan)" if self.heavy else ""))

    def run(self):
        """One timed pass -> (seconds, evaluations)."""
        orc = self.orc
        t0 = time.perf_counter()
        ev = 0.0
        if self.light.n_stars:
            orc.batch(self.cfg, self.light.row_ptr, self.light.t, self.light.y, self.light.dy, self.light.rho, K=3,
                      want_snr=True, threads=self.threads)
            ev += self.light_evals
        if self.heavy is not None:
            g, (t, y, dy), ks = self.heavy
            orc.spectrum_samples(self.cfg, g, t, y, dy, ks)
            ev += self.heavy_evals
        return time.perf_counter() - t0, ev


def cpu_baseline(batch, budget_s: float = 15.0):
    cores = os.cpu_count() or 1
    smp = OracleSample(batch, budget_s, cores)
    dt, ev = smp.run()
    return {"value": ev / dt, "unit": UNIT, "cores": cores, "kind": ORACLE_KIND, "note": ORACLE_NOTE,
            "sample": f"{smp.desc}, {dt:.1f} s", "seconds": dt}


def reference_workload(args, pool=None):
    """The stars the reference arm samples from: a prefix of the arm's own workload (at most 400 stars)."""
    n = max(1, min(args.stars, 400))
    return make_workload_ids(args.config, np.arange(n, dtype=np.int64), pool), n


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    with mp.get_context("fork").Pool(min(cores, 16)) as pool:
        batch, n = reference_workload(args, pool)
    smp = OracleSample(batch, float(getattr(args, "ref_budget", 4.0)), cores)
    for _ in range(args.warmup):
        smp.run()
    tot_t, tot_ev = 0.0, 0.0
    for _ in range(args.steps):
        dt, ev = smp.run()
        tot_t += dt; tot_ev += ev
    val = tot_ev / tot_t
    sample = f"per step: {smp.desc}; drawn from the first {n} stars; {args.steps} steps"
    out = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
           "config": {"workload": f"config{args.config}: bounded sample of BASELINE.json configs[{args.config - 1}] "
                                  f"({sample})", **({"grid": GRID_NOTE} if GRID_KW else {})},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": ORACLE_KIND, "note": ORACLE_NOTE,
                            "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    emit(json.dumps(out))


# ---------------------------------------------------------------------------------------------- the CUDA path
def aggregate_over_ranks(maxes, sums, world: int, device: str):
    """Whole-job figures: times = MAX over ranks, work = SUM over ranks (both all-reduces are of a few scalars)."""
    maxes, sums = [float(x) for x in maxes], [float(x) for x in sums]
    if world <= 1:
        return maxes, sums
    import torch
    import torch.distributed as dist
    mx = torch.tensor(maxes, dtype=torch.float64, device=device)
    sm = torch.tensor(sums, dtype=torch.float64, device=device)
    dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    dist.all_reduce(sm, op=dist.ReduceOp.SUM)
    return [float(x) for x in mx], [float(x) for x in sm]


def deal_stars_by_cost(config: int, n_per_rank: int, rank: int, world: int, pool, ctx, device: str):
    """every rank measures the cost N_pts x n_freq of its contiguous slice of star ids with a device
    grid pass over the timestamps alone, the costs are all-gathered (world x n_per_rank doubles), and every rank
    computes the same longest-processing-time partition.  -> (my star ids, info dict)."""
    import torch
    import torch.distributed as dist
    from paper_2302_01293_b200 import bls, shard
    mine = shard_star_ids(n_per_rank, rank)
    row_ptr, t, rho = make_times_ids(config, mine, pool)
    f = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(device)
    grid, _, _, _ = ctx.grid(f(row_ptr, np.int64), f(t, np.float64), f(rho, np.float64), None)
    g = bls.grid_to_numpy(grid)
    cost = (g["n_freq"].astype(np.float64) * np.diff(row_ptr)).astype(np.float64)
    allc = torch.empty(world * n_per_rank, dtype=torch.float64, device=device)
    dist.all_gather_into_tensor(allc, torch.from_numpy(cost).to(device))
    allc = allc.cpu().numpy()
    parts = shard.lpt_partition(allc, world)
    contiguous = [np.arange(r * n_per_rank, (r + 1) * n_per_rank) for r in range(world)]
    info = {"policy": "longest-processing-time greedy on N_pts x n_freq (device grid pass over the timestamps)",
            "max_over_mean_cost": shard.imbalance(allc, parts),
            "max_over_mean_cost_contiguous": shard.imbalance(allc, contiguous),
            "stars_per_rank": [int(p.size) for p in parts]}
    return parts[rank], info


def run_gpu(args):
    import multiprocessing as mp
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    n_workers = max(1, min((os.cpu_count() or 1) // max(world, 1), 16))
    pool = mp.get_context("fork").Pool(n_workers)      # forked before the CUDA context exists
    import torch
    import torch.distributed as dist
    from paper_2302_01293_b200 import build, bls, shard
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the QLP BLS path has no CPU fallback)")
    use_dist = world > 1 or os.environ.get("QLP_BENCH_FORCE_DIST") == "1"  # the latter: exercise NCCL at world 1
    device = f"cuda:{local}"
    if use_dist:
        if "RANK" not in os.environ:   # QLP_BENCH_FORCE_DIST outside torchrun: a one-rank group on this host
            os.environ.update(RANK="0", WORLD_SIZE="1", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1",
                              MASTER_PORT=os.environ.get("MASTER_PORT", "29533"))
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if use_dist:
        dist.barrier()
    torch.cuda.set_device(local)
    ctx = bls.QlpBls(device=local, top_k=3, **GRID_KW)
    K = ctx.top_k
    # stars are independent: each rank searches its own shard, no data-path collective
    n_global = world * args.stars
    if world > 1:
        my_ids, shard_info = deal_stars_by_cost(args.config, args.stars, rank, world, pool, ctx, device)
    else:
        my_ids, shard_info = shard_star_ids(args.stars, 0), {"policy": "one rank: all stars"}
    g0 = time.perf_counter()
    batch = make_workload_ids(args.config, my_ids, pool)
    gen_s = time.perf_counter() - g0
    pool.close()
    dev = bls.upload(batch, device)
    row_ptr, t, y, dy, rho, rstar = dev
    S = batch.n_stars
    # the one collective of a job: the per-star peak table of every rank, one all-gather per step
    hdr = torch.from_numpy(shard.pack_rows(np.zeros((S, 0), dtype=np.uint8), my_ids)).to(device)
    n_max = shard.max_rows_over_ranks(S, device)
    recv = torch.empty((world, n_max, 16 + K * bls.PEAK_DTYPE.itemsize), dtype=torch.uint8, device=device)

    def step():
        grid, freq_ptr, tf, tb = ctx.grid(row_ptr, t, rho, rstar)
        step.total_bins = tb
        sr, best = ctx.spectrum(row_ptr, t, y, dy, grid, freq_ptr, tf)
        _, peaks = ctx.snr(row_ptr, t, y, dy, grid, freq_ptr, sr, best, want_snr=False)
        ctx.peak_stats(row_ptr, t, y, dy, peaks)  # O7, the first row after the search
        if use_dist:
            shard.gather_rows(torch.cat([hdr, peaks.view(S, -1)], dim=1), n_max, out=recv)
        return grid, peaks, tf

    grid, peaks, tf = step()
    g = bls.grid_to_numpy(grid)
    evals = int((g["n_freq"] * np.diff(batch.row_ptr)).sum())
    for _ in range(max(args.warmup - 1, 0)):
        step()
    torch.cuda.synchronize()

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    ctx.fold_timing(True)
    barrier()
    if rank == 0:
        sampler.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        grid, peaks, tf = step()
    e1.record()
    barrier()
    launches = ctx.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    n_timed, fold_ms = ctx.fold_elapsed_ms()
    cc = ctx.fold_class_counters().astype(np.float64)
    ph = [float(cc[:, i].sum()) for i in range(3)]
    ctx.fold_timing(False)
    table = None
    if use_dist and rank == 0:
        table = shard.unpack_rows(recv.cpu().numpy(), n_global, bls.PEAK_DTYPE, (K,))

    # the rows after the search, measured on their own: not part of `value`
    n_small = max(1, min(args.steps, 5))
    ctx.trapezoid_fit(row_ptr, t, y, dy, peaks)
    torch.cuda.synchronize()
    ctx.fold_timing(True)    # also makes the fit kernels count their (point, sweep) pairs
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(n_small):
        fits = ctx.trapezoid_fit(row_ptr, t, y, dy, peaks)
    f1.record()
    torch.cuda.synchronize()
    fit_ms = f0.elapsed_time(f1) / n_small
    fit_pairs = ctx.fit_work() / n_small
    ctx.fold_timing(False)
    fit_np = bls.fits_to_numpy(fits, K)
    ctx.pink_noise(row_ptr, t, y, peaks, fits)
    f0.record()
    for _ in range(n_small):
        pink = ctx.pink_noise(row_ptr, t, y, peaks, fits)   # O9
    f1.record()
    torch.cuda.synchronize()
    pink_ms = f0.elapsed_time(f1) / n_small
    pink_np = bls.pink_to_numpy(pink, K)

    # end to end through the host-buffer API: pinned host inputs, H2D and D2H inside the timed region
    del dev, row_ptr, t, y, dy, grid, peaks, fits, pink
    torch.cuda.empty_cache()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    h = [pin(batch.row_ptr), pin(batch.t), pin(batch.y), pin(batch.dy), pin(batch.rho)]
    ctx.search_host(*h, want_stats=True)   # untimed: staging buffers of the full size, streams
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_small):
        pk_host, st_host, _, _ = ctx.search_host(*h, want_stats=True)
        if use_dist:   # the job's result is the gathered table here too
            shard.gather_rows(torch.cat([hdr, torch.from_numpy(pk_host.view(np.uint8).reshape(S, -1)).to(device)],
                                        dim=1), n_max, out=recv)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / n_small
    h2d = int(sum(a.nbytes for a in h))
    d2h = int(pk_host.nbytes + st_host.nbytes)
    ctx.vet_host(*h)                       # untimed: the fit workspace of the full size
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_small):
        vet = ctx.vet_host(*h)
    torch.cuda.synchronize()
    vet_s = (time.perf_counter() - t0) / n_small
    d2h_vet = int(sum(a.nbytes for a in vet))
    detected = int((vet[3]["detected"].max(axis=1) > 0).sum())

    (ms, e2e_ms, vet_ms), (evals_all, stars_all) = aggregate_over_ranks(
        [ms, e2e_s * 1e3, vet_s * 1e3], [evals, S], world if use_dist else 1, device)
    if rank != 0:
        if use_dist:
            dist.destroy_process_group()
        return
    peaks_info, src = _peaks()
    sm_max = float(peaks_info.get("sm_max_mhz", 1965.0))
    fold_per_launch_s = (fold_ms / max(n_timed, 1)) * 1e-3
    achieved = evals / fold_per_launch_s if fold_per_launch_s > 0 else 0.0
    peak = fold_peak_evals_per_s(sm_max)
    per_clk_peak = min(ATOMS_LANES_PER_CLK_SM / 2.0, FP64_LANES_PER_CLK_SM / 3.0)
    # per tile class: thread-0 SM clocks summed over CTAs (class 0 runs two CTAs per SM, the others one) and the
    # evaluations its tiles made -> share of the SM time and evaluations per SM clock, independent of the overlap
    sm_clk = np.array([(cc[c, 0] + cc[c, 1] + cc[c, 2]) / (2.0 if c == 0 else 1.0) for c in range(9)])
    classes = {}
    for c in range(9):
        if cc[c, 4] > 0:
            per_clk = cc[c, 3] / sm_clk[c] if sm_clk[c] > 0 else 0.0
            classes[str(c)] = {"columns": CLASS_COLS[c], "nb_max": CLASS_NBCAP[c],
                               "share_of_sm_time": float(sm_clk[c] / sm_clk.sum()),
                               "share_of_evals": float(cc[c, 3] / max(cc[:, 3].sum(), 1.0)),
                               "evals_per_clk_sm": float(per_clk), "frac": float(per_clk / per_clk_peak),
                               "scan_share": float(cc[c, 2] / max(cc[c, :3].sum(), 1.0))}
    n_points, n_freq = int(batch.n_points), int(tf)
    traffic = NCU_TRAFFIC.get((args.config, args.stars)) if world == 1 and not GRID_KW else None
    out = {
        "metric": METRIC, "value": evals_all * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
        "config": {"workload": f"config{args.config}: BASELINE.json configs[{args.config - 1}], "
                               + (f"first {args.stars} of 200000 stars" if args.config == 5 else f"{args.stars} stars")
                               + f" per GPU; rank 0: {n_points} points, {n_freq} frequencies",
                   "l2": "inputs larger than L2 (no flush needed)" if batch.n_points * 24 > 126e6 else
                         "inputs smaller than L2",
                   "parallelism": f"stars sharded over {world} GPU(s); the only collective is the all-gather of the "
                                  "peak table" if use_dist else "one GPU",
                   "shard": shard_info, "generation_s": gen_s,
                   **({"grid": GRID_NOTE} if GRID_KW else {})},
        "stars_per_s": stars_all * args.steps / (ms * 1e-3),
        "clocks": clocks,
        "e2e": {"value": evals_all / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "stars_per_s": stars_all / (e2e_ms * 1e-3), "steps": n_small,
                "call": "qlp_bls_search_host (pinned host buffers; peaks + statistics back)"},
        "e2e_vet": {"value": evals_all / (vet_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h_vet, "stars_per_s": stars_all / (vet_ms * 1e-3), "steps": n_small,
                    "detected_stars_rank0": detected,
                    "call": "qlp_bls_vet_host (search + trapezoid fit + noise / detection row, PAPER.md:44-55)"},
        "gpu_launches": int(launches),
        # rank 0's shard, outside the timed region of `value`: count + scan + fit kernels of qlp_bls_trapezoid_fit
        "trapezoid_fit": {"ms_per_call": fit_ms, "fits": int(fit_np.size), "fits_per_s": fit_np.size / (fit_ms * 1e-3),
                          "mean_points_per_fit": float(fit_np["n_fit"].mean()),
                          "mean_chi2_evaluations": float(fit_np["n_eval"].mean()),
                          "chi2_evaluations_p50_p90_max": [float(np.percentile(fit_np["n_eval"], 50)),
                                                           float(np.percentile(fit_np["n_eval"], 90)),
                                                           float(fit_np["n_eval"].max())],
                          "points_per_fit_p50_p90_max": [float(np.percentile(fit_np["n_fit"], 50)),
                                                         float(np.percentile(fit_np["n_fit"], 90)),
                                                         float(fit_np["n_fit"].max())],
                          # Algorithmic work of O8: one trapezoid evaluation = one (point inside the transit, candidate)
                          # pair = 8 FP64 instructions (|dt - c|, half - u, x inv_ing, min, w sh, three accumulations);
                          # the kernels count the (point, sweep) pairs, each is six evaluations.  Bound: the FP64 pipe.
                          "roofline": {"bound": "alu", "unit": "G trapezoid evaluations/s",
                                       "achieved": 6.0 * fit_pairs / (fit_ms * 1e-3) / 1e9,
                                       "peak": N_SM * sm_max * 1e6 * FP64_LANES_PER_CLK_SM / 8.0 / 1e9,
                                       "frac": 6.0 * fit_pairs / (fit_ms * 1e-3) /
                                               (N_SM * sm_max * 1e6 * FP64_LANES_PER_CLK_SM / 8.0),
                                       "evaluations_per_call": 6.0 * fit_pairs,
                                       "note": "latency-bound: ~90 serial sweeps per fit (pass, 18 reductions, solve, "
                                               "decision), DESIGN.md section 4 O8"}},
        "pink_noise": {"ms_per_call": pink_ms, "detected_stars": int((pink_np["detected"].max(axis=1) > 0).sum())},
        "roofline": {"bound": "alu", "kernel": "foldscan_kernel (9 class launches per step)",
                     "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "Gevals/s",
                     "frac": achieved / peak if peak > 0 else None,
                     # thread-0 SM clocks per phase of the fused kernel, summed over all tiles of the timed steps
                     "phase_share": {"setup_zero": ph[0] / max(sum(ph), 1), "fold_S2": ph[1] / max(sum(ph), 1),
                                     "scan_S3": ph[2] / max(sum(ph), 1)},
                     "fold_only_achieved": achieved / 1e9 / max(ph[1] / max(sum(ph), 1), 1e-9),
                     # S3 inside the fused kernel: (start bin, width) candidates per second over the scan's share of
                     # the kernel time, against the issue / MUFU bound of its 8-instruction candidate test
                     "scan_S3": scan_roofline(step.total_bins, ctx.widths().size, fold_per_launch_s,
                                              ph[2] / max(sum(ph), 1), sm_max),
                     "classes": classes,
                     "issue_bound": fold_issue_bound_evals_per_s(sm_max) / 1e9,
                     "frac_of_issue_bound": achieved / fold_issue_bound_evals_per_s(sm_max),
                     # measured DRAM bytes of the foldscan launches of one step, from an ncu capture of THIS workload
                     # kept under profiles/ (null if there is none), next to the method's compulsory bytes
                     "traffic": traffic[0] if traffic else None,
                     "traffic_source": (traffic[1] + "; a constant from that capture, not measured in this run")
                                       if traffic else None,
                     "compulsory_bytes_per_step": 16 * n_points + 8 * n_freq,
                     "compulsory_bytes_note": "16 B per point record read once + 8 B per frequency (SR + best) written",
                     "share_of_step": fold_ms / max(n_timed, 1) / (ms / args.steps),
                     "peak_source": f"148 SMs x {sm_max:.0f} MHz ({src}) x min(ATOMS lanes/2, FP64 lanes/3) per clk "
                                    "(profiles/ubench_r1.txt; DESIGN.md Roofline)"},
    }
    if table is not None:
        out["gathered_peak_table"] = {"stars": int(table.shape[0]), "bytes_per_rank_per_step": int(recv[0].numel()),
                                      "top_peaks_with_snr_gt_9": int((table[:, 0]["snr"] > 9.0).sum())}
    if world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(batch)
    emit(json.dumps(out))
    if use_dist:
        dist.destroy_process_group()


def run_full(args):
    """--chunk C: the whole batch of --stars stars (config 5: 200,000, north_star's target) searched in chunks of C
    stars.  Chunks are generated on the host cores OUTSIDE the timed regions (no host holds the 100 GB batch at
    once); each chunk is searched once from device-resident inputs (CUDA events -> `value`) and once through
    qlp_bls_search_host from pinned host buffers (-> `e2e`); times and work are summed over the chunks."""
    import multiprocessing as mp
    import torch
    from paper_2302_01293_b200 import build, bls
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the QLP BLS path has no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("bench.py --chunk: one GPU only (shard --stars over ranks instead)")
    build.build()
    pool = mp.get_context("fork").Pool(os.cpu_count() or 1)   # forked before the CUDA context exists
    torch.cuda.set_device(0)
    ctx = bls.QlpBls(device=0, top_k=3, **GRID_KW)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    tot = {"ms": 0.0, "e2e_s": 0.0, "evals": 0, "points": 0, "freqs": 0, "bins": 0, "h2d": 0, "d2h": 0,
           "launches": 0, "gen_s": 0.0}
    rec = {"injected": 0, "top_peak_at_period": 0, "top_peak_at_period_or_harmonic": 0, "snr_gt_9": 0}
    sampler = ClockSampler(0)
    sampler.start()
    first = True
    fold_ms, ph = 0.0, [0, 0, 0]
    for lo in range(0, args.stars, args.chunk):
        hi = min(lo + args.chunk, args.stars)
        g0 = time.perf_counter()
        batch = make_workload_parallel(args.config, lo, hi, pool)
        tot["gen_s"] += time.perf_counter() - g0
        row_ptr, t, y, dy, rho, rstar = bls.upload(batch, "cuda:0")

        def step():
            grid, freq_ptr, tf, tb = ctx.grid(row_ptr, t, rho, rstar)
            sr, best = ctx.spectrum(row_ptr, t, y, dy, grid, freq_ptr, tf)
            _, peaks = ctx.snr(row_ptr, t, y, dy, grid, freq_ptr, sr, best, want_snr=False)
            ctx.peak_stats(row_ptr, t, y, dy, peaks)
            return grid, peaks, tf, tb

        if first:   # warm-up steps on the first chunk (workspace growth, module load), outside the timed region
            for _ in range(args.warmup):
                step()
        ctx.fold_timing(True)   # resets the library's fold timers: the device leg of this chunk only
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        grid, peaks, tf, tb = step()
        e1.record()
        torch.cuda.synchronize()
        tot["launches"] += ctx.launch_count() - l0
        tot["ms"] += e0.elapsed_time(e1)
        fold_ms += ctx.fold_elapsed_ms()[1]
        ph = [a + b for a, b in zip(ph, ctx.fold_phase_clocks())]
        ctx.fold_timing(False)
        g = bls.grid_to_numpy(grid)
        tot["evals"] += int((g["n_freq"] * np.diff(batch.row_ptr)).sum())
        tot["points"] += int(batch.n_points); tot["freqs"] += int(tf); tot["bins"] += int(tb)
        pk = bls.peaks_to_numpy(peaks, ctx.top_k)
        del row_ptr, t, y, dy, grid, peaks
        torch.cuda.empty_cache()

        h = [pin(batch.row_ptr), pin(batch.t), pin(batch.y), pin(batch.dy), pin(batch.rho)]
        if first:   # one untimed call on the first 1,000 stars (staging buffers, streams)
            ctx.search_host(h[0][:1001], h[1], h[2], h[3], h[4][:1000], want_stats=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        pk_host, st_host, _, _ = ctx.search_host(*h, want_stats=True)
        torch.cuda.synchronize()
        tot["e2e_s"] += time.perf_counter() - t0
        tot["h2d"] += int(sum(a.nbytes for a in h)); tot["d2h"] += int(pk_host.nbytes + st_host.nbytes)
        if np.ascontiguousarray(pk_host).tobytes() != np.ascontiguousarray(pk).tobytes():
            raise SystemExit("bench.py --chunk: host-path peaks differ from the device path")
        # the S/N-detrended top peak per star against the injected period (BASELINE.json configs[4])
        top = pk[:, 0]
        inj = batch.truth["period"] > 0
        ratio = top["period"][inj] / batch.truth["period"][inj]
        near = lambda r, c: np.abs(r / c - 1.0) < 0.01
        rec["injected"] += int(inj.sum())
        rec["top_peak_at_period"] += int(near(ratio, 1.0).sum())
        rec["top_peak_at_period_or_harmonic"] += int(sum(near(ratio, c) for c in (1.0, 0.5, 2.0, 1 / 3, 3.0)).sum())
        rec["snr_gt_9"] += int((top["snr"] > 9.0).sum())
        first = False
        del h
        print(f"[bench] stars {lo}..{hi}: device {tot['ms'] * 1e-3:.1f} s, host path {tot['e2e_s']:.1f} s, "
              f"generation {tot['gen_s']:.0f} s (cumulative)", file=sys.stderr, flush=True)
    pool.close()
    clocks = sampler.stop()
    peaks_info, src = _peaks()
    sm_max = float(peaks_info.get("sm_max_mhz", 1965.0))
    achieved = tot["evals"] / (fold_ms * 1e-3)
    peak = fold_peak_evals_per_s(sm_max)
    n_chunks = -(-args.stars // args.chunk)
    out = {
        "metric": METRIC, "value": tot["evals"] / (tot["ms"] * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": 1,
        "warmup": args.warmup, "ms_per_step": tot["ms"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
        "config": {"workload": f"config{args.config}: BASELINE.json configs[{args.config - 1}], {args.stars} stars in "
                               f"{n_chunks} chunks of {args.chunk}, {tot['points']} points, {tot['freqs']} frequencies",
                   "l2": "inputs larger than L2 (no flush needed)",
                   "parallelism": "one GPU; chunks generated on the host between the timed regions "
                                  f"({tot['gen_s']:.0f} s of generation, not timed)"},
        "stars_per_s": args.stars / (tot["ms"] * 1e-3),
        "clocks": clocks,
        "e2e": {"value": tot["evals"] / tot["e2e_s"], "unit": UNIT, "h2d_bytes_per_step": tot["h2d"],
                "d2h_bytes_per_step": tot["d2h"], "stars_per_s": args.stars / tot["e2e_s"], "seconds": tot["e2e_s"],
                "peaks_bitwise_equal_to_device_path": True},
        "gpu_launches": int(tot["launches"]),
        "recovery": rec,
        "roofline": {"bound": "alu", "kernel": "foldscan_kernel", "achieved": achieved / 1e9, "peak": peak / 1e9,
                     "unit": "Gevals/s", "frac": achieved / peak,
                     "phase_share": {"setup_zero": ph[0] / max(sum(ph), 1), "fold_S2": ph[1] / max(sum(ph), 1),
                                     "scan_S3": ph[2] / max(sum(ph), 1)},
                     "scan_S3": scan_roofline(tot["bins"], ctx.widths().size, fold_ms * 1e-3,
                                              ph[2] / max(sum(ph), 1), sm_max),
                     "traffic": None, "compulsory_bytes_per_step": 16 * tot["points"] + 8 * tot["freqs"],
                     "share_of_step": fold_ms / tot["ms"],
                     "peak_source": f"148 SMs x {sm_max:.0f} MHz ({src}) x min(ATOMS lanes/2, FP64 lanes/3) per clk "
                                    "(profiles/ubench_r1.txt; DESIGN.md Roofline)"},
    }
    emit(json.dumps(out))


_REAL_STDOUT = None


def _quiet_stdout():
    """Libraries (NCCL prints its version line) may write to stdout; the driver wants exactly one JSON line there.
    File descriptor 1 is pointed at stderr for the run and the JSON line goes to the saved descriptor."""
    global _REAL_STDOUT
    sys.stdout.flush()
    _REAL_STDOUT = os.fdopen(os.dup(1), "w")
    os.dup2(2, 1)


def emit(line: str):
    out = _REAL_STDOUT or sys.stdout
    out.write(line + "\n")
    out.flush()


def respawn_under_torchrun(args):
    """`--gpus N` outside a torchrun environment: replace this process by `python -m torch.distributed.run` with N
    ranks of this same command line, one per GPU (rendezvous on 127.0.0.1)."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but {have} CUDA device(s) visible (one rank per GPU; ranks are "
                         "never stacked on one GPU)")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.stdout.flush(); sys.stderr.flush()
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, help="BASELINE.json configs[config-1]")
    ap.add_argument("--stars", type=int, default=None, help="stars per GPU (default: 4000 for config 5, else the "
                                                            "config's own size up to 1000)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--chunk", type=int, default=0,
                    help="search --stars stars in chunks of this many (one GPU; e.g. --config 5 --stars 200000 "
                         "--chunk 20000 is the whole production-shaped batch)")
    ap.add_argument("--comparison-grid", action="store_true",
                    help="search the comparison grid of DESIGN.md O1.10 (PAPER.md:13: periods up to 56 d, at most "
                         "80,000 frequencies per star) instead of the paper's GPU grid")
    ap.add_argument("--comparison-grid-uniform", action="store_true",
                    help="the same caps on a grid with equal steps in FREQUENCY (DESIGN.md O1.10c: the comparison "
                         "workload as SURVEY.md 8(f) words it)")
    ap.add_argument("--ref-budget", type=float, default=4.0, help="--impl reference: seconds of oracle work per step")
    args = ap.parse_args()
    if args.stars is None:
        from paper_2302_01293_b200 import synth
        args.stars = DEFAULT_STARS if args.config == 5 else min(synth.N_STARS[args.config], 1000)
    if args.comparison_grid or args.comparison_grid_uniform:
        GRID_KW.update(max_period_days=56.0, max_freq=80000)
    if args.comparison_grid_uniform:
        global GRID_NOTE
        GRID_KW.update(uniform_freq=1)
        GRID_NOTE = ("comparison grid O1.10c (PAPER.md:13; SURVEY.md 8(f) f4): equal steps in frequency, P <= 56 d, "
                     "<= 80,000 frequencies per star")
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.chunk == 0:
        respawn_under_torchrun(args)
    _quiet_stdout()
    if args.impl == "reference":
        run_reference(args)
    elif args.chunk > 0:
        run_full(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
