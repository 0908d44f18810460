#!/usr/bin/env python
"""bench.py -- throughput of the QLP BLS hot path (S0..S4) on synthetic TESS-shaped light curves.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C] [--stars S]

One "step" = one pass of the whole hot path (grid -> prep -> fold+box-scan -> S/N + peaks -> peak statistics) over one
batch.  Default workload = BASELINE.json configs[1] ("config 2": 1,000 stars, one sector at 200 s
cadence, ~11.4k points and ~4.5k-10k frequencies per star).  Prints ONE JSON line (rank 0).

  value     : point x frequency BLS evaluations per second, whole job, inputs resident in HBM
  e2e       : the same metric through qlp_bls_search_host with pinned HOST buffers (H2D + D2H inside)
  roofline  : fold+box-scan launches, CUDA-event timed inside the timed region, against the
              shared-memory-atomic issue ceiling derived in DESIGN.md ("bound": "alu")
  cpu_baseline : oracle/ timed on this box's host cores on a bounded sample (N=1, rank 0 only)

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
# per evaluation the fold needs 2 shared-memory integer atomic lanes and 3 FP64
# lanes (the exact bin takes three FP64 instructions); measured ceilings on B200 (profiles/ubench_r1.txt):
# ATOMS.ADD lanes/clk/SM and FP64 lanes/clk/SM.  The binding one is the atomic path.
ATOMS_LANES_PER_CLK_SM = 31.6
FP64_LANES_PER_CLK_SM = 62.3
N_SM = 148
NCU_DRAM_BYTES_PER_STEP = 719.3e6  # 676.8 MB read + 42.5 MB written, profiles/r1_foldscan_ncu.txt


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


def make_workload(config: int, n_stars: int, rank: int):
    """Seeded synthetic batch; rank r takes star ids [r*n, (r+1)*n)."""
    from paper_2302_01293_b200 import synth
    return synth.make_batch(config, star_ids=shard_star_ids(n_stars, rank))


def oracle_evals(orc, cfg, batch):
    """Fold evaluations (points x frequencies) the oracle performs on this batch."""
    tot = 0
    for s in range(batch.n_stars):
        t, _, _ = batch.star(s)
        g = orc.grid(cfg, t, float(batch.rho[s]))
        tot += int(g["n_freq"]) * t.size
    return tot


GRID_NOTE = "comparison grid O1.10 (PAPER.md:13): P <= 56 d, <= 80,000 frequencies per star"
GRID_KW = {}   # --comparison-grid: the O1.10 caps, given to both the CUDA context and the oracle config


def time_oracle(batch, n_stars: int, threads: int):
    """Run the oracle as it stands (OpenMP over stars) on the first n_stars -> (seconds, evals)."""
    from oracle import oracle as orc
    from paper_2302_01293_b200 import synth
    cfg = orc.default_config(**GRID_KW)
    sub = synth.from_arrays([batch.star(s) for s in range(n_stars)], rho=batch.rho[:n_stars])
    ev = oracle_evals(orc, cfg, sub)
    t0 = time.perf_counter()
    orc.batch(cfg, sub.row_ptr, sub.t, sub.y, sub.dy, sub.rho, K=3, want_snr=True, threads=threads)
    return time.perf_counter() - t0, ev


def cpu_baseline(batch, budget_s: float = 15.0):
    cores = os.cpu_count() or 1
    from oracle import oracle as orc
    orc.build()
    n0 = min(batch.n_stars, cores)
    dt0, ev0 = time_oracle(batch, n0, cores)
    n1 = int(min(batch.n_stars, max(n0, n0 * budget_s / max(dt0, 1e-3))))
    if n1 > n0:
        dt, ev = time_oracle(batch, n1, cores)
    else:
        dt, ev, n1 = dt0, ev0, n0
    return {"value": ev / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n1} stars of the workload, whole path (grid+SR+S/N+peaks), {dt:.1f} s",
            "stars_per_s": n1 / dt}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import oracle as orc
    orc.build()
    cores = os.cpu_count() or 1
    n = max(1, min(args.stars, 2 * cores))
    batch = make_workload(args.config, n, 0)
    for _ in range(args.warmup):
        time_oracle(batch, min(n, cores), cores)
    tot_t, tot_ev = 0.0, 0
    for _ in range(args.steps):
        dt, ev = time_oracle(batch, n, cores)
        tot_t += dt; tot_ev += ev
    val = tot_ev / tot_t
    out = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
           "config": {"workload": f"config{args.config}: {n}-star sample of BASELINE.json configs[{args.config - 1}]",
                      **({"grid": GRID_NOTE} if GRID_KW else {})},
           "stars_per_s": n * args.steps / tot_t,
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{n} stars per step, {args.steps} steps"},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    emit(json.dumps(out))


def shard_star_ids(n_stars_per_gpu: int, rank: int) -> np.ndarray:
    """Stars are independent: rank r searches ids [r*n, (r+1)*n); no data-path collective."""
    return np.arange(rank * n_stars_per_gpu, (rank + 1) * n_stars_per_gpu, dtype=np.int64)


def aggregate_over_ranks(ms: float, e2e_ms: float, evals: int, stars: int, world: int, device: str):
    """Whole-job figures: time = MAX over ranks, work = SUM over ranks (the only collective of the run)."""
    if world <= 1:
        return ms, e2e_ms, float(evals), float(stars)
    import torch
    import torch.distributed as dist
    v = torch.tensor([ms, e2e_ms, float(evals), float(stars)], dtype=torch.float64, device=device)
    mx = v.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    sm = v.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
    return float(mx[0]), float(mx[1]), float(sm[2]), float(sm[3])


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2302_01293_b200 import build, bls
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the QLP BLS path has no CPU fallback)")
    use_dist = world > 1 or os.environ.get("QLP_BENCH_FORCE_DIST") == "1"  # the latter: exercise NCCL at world 1
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if use_dist:
        dist.barrier()
    torch.cuda.set_device(local)
    ctx = bls.QlpBls(device=local, top_k=3, **GRID_KW)
    # stars are independent: each rank searches its own shard, no data-path collective
    batch = make_workload(args.config, args.stars, rank)
    dev = bls.upload(batch, f"cuda:{local}")
    row_ptr, t, y, dy, rho, rstar = dev
    S = batch.n_stars

    def step():
        grid, freq_ptr, tf, tb = ctx.grid(row_ptr, t, rho, rstar)
        step.total_bins = tb
        sr, best = ctx.spectrum(row_ptr, t, y, dy, grid, freq_ptr, tf)
        _, peaks = ctx.snr(row_ptr, t, y, dy, grid, freq_ptr, sr, best, want_snr=False)
        ctx.peak_stats(row_ptr, t, y, dy, peaks)  # O7, the first row after the search
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
        step()
    e1.record()
    barrier()
    launches = ctx.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    n_timed, fold_ms = ctx.fold_elapsed_ms()
    ph = ctx.fold_phase_clocks()
    ctx.fold_timing(False)

    # the row after the search, measured on its own: it is not part of `value`
    ctx.trapezoid_fit(row_ptr, t, y, dy, peaks)
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(args.steps):
        fits = ctx.trapezoid_fit(row_ptr, t, y, dy, peaks)
    f1.record()
    torch.cuda.synchronize()
    fit_ms = f0.elapsed_time(f1) / args.steps
    fit_np = bls.fits_to_numpy(fits, ctx.top_k)
    ctx.pink_noise(row_ptr, t, y, peaks, fits)
    f0.record()
    for _ in range(args.steps):
        pink = ctx.pink_noise(row_ptr, t, y, peaks, fits)   # O9
    f1.record()
    torch.cuda.synchronize()
    pink_ms = f0.elapsed_time(f1) / args.steps
    pink_np = bls.pink_to_numpy(pink, ctx.top_k)

    # end to end through the host-buffer API: pinned host inputs, H2D and D2H inside the timed region
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    h = [pin(batch.row_ptr), pin(batch.t), pin(batch.y), pin(batch.dy), pin(batch.rho)]
    ctx.search_host(*h, want_stats=True)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pk_host, st_host, _, _ = ctx.search_host(*h, want_stats=True)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    h2d = int(sum(a.nbytes for a in h))
    d2h = int(pk_host.nbytes + st_host.nbytes)

    ms, e2e_ms, evals_all, stars_all = aggregate_over_ranks(ms, e2e_s * 1e3, evals, S, 2 if use_dist else 1,
                                                            f"cuda:{local}")
    if rank != 0:
        if use_dist:
            dist.destroy_process_group()
        return
    peaks_info, src = _peaks()
    sm_max = float(peaks_info.get("sm_max_mhz", 1965.0))
    fold_per_launch_s = (fold_ms / max(n_timed, 1)) * 1e-3
    achieved = evals / fold_per_launch_s if fold_per_launch_s > 0 else 0.0
    peak = fold_peak_evals_per_s(sm_max)
    out = {
        "metric": METRIC, "value": evals_all * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 phase / int32 fixed-point accumulators / f32 box scan",
        "data": "synthetic",
        "config": {"workload": f"config{args.config}: BASELINE.json configs[{args.config - 1}], {S} stars per GPU, "
                               f"{int(batch.n_points)} points, {int(tf)} frequencies",
                   "l2": "inputs larger than L2 (no flush needed)" if batch.n_points * 24 > 126e6 else
                         "inputs smaller than L2", "parallelism": f"stars sharded over {world} GPU(s), no collective",
                   **({"grid": GRID_NOTE} if GRID_KW else {})},
        "stars_per_s": stars_all * args.steps / (ms * 1e-3),
        "clocks": clocks,
        "e2e": {"value": evals_all * args.steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "stars_per_s": stars_all * args.steps / (e2e_ms * 1e-3)},
        "gpu_launches": int(launches),
        # rank 0's shard, outside the timed region of `value`: count + scan + fit kernels of qlp_bls_trapezoid_fit
        "trapezoid_fit": {"ms_per_call": fit_ms, "fits": int(fit_np.size), "fits_per_s": fit_np.size / (fit_ms * 1e-3),
                          "mean_points_per_fit": float(fit_np["n_fit"].mean()),
                          "mean_chi2_evaluations": float(fit_np["n_eval"].mean())},
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
                     "issue_bound": fold_issue_bound_evals_per_s(sm_max) / 1e9,
                     "frac_of_issue_bound": achieved / fold_issue_bound_evals_per_s(sm_max),
                     # dram__bytes_read+write of the foldscan launches of one step of THIS workload
                     # (profiles/r1_foldscan_ncu.txt); valid for the default config-2 / 1000-star run only
                     "traffic": NCU_DRAM_BYTES_PER_STEP if (args.config == 2 and args.stars == 1000) else None,
                     "traffic_unit": "bytes per step (ncu dram read+write over the foldscan launches); algorithmic: "
                                     f"{4 * 16 * int(batch.n_points) + 8 * int(tf)} (points read once per tile class + SR/best)",
                     "share_of_step": fold_ms / max(n_timed, 1) / (ms / args.steps),
                     "peak_source": f"148 SMs x {sm_max:.0f} MHz ({src}) x min(ATOMS lanes/2, FP64 lanes/3) per clk "
                                    "(profiles/ubench_r1.txt; DESIGN.md Roofline)"},
    }
    if world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(batch)
    emit(json.dumps(out))
    if use_dist:
        dist.destroy_process_group()


def _gen_block(job):
    from paper_2302_01293_b200 import synth
    config, lo, hi = job
    b = synth.make_batch(config, star_ids=np.arange(lo, hi, dtype=np.int64))
    return b.row_ptr, b.t, b.y, b.dy, b.rho, b.rstar, b.truth


def make_workload_parallel(config: int, lo: int, hi: int, pool, block: int = 250):
    """Stars [lo, hi) of a config, generated by the worker pool in blocks of stars (every star has its own seed,
    paper_2302_01293_b200.synth), packed into one CSR batch."""
    from paper_2302_01293_b200 import synth
    parts = pool.map(_gen_block, [(config, a, min(a + block, hi)) for a in range(lo, hi, block)])
    sizes = np.concatenate([np.diff(p[0]) for p in parts])
    row_ptr = np.zeros(sizes.size + 1, dtype=np.int64)
    np.cumsum(sizes, out=row_ptr[1:])
    cat = lambda k: np.concatenate([p[k] for p in parts])
    return synth.Batch(config, 0, np.arange(lo, hi, dtype=np.int64), row_ptr, cat(1), cat(2), cat(3), cat(4), cat(5),
                       cat(6))


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
        "vs_baseline": None, "dtype": "f64 phase / int32 fixed-point accumulators / f32 box scan", "data": "synthetic",
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
                     "traffic": None, "share_of_step": fold_ms / tot["ms"],
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[config-1]")
    ap.add_argument("--stars", type=int, default=1000, help="stars per GPU")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--chunk", type=int, default=0,
                    help="search --stars stars in chunks of this many (one GPU; e.g. --config 5 --stars 200000 "
                         "--chunk 20000 is the whole production-shaped batch)")
    ap.add_argument("--comparison-grid", action="store_true",
                    help="search the comparison grid of DESIGN.md O1.10 (PAPER.md:13: periods up to 56 d, at most "
                         "80,000 frequencies per star) instead of the paper's GPU grid")
    args = ap.parse_args()
    if args.comparison_grid:
        GRID_KW.update(max_period_days=56.0, max_freq=80000)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    _quiet_stdout()
    if args.impl == "reference":
        run_reference(args)
    elif args.chunk > 0:
        run_full(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
