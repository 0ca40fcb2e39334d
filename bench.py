#!/usr/bin/env python
"""bench.py -- the batched SuperSmoother periodogram on BASELINE.json's 10,000-object config.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mode cv|gv]

A step = one pass of the whole hot path (prep, fold, sort, smoother, statistic, argmax) over the whole
synthetic catalog of config 3 (10,000 objects, n ~ U[50,200], 50,000 frequencies on [0.5, 24) 1/d),
cross-validation mode, periodogram materialised (4 GB) plus best frequency per object.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
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

import ss_inputs  # noqa: E402

METRIC = "object_frequency_evals_per_second"
UNIT = "evals/s"

# Algorithmic on-chip traffic per point-eval: prefix arrays written once + window-end
# reads, 8 B each: 15 + 50 words (CV), 6 + 30 (GV).  The shared-memory / LSU data pipe is the unit that binds the
# eval kernels (ncu: l1tex__data_pipe_lsu_wavefronts 77-83 % of peak, fp64 pipe 37-44 %), so this is `roofline`.
SMEM_BYTES_PER_POINT_EVAL = {"cv": 520.0, "gv": 288.0}
# Secondary: fp64 pipe lane-instructions ("slots") per point-eval.  SURVEY.md 8(d) counts 133 add/mul/fma + 10 div/sqrt at
# 8 slots each (CV), 85 + 10 (GV); the kernels pay less for a division (MUFU seed + 3 DFMA + the multiply = 4 slots) and
# a square root (MUFU seed + 6 DFMA = 7 slots), reported beside it as "as implemented".
SLOTS_PER_POINT_EVAL = {"cv": 213.0, "gv": 165.0}
SLOTS_AS_IMPLEMENTED = {"cv": 133.0 + 10 * 4.0, "gv": 85.0 + 7 * 4.0 + 3 * 7.0}
FLOP_PER_POINT_EVAL = {m: 2.0 * s for m, s in SLOTS_PER_POINT_EVAL.items()}
# HBM traffic of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full):
# read from the committed summary of the capture taken at the commit it names, never a literal here.
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r2_traffic.json")
FP64_LANES_PER_SM = 64          # B200 fp64 pipe: 64 FMA lanes per SM per clock
N_SM = 148


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="cv", choices=["cv", "gv"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5],
                    help="another BASELINE.json config (profiles/r2_bench_configs.md); the bench line proper is config 3")
    ap.add_argument("--objects", type=int, default=None, help="(debug) fewer objects than the config has (configs 3, 4)")
    ap.add_argument("--freqs", type=int, default=None, help="(debug) fewer frequencies than the config has")
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="mixed = the paper's FP32 switch as built here (fp32 smoother for n <= 3,584; never the headline)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "500",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        """The timed region starts now: only samples taken from here on are reported.  (nvidia-smi is started
        before the warm-up because its own start-up stalls CUDA calls for a few hundred milliseconds.)"""
        self.t_mark = time.time()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, r in self.rows:
            if ts < getattr(self, "t_mark", 0.0):
                continue
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def make_catalog(args, rank):
    """Rank r times its own catalog of config 3's shape, seed 2 + r."""
    cfg = getattr(args, "config", 3)
    if cfg == 3:
        return ss_inputs.config3(seed=2 + rank, n_objects=args.objects or 10000, n_freq=args.freqs or 50000)
    if cfg == 4:
        return ss_inputs.config4(seed=3 + rank, n_objects=args.objects or 1000, n_freq=args.freqs or 500000)
    cat = ss_inputs.make(cfg)
    return cat.with_grid(n_freq=args.freqs) if args.freqs else cat


def max_over_ranks(x: float, dist=None, device=None) -> float:
    """The slowest rank's figure (the only collective of the bench: all-reduce MAX of one double)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world: int, units_per_rank_step: int, steps: int, elapsed_ms_max: float) -> float:
    """Whole-job units/s: every rank processed units_per_rank_step per step in the slowest rank's time."""
    return world * units_per_rank_step * steps / (elapsed_ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------
def cpu_baseline(cat, mode, budget_s=15.0):
    """The oracle as it stands (fast variant, OpenMP over objects), on a bounded sample of the same
    catalog: every (n_objects/m)-th object, all frequencies.  evals/s on the host cores."""
    import oracle
    omode = oracle.CV if mode == "cv" else oracle.GV
    cores = oracle.max_threads()
    # calibrate on 2*cores objects x 256 frequencies
    m0 = min(cat.n_objects, 2 * cores)
    sub = cat.subset(np.linspace(0, cat.n_objects - 1, m0).astype(int))
    t0 = time.perf_counter()
    oracle.periodogram(sub.times, sub.mags, sub.errs, sub.offsets, cat.f_min, cat.f_max, cat.n_freq,
                       mode=omode, variant=oracle.FAST, k_count=min(256, cat.n_freq))
    rate = m0 * min(256, cat.n_freq) / (time.perf_counter() - t0)
    m = int(max(cores, min(cat.n_objects, budget_s * rate / cat.n_freq)))
    m = max(1, min(m, cat.n_objects))
    sub = cat.subset(np.linspace(0, cat.n_objects - 1, m).astype(int))
    t0 = time.perf_counter()
    oracle.periodogram(sub.times, sub.mags, sub.errs, sub.offsets, cat.f_min, cat.f_max, cat.n_freq,
                       mode=omode, variant=oracle.FAST)
    dt = time.perf_counter() - t0
    return {"value": m * cat.n_freq / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{m} of {cat.n_objects} objects (evenly spaced), all {cat.n_freq} frequencies, "
                      f"{mode} mode, fast oracle variant, {dt:.1f} s"}, dt, m


def run_reference(args):
    rank, world, local = dist_env()
    if rank != 0:
        return
    cat = make_catalog(args, 0)
    import oracle
    times = []
    info = None
    for s in range(args.warmup + args.steps):
        info, dt, m = cpu_baseline(cat, args.mode, budget_s=8.0)
        if s >= args.warmup:
            times.append((dt, m))
    tot_t = sum(t for t, _ in times)
    tot_e = sum(m for _, m in times) * cat.n_freq
    val = tot_e / tot_t
    info["value"] = val
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, len(times)),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": f"config{args.config}: {cat.n_objects} objects x {cat.n_freq} frequencies, {args.mode}",
                      "sampled": True},
           "cpu_baseline": info,
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_2111_07396_b200 as ss

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    use_dist = world > 1
    if use_dist:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    ss.load()
    cat = make_catalog(args, rank)
    mode = ss.CROSS_VALIDATION if args.mode == "cv" else ss.GENERALIZED_VALIDATION
    n_obj, n_freq = cat.n_objects, cat.n_freq
    evals_per_step = n_obj * n_freq
    point_evals_per_step = int(cat.n_points) * n_freq

    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.empty((n_obj, n_freq), dtype=torch.float64, device=dev)
    bf = torch.empty(n_obj, dtype=torch.float64, device=dev)
    bi = torch.empty(n_obj, dtype=torch.int64, device=dev)
    stream = torch.cuda.current_stream()

    def step(m=mode, profile=False):
        o = ss.default_options(profile=1 if profile else 0, precision=1 if args.precision == "mixed" else 0)
        ss.ss_periodogram(t, y, e, off, n_obj, cat.f_min, cat.f_max, n_freq, m, pg, bf, bi, o)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        step()
    launches_per_step = ss.last_launch_count()
    barrier()
    sampler.mark()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms, kernel_launches = 0.0, 0
    ev0.record(stream)
    for _ in range(args.steps):
        step(profile=True)
        ms, cnt = ss.last_kernel_ms()
        kernel_ms += ms; kernel_launches += cnt
    ev1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    elapsed_ms = max_over_ranks(ev0.elapsed_time(ev1), dist if use_dist else None, dev)
    ms_per_step = elapsed_ms / args.steps
    value = job_throughput(world, evals_per_step, args.steps, elapsed_ms)
    best_idx_checksum = int(bi.sum().item())

    # the other mode, same catalog, same launch configuration (reported, not the headline)
    other = ss.GENERALIZED_VALIDATION if mode == ss.CROSS_VALIDATION else ss.CROSS_VALIDATION
    step(other); step(other)
    torch.cuda.synchronize()
    other_times = []
    for _ in range(3):                      # median of three single steps (reported, not the headline)
        o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        o0.record(stream)
        step(other)
        o1.record(stream)
        torch.cuda.synchronize()
        other_times.append(o0.elapsed_time(o1))
    other_ms = sorted(other_times)[1]

    # ---- e2e: host buffers through ss_periodogram_host, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        ht = torch.from_numpy(cat.times).pin_memory(); hy = torch.from_numpy(cat.mags).pin_memory()
        he = torch.from_numpy(cat.errs).pin_memory(); hoff = torch.from_numpy(cat.offsets).pin_memory()
        hpg = torch.empty((n_obj, n_freq), dtype=torch.float64).pin_memory()
        hbf = torch.empty(n_obj, dtype=torch.float64).pin_memory()
        hbi = torch.empty(n_obj, dtype=torch.int64).pin_memory()
        def estep():
            ss.ss_periodogram_host(ht, hy, he, hoff, n_obj, cat.f_min, cat.f_max, n_freq, mode, hpg, hbf, hbi,
                                   ss.default_options(precision=1 if args.precision == "mixed" else 0))
        estep()
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            estep()
        barrier()
        dt = max_over_ranks(time.perf_counter() - t0, dist if use_dist else None, dev)
        e2e = {"value": job_throughput(world, evals_per_step, n_e2e, dt * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": int(3 * 8 * cat.n_points + 8 * (n_obj + 1)),
               "d2h_bytes_per_step": int(8 * n_obj * n_freq + 16 * n_obj),
               "api": "ss_periodogram_host (pinned host buffers, tiled D2H overlapped with kernels)"}
        assert int(hbi.sum().item()) == best_idx_checksum, "host and device entry points disagree"
        del hpg

    if rank != 0:
        return
    pk, pk_src = peaks()
    fp64_meas, smem_meas = ss.microbench()
    sm_max = float(pk.get("sm_max_mhz", 1965.0))
    peak_tflops = N_SM * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    k_ms = kernel_ms / max(1, kernel_launches)
    k_units = point_evals_per_step * args.steps / max(1, kernel_launches)   # point-evals per launch
    smem_achieved = SMEM_BYTES_PER_POINT_EVAL[args.mode] * k_units / (k_ms * 1e-3)
    fp64_achieved = FLOP_PER_POINT_EVAL[args.mode] * k_units / (k_ms * 1e-3) / 1e12
    traffic, traffic_note = None, "no capture for this workload"
    if os.path.exists(TRAFFIC_JSON):
        with open(TRAFFIC_JSON) as f:
            tj = json.load(f)
        traffic_note = tj.get("note", "")
        if (args.config, n_obj, n_freq, args.mode) == (tj.get("config"), tj.get("n_objects"), tj.get("n_freq"), tj.get("mode")):
            traffic = float(tj["dram_bytes_read"]) + float(tj["dram_bytes_write"])
    if args.precision == "mixed":
        # the mixed kernels keep their prefix arrays in float2: half the algorithmic shared-memory bytes, and the
        # smoother's arithmetic leaves the fp64 pipe; this line is never the headline
        smem_achieved *= 0.5
        traffic_note = "precision=mixed: shared-memory bytes per point-eval halved (float2 prefix arrays); the fp64 sub-object does not apply"
    roofline = {"bound": "smem", "kernel": "eval kernel (fold+sort+smoother+statistic fused)",
                "achieved": smem_achieved / 1e12, "peak": smem_meas / 1e12, "unit": "TB/s", "frac": smem_achieved / smem_meas,
                "traffic": traffic, "traffic_note": traffic_note,
                "peak_source": "shared-memory read microbenchmark of this run (ss_microbench; 148 SM x 128 B/clk x "
                               f"{sm_max:.0f} MHz = {N_SM * 128 * sm_max * 1e6 / 1e12:.2f} TB/s nominal)",
                "bytes_per_point_eval": SMEM_BYTES_PER_POINT_EVAL[args.mode] * (0.5 if args.precision == "mixed" else 1.0),
                "point_evals_per_launch": k_units, "kernel_ms_per_launch": k_ms,
                "kernel_share_of_step": kernel_ms / elapsed_ms,
                "fp64": {"achieved": fp64_achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": fp64_achieved / peak_tflops,
                         "frac_as_implemented": fp64_achieved / peak_tflops * SLOTS_AS_IMPLEMENTED[args.mode] / SLOTS_PER_POINT_EVAL[args.mode],
                         "flop_per_point_eval": FLOP_PER_POINT_EVAL[args.mode],
                         "note": f"secondary roofline: SURVEY 8(d) slots per point-eval against {N_SM} SM x {FP64_LANES_PER_SM} fp64 "
                                 f"FMA lanes x 2 x {sm_max:.0f} MHz ({pk_src} clock); DFMA microbenchmark of this run "
                                 f"{fp64_meas / 1e12:.2f} TFLOP/s; as_implemented prices a division at 4 slots and a square root at 7"},
                "hbm_gbs_algorithmic": 8.0 * evals_per_step / (ms_per_step * 1e-3) / 1e9}
    cpu = None
    if not args.no_cpu:
        cpu, _, _ = cpu_baseline(cat, args.mode)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64" if args.precision == "f64" else "f32", "data": "synthetic",
           "config": {"workload": f"config{args.config}: {n_obj} objects ({cat.n_points} points) x {n_freq} "
                      f"frequencies on [{cat.f_min},{cat.f_max}), mode={args.mode}, periodogram materialised"
                      + (", precision=mixed (fp32 smoother on the warp and group paths; fp64 fold, sort and prefix accumulation across threads)" if args.precision == "mixed" else ""),
                      "objects_per_second": world * n_obj * args.steps / (elapsed_ms * 1e-3),
                      "l2": (f"inputs ({24 * cat.n_points / 1e6:.0f} MB catalog) are re-read per frequency by design; the "
                             f"{8 * evals_per_step / 1e9:.2f} GB periodogram written every step "
                             + ("exceeds the 126 MB L2, nothing is cached between steps" if 8 * evals_per_step > 126e6
                                else "FITS the L2: reduced debug size, not a bench line")),
                      "other_mode": {"mode": "gv" if args.mode == "cv" else "cv",
                                     "value": evals_per_step / (other_ms * 1e-3), "unit": UNIT},
                      "parallelism": f"objects sharded over {world} rank(s), no collective"},
           "gpu_launches": int(launches_per_step * args.steps), "clocks": clocks,
           "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out), flush=True)


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
