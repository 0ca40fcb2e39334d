"""Path-crossover sweep over the light-curve length n (the analogue of the paper's
kernel-cascade study).

For each n a catalog of equal-length light curves is timed through the device entry point on every path
class that can serve it (SS_PATH_WARP for n <= 256, SS_PATH_GROUP for n <= 3,584, SS_PATH_BLOCK for n <= 2,055,
SS_PATH_CLUSTER for 2,055 < n <= 40,960, SS_PATH_STAGE for any n), in both modes; the table reports point-evals/s (n x frequencies x objects / second), which is flat
where a path scales and drops where it stops fitting.  The path the library picks by itself is marked.

    python -m paper_2111_07396_b200.sweep [--ns 50,100,...] [--target-ms 150] [--md out.md]
    python -m paper_2111_07396_b200.sweep --options [--md out.md]     # the listing's options vs the default call
    python -m paper_2111_07396_b200.sweep --shared | --mixed          # shared time sampling / mixed precision vs the plain call

Needs a CUDA device (no CPU fallback).  Inputs are synthetic: times uniform over 30 nights (8 h per
night), a sinusoid of random period plus Gaussian noise; the arithmetic under test is all in the library.
"""
from __future__ import annotations

import argparse
import sys

import time

import numpy as np

from . import (CROSS_VALIDATION, GENERALIZED_VALIDATION, PATH_BLOCK, PATH_CLUSTER, PATH_GROUP, PATH_STAGE, PATH_WARP, default_options,
               load,
               path_for_n, ss_periodogram)

DEFAULT_NS = [50, 64, 96, 128, 160, 200, 256, 257, 320, 400, 512, 700, 1000, 1400, 2055, 2056, 3000, 3584, 3585, 5000, 10000, 20000, 40000]
PATH_NAME = {PATH_WARP: "warp", PATH_GROUP: "group", PATH_CLUSTER: "cluster", PATH_BLOCK: "cta-smem", PATH_STAGE: "cta-staged"}
WARP_MAX_N, BLOCK_MAX_N, GROUP_LONG_MAX_N, CLUSTER_MAX_N = 256, 2055, 3584, 40960


def catalog(n: int, n_objects: int, seed: int):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.integers(0, 30, size=(n_objects, n)) + rng.uniform(0.0, 0.33, size=(n_objects, n)), axis=1)
    period = np.exp(rng.uniform(np.log(0.1), np.log(2.0), size=(n_objects, 1)))
    y = 15.0 + 0.4 * np.sin(2 * np.pi * t / period) + rng.normal(0.0, 0.05, size=(n_objects, n))
    e = np.full((n_objects, n), 0.05)
    off = np.arange(n_objects + 1, dtype=np.int64) * n
    return t.ravel(), y.ravel(), e.ravel(), off


def time_call(torch, dev, arrs, n_objects, n_freq, mode, path, reps=3, **opts):
    t, y, e, off = arrs
    pg = torch.empty((n_objects, n_freq), dtype=torch.float64, device=dev)
    bi = torch.empty(n_objects, dtype=torch.int64, device=dev)
    opt = default_options(force_path=path, skip_validation=1, **opts)

    def call():
        ss_periodogram(t, y, e, off, n_objects, 0.5, 24.0, n_freq, mode, pg, None, bi, opt)

    call()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    best = float("inf")
    for _ in range(reps):
        torch.cuda.synchronize()
        ev[0].record()
        call()
        ev[1].record()
        torch.cuda.synchronize()
        best = min(best, ev[0].elapsed_time(ev[1]))
    return best


def options_table(torch, dev, md):
    """Listing 1's options through the device entry point, on config-3-shaped objects (n ~ U[50, 200]: warp path) and
    config-4-shaped ones (n ~ U[500, 2,000]: group path)."""
    import ss_inputs
    lines = ["| catalog | options | CV evals/s | GV evals/s | CV time vs default |", "|---|---|---|---|---|"]
    for cat, label in ((ss_inputs.config3(n_objects=1000, n_freq=5000), "config 3 shape, 1,000 x 5,000"),
                       (ss_inputs.config4(n_objects=300, n_freq=4000), "config 4 shape, 300 x 4,000")):
        arrs = tuple(torch.as_tensor(a, device=dev) for a in (cat.times, cat.mags, cat.errs, cat.offsets))
        base = None
        for name, opts in (("default", {}), ("iper=2", dict(iper=2)), ("span=0.2", dict(span=0.2)),
                           ("iper=2, span=0.2", dict(iper=2, span=0.2)), ("alpha=0", dict(alpha=0.0)), ("alpha=5", dict(alpha=5.0))):
            row = []
            for mode in (CROSS_VALIDATION, GENERALIZED_VALIDATION):
                t, y, e, off = arrs
                pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev)
                opt = default_options(skip_validation=1, **opts)
                best = float("inf")
                for _ in range(4):
                    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
                    torch.cuda.synchronize()
                    ev[0].record()
                    ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, None, None, opt)
                    ev[1].record()
                    torch.cuda.synchronize()
                    best = min(best, ev[0].elapsed_time(ev[1]))
                row.append(cat.n_objects * cat.n_freq / (best * 1e-3))
            base = base or row[0]
            lines.append(f"| {label} | {name} | {row[0]:.4g} | {row[1]:.4g} | {base / row[0]:.2f}x |")
            print(lines[-1], flush=True)
    if md:
        with open(md, "w") as f:
            f.write("\n".join(lines) + "\n")
    return 0


def _best_of(torch, call, reps=4):
    """Best wall time of `reps` calls after one untimed call (module load, clocks)."""
    call()
    best = float("inf")
    for _ in range(reps):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        call()
        torch.cuda.synchronize()
        best = min(best, time.perf_counter() - t0)
    return best


def shared_table(torch, dev, md):
    """shared_times = 1 (one fold + sort per frequency for 4 objects) against the ordinary call."""
    lines = ["| n | objects x frequencies | mode | plain evals/s | shared_times evals/s | speed-up |", "|---|---|---|---|---|---|"]
    # n <= 256: warp path, 2,000 objects x 10,000 frequencies; beyond: group path, 400 x 3,000
    for n, n_obj, nf in ((64, 2000, 10000), (125, 2000, 10000), (200, 2000, 10000), (500, 400, 3000), (1000, 400, 3000),
                         (2000, 400, 3000)):
        rng = np.random.default_rng(n)
        t1 = np.sort(rng.integers(0, 30 if n <= 256 else 900, size=n) + rng.uniform(0.0, 0.33, size=n))
        t = np.tile(t1, n_obj)
        e = rng.uniform(0.02, 0.1, size=n_obj * n)
        y = 15 + 0.4 * np.sin(2 * np.pi * t / np.repeat(np.exp(rng.uniform(np.log(0.1), np.log(2.0), size=n_obj)), n)) \
            + rng.normal(0, 1.0, size=n_obj * n) * e
        off = np.arange(n_obj + 1, dtype=np.int64) * n
        a = [torch.as_tensor(v, device=dev) for v in (t, y, e, off)]
        pg = torch.empty((n_obj, nf), dtype=torch.float64, device=dev)
        for mode, name in ((CROSS_VALIDATION, "cv"), (GENERALIZED_VALIDATION, "gv")):
            r = []
            for sh in (0, 1):
                o = default_options(shared_times=sh, skip_validation=1)
                r.append(n_obj * nf / _best_of(torch, lambda: ss_periodogram(*a, n_obj, 0.5, 24.0, nf, mode, pg, None, None, o)))
            lines.append(f"| {n} | {n_obj} x {nf} | {name} | {r[0]:.4g} | {r[1]:.4g} | {r[1] / r[0]:.3f} |")
            print(lines[-1], flush=True)
    if md:
        with open(md, "w") as f:
            f.write("\n".join(lines) + "\n")
    return 0


def mixed_table(torch, dev, md):
    """precision = SS_PRECISION_MIXED (fp32 smoother on the warp and group paths) against fp64."""
    import ss_inputs
    lines = ["| catalog | mode | fp64 evals/s | mixed evals/s | speed-up |", "|---|---|---|---|---|"]
    # the third catalog: eight light curves of the paper's ObjLarge length (N_t = 3,554)
    t3, y3, e3, o3 = catalog(3554, 8, seed=3554)
    long = ss_inputs.Catalog("long", t3, y3, e3, o3, 0.5, 24.0, 20000, np.full(8, np.nan))
    for cat, label in ((ss_inputs.config3(n_objects=1000, n_freq=5000), "config 3 shape, 1,000 x 5,000 (warp path)"),
                       (ss_inputs.config4(n_objects=300, n_freq=4000), "config 4 shape, 300 x 4,000 (group path)"),
                       (long, "n = 3,554, 8 x 20,000 (group path, 16 warps x 7 points)")):
        a = [torch.as_tensor(v, device=dev) for v in (cat.times, cat.mags, cat.errs, cat.offsets)]
        pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev)
        for mode, name in ((CROSS_VALIDATION, "cv"), (GENERALIZED_VALIDATION, "gv")):
            r = []
            for pr in (0, 1):
                o = default_options(precision=pr, skip_validation=1)
                r.append(cat.n_objects * cat.n_freq / _best_of(torch, lambda: ss_periodogram(
                    *a, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, None, None, o)))
            lines.append(f"| {label} | {name} | {r[0]:.4g} | {r[1]:.4g} | {r[1] / r[0]:.3f} |")
            print(lines[-1], flush=True)
    if md:
        with open(md, "w") as f:
            f.write("\n".join(lines) + "\n")
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--ns", default=",".join(map(str, DEFAULT_NS)))
    ap.add_argument("--target-ms", type=float, default=150.0, help="aim each timed call at about this long")
    ap.add_argument("--md", default=None, help="also write the table as markdown to this file")
    ap.add_argument("--options", action="store_true",
                    help="instead of the sweep over n: the listing's options (iper = 2, fixed span; PAPER.md:199-210) "
                         "against the default call on config-3- and config-4-shaped catalogs")
    ap.add_argument("--shared", action="store_true",
                    help="instead: shared_times = 1 against the ordinary call on catalogs with one time vector "
                         "(PAPER.md:125), n = 64 ... 2,000")
    ap.add_argument("--mixed", action="store_true",
                    help="instead: precision = mixed against fp64 on config-3- and config-4-shaped catalogs (PAPER.md:604-616)")
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("sweep needs a CUDA device (the library has no CPU path)")
    load()
    dev = torch.device("cuda")
    if args.options:
        return options_table(torch, dev, args.md)
    if args.shared:
        return shared_table(torch, dev, args.md)
    if args.mixed:
        return mixed_table(torch, dev, args.md)
    lines = ["| n | path | auto | objects x frequencies | CV point-evals/s | CV evals/s | GV point-evals/s | GV evals/s |",
             "|---|---|---|---|---|---|---|---|"]
    for n in [int(v) for v in args.ns.split(",")]:
        paths = [p for p in (PATH_WARP, PATH_GROUP, PATH_CLUSTER, PATH_BLOCK, PATH_STAGE)
                 if (p != PATH_WARP or n <= WARP_MAX_N) and (p != PATH_BLOCK or n <= BLOCK_MAX_N)
                 and (p != PATH_GROUP or n <= GROUP_LONG_MAX_N)
                 and (p != PATH_CLUSTER or BLOCK_MAX_N < n <= CLUSTER_MAX_N)]
        auto = path_for_n(n)
        for path in paths:
            # size the call: enough (object, frequency) items to fill 148 SMs several times over
            n_objects = 296 if n <= 2055 else 8
            arrs_h = catalog(n, n_objects, seed=1000 + n)
            arrs = tuple(torch.as_tensor(a, device=dev) for a in arrs_h)
            row = []
            for mode in (CROSS_VALIDATION, GENERALIZED_VALIDATION):
                # grow the grid until one call lasts about target-ms (the per-call overhead -- workspace
                # allocation, one host sync -- is about a millisecond and must not dominate)
                nf, ms = 64, 0.0
                for _ in range(6):
                    ms = time_call(torch, dev, arrs, n_objects, nf, mode, path, reps=2)
                    if ms >= 0.5 * args.target_ms or nf >= 400000:
                        break
                    nf = int(min(400000, max(2 * nf, nf * args.target_ms / max(ms, 0.05))))
                ms = time_call(torch, dev, arrs, n_objects, nf, mode, path)
                ev = n_objects * nf / (ms * 1e-3)
                row.append((nf, ev * n, ev))
            lines.append(f"| {n} | {PATH_NAME[path]} | {'*' if path == auto else ''} | {n_objects} x {row[0][0]} / {row[1][0]} | "
                         f"{row[0][1]:.3g} | {row[0][2]:.3g} | {row[1][1]:.3g} | {row[1][2]:.3g} |")
            print(lines[-1], flush=True)
    if args.md:
        with open(args.md, "w") as f:
            f.write("\n".join(lines) + "\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
