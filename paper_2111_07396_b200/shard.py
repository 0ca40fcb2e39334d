"""Multi-GPU object sharding.

The paper hands whole objects to GPUs ("an object is computed by a single GPU", dynamic assignment
because execution time varies with N_t).  Here: one process per GPU, every rank computes the same
static partition of the catalog's objects, balanced by a cost model, runs the single-GPU library on
its own shard and writes its own rows.  There is no collective on the data path; the only exchange
is the optional gather of the per-object best frequency (16 bytes per object) at the end.

Host-side logic only: no SuperSmoother arithmetic lives here.
"""
from __future__ import annotations

import numpy as np

# Point-evals per second each path class sustains on one B200 (profiles/r2_crossover.md, CV mode: warp / group /
# cluster / global staging): the relative cost of an object is n / rate(path(n)).  Only the ratios matter.
_RATE = ((256, 3.3e10), (3584, 2.2e10), (40960, 5.5e9), (1 << 62, 1.4e9))


def object_cost(n) -> np.ndarray:
    """Relative cost of one (object, frequency) eval for light curves of n points."""
    n = np.asarray(n, dtype=np.float64)
    rate = np.full(n.shape, _RATE[-1][1])
    for limit, r in reversed(_RATE):
        rate = np.where(n <= limit, r, rate)
    return np.where(n >= 5, n / rate, 0.0)       # n < 5: NaN row, no eval (R17)


def shard_objects(offsets, world_size: int) -> list[np.ndarray]:
    """Partition object indices over world_size ranks: longest-processing-time-first greedy on
    object_cost, each rank's list returned in ascending object order.  Deterministic (ties by index),
    so every rank computes the same partition without communicating."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    offsets = np.asarray(offsets, dtype=np.int64)
    cost = object_cost(np.diff(offsets))
    order = np.lexsort((np.arange(len(cost)), -cost))       # cost descending, index ascending
    load = np.zeros(world_size)
    count = np.zeros(world_size, dtype=np.int64)
    owner = np.empty(len(cost), dtype=np.int64)
    for i in order:
        # least loaded rank; among equals the one with fewer objects, then the lowest rank
        r = int(np.lexsort((np.arange(world_size), count, load))[0])
        owner[i] = r
        load[r] += cost[i]
        count[r] += 1
    return [np.nonzero(owner == r)[0] for r in range(world_size)]


def sub_catalog(times, mags, errs, offsets, idx):
    """CSR sub-catalog of the objects idx (in that order): (times, mags, errs, offsets)."""
    offsets = np.asarray(offsets, dtype=np.int64)
    idx = np.asarray(idx, dtype=np.int64)
    lens = offsets[idx + 1] - offsets[idx]
    off = np.zeros(len(idx) + 1, dtype=np.int64)
    np.cumsum(lens, out=off[1:])
    sel = np.concatenate([np.arange(offsets[i], offsets[i + 1]) for i in idx]) if len(idx) else np.zeros(0, np.int64)
    return (np.ascontiguousarray(np.asarray(times)[sel]), np.ascontiguousarray(np.asarray(mags)[sel]),
            np.ascontiguousarray(np.asarray(errs)[sel]), off)


def periodogram_sharded(times, mags, errs, offsets, f_min, f_max, n_freq, mode=0, *, rank: int, world_size: int,
                        want_pgram: bool = True, **opts):
    """This rank's share of the catalog through the single-GPU library (ss_periodogram_host on the
    current CUDA device).  Returns (idx, Result): idx = the object indices this rank owns, Result
    rows in that order."""
    from . import periodogram
    idx = shard_objects(offsets, world_size)[rank]
    t, y, e, off = sub_catalog(times, mags, errs, offsets, idx)
    return idx, periodogram(t, y, e, off, f_min, f_max, n_freq, mode, want_pgram=want_pgram, **opts)


def gather_best(idx, best_freq, best_index, n_objects: int, group=None):
    """Assemble the per-object best frequency / index of all ranks on every rank (torch.distributed
    all_gather_object; 16 bytes per object, off the data path).  Without an initialised process group
    this is the single-rank identity."""
    bf = np.full(n_objects, np.nan)
    bi = np.full(n_objects, -1, dtype=np.int64)
    parts = [(np.asarray(idx), np.asarray(best_freq), np.asarray(best_index))]
    try:
        import torch.distributed as dist
        if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
            parts = [None] * dist.get_world_size(group)
            dist.all_gather_object(parts, (np.asarray(idx), np.asarray(best_freq), np.asarray(best_index)), group=group)
    except ImportError:
        pass
    seen = np.zeros(n_objects, dtype=bool)
    for i, f, k in parts:
        if np.any(seen[i]):
            raise ValueError("shards overlap")
        seen[i] = True
        bf[i] = f
        bi[i] = k
    if not np.all(seen):
        raise ValueError("shards do not cover the catalog")
    return bf, bi


# ---- one (or a few) long light curves: split the frequency range instead ------------
def shard_frequencies(n_freq: int, world_size: int) -> list[tuple[int, int]]:
    """Contiguous, near-equal ranges (k_begin, k_count) of the grid indices 0..n_freq-1, one per rank
    (ranks beyond n_freq get an empty range)."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    base, extra = divmod(int(n_freq), world_size)
    out, k = [], 0
    for r in range(world_size):
        c = base + (1 if r < extra else 0)
        out.append((k, c))
        k += c
    return out


def periodogram_freq_sharded(times, mags, errs, offsets, f_min, f_max, n_freq, mode=0, *, rank: int, world_size: int,
                             **opts):
    """This rank's frequency range of every object, through the library's k_begin / k_count options: the
    grid (f_min, f_max, n_freq) is unchanged, so every f_k keeps its bits.  Returns ((k_begin, k_count), Result);
    Result.pgram has k_count columns, Result.best_index indexes the whole grid."""
    from . import periodogram
    k_begin, k_count = shard_frequencies(n_freq, world_size)[rank]
    if k_count == 0:
        return (k_begin, 0), None
    return (k_begin, k_count), periodogram(times, mags, errs, offsets, f_min, f_max, n_freq, mode, want_pgram=True,
                                           k_begin=k_begin, k_count=k_count, **opts)


def merge_best_over_ranges(parts, n_objects: int):
    """parts: iterable of (k_begin, best_index[n_objects], best_power[n_objects]) from disjoint frequency ranges.
    Per object the highest power wins, ties go to the lowest index (the argmax rule of the single call, O8);
    best_index -1 (object with fewer than 5 points) stays -1."""
    bi = np.full(n_objects, -1, dtype=np.int64)
    bp = np.full(n_objects, -np.inf)
    for _, idx, pw in sorted(parts, key=lambda t: t[0]):
        idx = np.asarray(idx, dtype=np.int64)
        pw = np.asarray(pw, dtype=np.float64)
        take = (idx >= 0) & ((pw > bp) | (bi < 0))          # ranges come in ascending k: '>' keeps the first maximum
        bi = np.where(take, idx, bi)
        bp = np.where(take, pw, bp)
    return bi, bp


def gather_best_over_ranges(k_range, result, n_objects: int, group=None):
    """All ranks exchange (best index, best power) of their frequency range (all_gather_object, 16 bytes per
    object) and every rank returns the merged (best_index, best_power)."""
    if result is None:
        mine = (k_range[0], np.full(n_objects, -1, dtype=np.int64), np.full(n_objects, -np.inf))
    else:
        cols = np.clip(result.best_index - k_range[0], 0, max(k_range[1] - 1, 0))
        power = np.where(result.best_index >= 0, result.pgram[np.arange(n_objects), cols], -np.inf)
        mine = (k_range[0], result.best_index, power)
    parts = [mine]
    try:
        import torch.distributed as dist
        if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
            parts = [None] * dist.get_world_size(group)
            dist.all_gather_object(parts, mine, group=group)
    except ImportError:
        pass
    return merge_best_over_ranges(parts, n_objects)
