"""Multi-GPU object sharding (paper_2111_07396_b200/shard.py): host logic on CPU,
the world_size-2 exchange over gloo, and -- on a GPU -- that the shards reproduce the unsharded bits."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import ss_inputs
from paper_2111_07396_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_covers_every_object_once_and_is_balanced():
    cat = ss_inputs.config3(n_objects=2000, n_freq=8)
    ns = np.diff(cat.offsets)
    cost = shard.object_cost(ns)
    for world in (1, 2, 3, 4, 8):
        parts = shard.shard_objects(cat.offsets, world)
        assert len(parts) == world
        allidx = np.concatenate(parts)
        assert np.array_equal(np.sort(allidx), np.arange(cat.n_objects))          # exactly once
        for p in parts:
            assert np.all(np.diff(p) > 0)                                          # ascending
        loads = np.array([cost[p].sum() for p in parts])
        assert loads.max() <= loads.mean() * 1.001 + cost.max()                   # LPT bound: within one object
        again = shard.shard_objects(cat.offsets, world)
        assert all(np.array_equal(a, b) for a, b in zip(parts, again))             # deterministic


def test_cost_model_orders_paths_and_ignores_degenerate_objects():
    c = shard.object_cost([0, 4, 5, 100, 256, 257, 3584, 3585, 20000])
    assert c[0] == 0 and c[1] == 0 and c[2] > 0
    assert np.all(np.diff(c[2:]) > 0)                        # longer light curves cost more
    assert 1.2 < c[5] / c[4] < 2.0                           # the group path costs ~1.4x more per point than the warp path
    assert c[7] / c[6] > 3.0                                 # the cluster path ~4x more than the group path
    # a mixed catalog: one huge object must not share its rank with much else
    off = np.concatenate([[0], np.cumsum([20000] + [100] * 50)])
    parts = shard.shard_objects(off, 2)
    owner0 = [p for p in parts if 0 in p][0]
    assert len(owner0) == 1


def test_sub_catalog_is_the_csr_subset():
    cat = ss_inputs.config3(n_objects=30, n_freq=8)
    idx = np.array([3, 7, 8, 29])
    t, y, e, off = shard.sub_catalog(cat.times, cat.mags, cat.errs, cat.offsets, idx)
    assert off[0] == 0 and len(off) == 5
    for m, i in enumerate(idx):
        ti, yi, ei = cat.obj(int(i))
        assert np.array_equal(t[off[m]:off[m + 1]], ti)
        assert np.array_equal(y[off[m]:off[m + 1]], yi)
        assert np.array_equal(e[off[m]:off[m + 1]], ei)
    t, y, e, off = shard.sub_catalog(cat.times, cat.mags, cat.errs, cat.offsets, [])
    assert len(t) == 0 and np.array_equal(off, [0])


def test_gather_best_single_rank_identity_and_checks():
    bf, bi = shard.gather_best([0, 1, 2], [1.0, 2.0, 3.0], [10, 20, 30], 3)
    assert np.array_equal(bf, [1.0, 2.0, 3.0]) and np.array_equal(bi, [10, 20, 30])
    with pytest.raises(ValueError):
        shard.gather_best([0, 1], [1.0, 2.0], [10, 20], 3)          # object 2 missing


WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import numpy as np
import torch.distributed as dist
import ss_inputs
from paper_2111_07396_b200 import shard
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
cat = ss_inputs.config3(n_objects=101, n_freq=8)
idx = shard.shard_objects(cat.offsets, world)[rank]
t, y, e, off = shard.sub_catalog(cat.times, cat.mags, cat.errs, cat.offsets, idx)
# stand-in for the GPU call (no device here): a per-object figure that depends on the object's own data
bf = np.array([t[off[m]:off[m + 1]].sum() for m in range(len(idx))])
bi = (np.diff(off) * 7).astype(np.int64)
full_bf, full_bi = shard.gather_best(idx, bf, bi, cat.n_objects)
print(json.dumps({"rank": rank, "n_mine": int(len(idx)), "bf": full_bf.tolist(), "bi": full_bi.tolist()}), flush=True)
dist.destroy_process_group()
"""


def test_two_rank_shard_and_gather_over_gloo():
    port = 29100 + os.getpid() % 300
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER, ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    cat = ss_inputs.config3(n_objects=101, n_freq=8)
    want_bf = [float(cat.obj(i)[0].sum()) for i in range(cat.n_objects)]
    want_bi = (np.diff(cat.offsets) * 7).tolist()
    assert outs[0]["n_mine"] + outs[1]["n_mine"] == 101 and min(o["n_mine"] for o in outs) > 30
    for o in outs:                                   # every rank ends up with the whole catalog's answer
        assert o["bf"] == want_bf and o["bi"] == want_bi


def test_frequency_ranges_and_best_merge():
    for n_freq, world in ((10, 3), (7, 8), (1000000, 4)):
        r = shard.shard_frequencies(n_freq, world)
        assert len(r) == world and r[0][0] == 0 and sum(c for _, c in r) == n_freq
        assert all(r[i][0] + r[i][1] == r[i + 1][0] for i in range(world - 1))
        assert max(c for _, c in r) - min(c for _, c in r) <= 1
    # merge = argmax over the concatenated row, first maximum wins; degenerate objects stay -1
    rng = np.random.default_rng(5)
    row = rng.normal(size=(4, 90)); row[1, 70] = row[1, 20] = row[1].max() + 1.0     # a tie across ranges
    parts = []
    for kb, kc in shard.shard_frequencies(90, 3):
        seg = row[:, kb:kb + kc]
        idx = kb + np.argmax(seg, axis=1); pw = seg.max(axis=1)
        idx[3] = -1; pw[3] = -np.inf
        parts.append((kb, idx, pw))
    bi, bp = shard.merge_best_over_ranges(parts[::-1], 4)             # order of arrival must not matter
    assert np.array_equal(bi[:3], np.argmax(row[:3], axis=1)) and bi[1] == 20 and bi[3] == -1
    assert np.array_equal(bp[:3], row[:3].max(axis=1))


@pytest.mark.gpu
@pytest.mark.parametrize("mode", [0, 1])
def test_frequency_ranges_reproduce_the_whole_grid_bit_for_bit(mode):
    """k_begin / k_count (one object's grid split over 'ranks', run one after the other here): the pieces
    concatenate to the single-call periodogram exactly and the merged best index is the single call's.
    Covers the warp, CTA and staging classes and both entry points."""
    import torch
    import paper_2111_07396_b200 as ss
    a = ss_inputs.config3(n_objects=5, n_freq=203)
    b = ss_inputs.config4(n_objects=2, n_freq=203)
    times = np.concatenate([a.times, b.times, np.linspace(0, 50, 3)]); mags = np.concatenate([a.mags, b.mags, [15., 15.1, 15.2]])
    errs = np.concatenate([a.errs, b.errs, [0.1, 0.1, 0.1]])
    offsets = np.concatenate([a.offsets, a.offsets[-1] + b.offsets[1:], [a.offsets[-1] + b.offsets[-1] + 3]])
    n_obj = len(offsets) - 1                                                      # the last object has 3 points: NaN row
    whole = ss.periodogram(times, mags, errs, offsets, 0.5, 24.0, 203, mode)
    for world in (2, 3):
        pieces, parts = [], []
        for rank in range(world):
            kr, res = shard.periodogram_freq_sharded(times, mags, errs, offsets, 0.5, 24.0, 203, mode, rank=rank,
                                                     world_size=world)
            assert res.pgram.shape == (n_obj, kr[1])
            pieces.append(res.pgram)
            cols = np.clip(res.best_index - kr[0], 0, kr[1] - 1)
            parts.append((kr[0], res.best_index, np.where(res.best_index >= 0, res.pgram[np.arange(n_obj), cols], -np.inf)))
        assert np.array_equal(np.concatenate(pieces, axis=1), whole.pgram, equal_nan=True)
        bi, _ = shard.merge_best_over_ranges(parts, n_obj)
        assert np.array_equal(bi, whole.best_index)
    # device entry point with a sub-range, forced staging path
    dev = torch.device("cuda")
    t = torch.as_tensor(times, device=dev); y = torch.as_tensor(mags, device=dev); e = torch.as_tensor(errs, device=dev)
    off = torch.as_tensor(offsets, device=dev)
    pg = torch.empty((n_obj, 50), dtype=torch.float64, device=dev)
    bi_d = torch.empty(n_obj, dtype=torch.int64, device=dev); bf_d = torch.empty(n_obj, dtype=torch.float64, device=dev)
    ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, 203, mode, pg, bf_d, bi_d,
                      ss.default_options(k_begin=100, k_count=50, force_path=ss.PATH_STAGE))
    staged = ss.periodogram(times, mags, errs, offsets, 0.5, 24.0, 203, mode, force_path=ss.PATH_STAGE)   # same kernel, whole grid
    assert np.array_equal(pg.cpu().numpy(), staged.pgram[:, 100:150], equal_nan=True)
    k = bi_d.cpu().numpy()
    assert np.all((k[:-1] >= 100) & (k[:-1] < 150)) and k[-1] == -1
    with pytest.raises(ss.SSError):
        ss.periodogram(times, mags, errs, offsets, 0.5, 24.0, 203, mode, k_begin=200, k_count=10)


@pytest.mark.gpu
@pytest.mark.parametrize("mode", [0, 1])
def test_shards_reproduce_the_unsharded_result_bit_for_bit(mode):
    """Two 'ranks' run one after the other on the one GPU there is: rows and best frequencies of the
    shards, put back in catalog order, equal the single-call result exactly (evals are independent)."""
    import paper_2111_07396_b200 as ss
    cat = ss_inputs.config3(n_objects=60, n_freq=193)
    whole = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode)
    pg = np.full_like(whole.pgram, np.nan)
    parts = []
    for rank in range(2):
        idx, res = shard.periodogram_sharded(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max,
                                             cat.n_freq, mode, rank=rank, world_size=2)
        pg[idx] = res.pgram
        parts.append((idx, res))
    assert np.array_equal(pg, whole.pgram)
    bf = np.full(cat.n_objects, np.nan); bi = np.full(cat.n_objects, -1)
    for idx, res in parts:
        bf[idx] = res.best_freq; bi[idx] = res.best_index
    assert np.array_equal(bf, whole.best_freq) and np.array_equal(bi, whole.best_index)
