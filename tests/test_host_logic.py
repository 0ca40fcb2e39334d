"""CPU-only checks of the product's host logic: the C-ABI library loads and exports every symbol
include/ss_periodogram.h declares, the batch planner (P6) and the argument validation that needs no
device.  No compute call is made here."""
import os
import re

import numpy as np
import pytest

import paper_2111_07396_b200 as ss

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "ss_periodogram.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ss_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    lib = ss.load()
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert declared == set(ss.EXPORTS)
    assert ss.version() == 200


def test_paper_footprint_fixture():
    """15*N_t*N_f words = 5.59 GiB at N_t=50, N_f=1e6, FP64."""
    for line in open(os.path.join(GOLD, "footprint.txt")):
        if line.startswith("#") or not line.strip():
            continue
        nt, nf, words, bpw, gib = line.split()
        got = ss.paper_footprint_bytes(int(nt), int(nf)) / 2 ** 30
        assert abs(got - float(gib)) < 0.005
        assert abs(got - int(words) * int(bpw) * int(nt) * int(nf) / 2 ** 30) < 1e-9


def test_paper_batch_count_eq1():
    """N_b = r/(beta*s); r_orig has 160 N_f N_t bytes, r_sp 96; monotone in N_f."""
    nt, s, beta = 3554, 16.0, 0.75
    prev = 0
    for nf in (10 ** 4, 10 ** 5, 5 * 10 ** 5, 10 ** 6):
        r = (8 * nf + 24 * nt + 160 * nf * nt) / 2 ** 30
        nb = ss.paper_batches(nt, nf, ss.CROSS_VALIDATION, s, beta)
        assert nb == max(1, int(np.ceil(r / (beta * s))))
        assert nb >= prev
        prev = nb
        assert ss.paper_batches(nt, nf, ss.GENERALIZED_VALIDATION, s, beta) <= nb
    # ratio of the N_f*N_t terms is 160/96 = 1.67
    assert abs(160 / 96 - 1.67) < 0.01


def test_path_classes():
    assert ss.path_for_n(5) == ss.PATH_WARP
    assert ss.path_for_n(256) == ss.PATH_WARP
    assert ss.path_for_n(257) == ss.PATH_GROUP
    assert ss.path_for_n(2000) == ss.PATH_GROUP
    assert ss.path_for_n(2055) == ss.PATH_GROUP
    assert ss.path_for_n(2056) == ss.PATH_GROUP          # the long group variants (y, w read from global memory)
    assert ss.path_for_n(3584) == ss.PATH_GROUP
    assert ss.path_for_n(3585) == ss.PATH_CLUSTER
    assert ss.path_for_n(20000) == ss.PATH_CLUSTER
    assert ss.path_for_n(40960) == ss.PATH_CLUSTER
    assert ss.path_for_n(40961) == ss.PATH_STAGE


@pytest.mark.parametrize("cap_mib", [128, 256, 1024, 16384])
def test_planner_tiles_cover_the_grid_once(cap_mib):
    """Tiles partition objects x frequencies exactly; the plan never exceeds the cap."""
    n_obj, n_freq, total, max_n = 1000, 500000, 1250000, 2000      # config 4 sizes
    p = ss.plan(total, max_n, n_obj, n_freq, cap_bytes=cap_mib << 20, host_tiles=True)
    assert p.total_bytes <= cap_mib << 20
    assert p.freq_per_tile >= 1 and p.objects_per_tile >= 1
    assert p.n_freq_tiles == -(-n_freq // p.freq_per_tile)
    assert p.n_object_tiles == -(-n_obj // p.objects_per_tile)
    covered = 0
    for ot in range(p.n_object_tiles):
        o0, o1 = ot * p.objects_per_tile, min(n_obj, (ot + 1) * p.objects_per_tile)
        for ft in range(p.n_freq_tiles):
            k0, k1 = ft * p.freq_per_tile, min(n_freq, (ft + 1) * p.freq_per_tile)
            assert o1 > o0 and k1 > k0
            covered += (o1 - o0) * (k1 - k0)
    assert covered == n_obj * n_freq
    assert p.tile_bytes == 8 * p.freq_per_tile * p.objects_per_tile
    if cap_mib <= 1024:
        assert p.n_freq_tiles > 1          # config 4's 4 GB periodogram must be tiled (BASELINE.json)


def test_planner_monotone_and_failure():
    a = ss.plan(1250000, 200, 10000, 50000, cap_bytes=1 << 30, host_tiles=True)
    b = ss.plan(1250000, 200, 10000, 100000, cap_bytes=1 << 30, host_tiles=True)
    assert b.n_freq_tiles >= a.n_freq_tiles
    with pytest.raises(ss.SSError) as ei:
        ss.plan(1250000, 200, 10000, 50000, cap_bytes=1 << 20, host_tiles=True)
    assert ei.value.status == ss.SS_ERR_OUT_OF_MEMORY
    # device-output calls allocate no periodogram tile
    c = ss.plan(1250000, 200, 10000, 50000, cap_bytes=1 << 30, host_tiles=False)
    assert c.tile_bytes == 0 and c.n_freq_tiles == 1
    assert ss.workspace_bytes(1250000, 200, 10000, 50000) == c.total_bytes
    # a 20,000-point object needs the global staging scratch
    d = ss.plan(20000, 20000, 1, 10 ** 6, cap_bytes=1 << 34, host_tiles=False)
    assert d.stage_bytes > 0 and c.stage_bytes == 0


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(ss.SSError):
        ss.periodogram(np.arange(6.0), np.arange(6.0), np.ones(6), [0, 6], 0.1, 1.0, 10)
