"""ss_periodogram_static (include/ss_periodogram.h): the entry point that allocates nothing on the device.  Its
workspace is the library's built-in `static __device__` scratch array; the kernels are the ones ss_periodogram_ex
launches.  Checked here against the existing path (ss_periodogram_ex with its pooled cudaMalloc workspace) within the
bar the parity tests use (1e-9 relative + 1e-12 per periodogram value, identical best index), on two calls in a
row -- the second call finds the first call's contents in the scratch -- and for the free device memory staying put.

Collected last (file name) so that a failure here hides no other test under `pytest -x`; passes alone in a fresh
process and after the other tests.
"""
import numpy as np
import pytest

import ss_inputs

pytestmark = pytest.mark.gpu

CV, GV = 0, 1
RTOL, ATOL = 1e-9, 1e-12


@pytest.fixture(scope="module")
def ss():
    import torch
    assert torch.cuda.is_available()
    import paper_2111_07396_b200 as m
    m.load()
    return m


def _catalog():
    """Warp-path (config 3 shape) and group-path (config 4 shape) objects in one ragged catalog, plus an object with a
    duplicated time stamp (handed over whole to the generic kernel) and a degenerate one (n < 5: NaN row)."""
    a = ss_inputs.config3(n_objects=24, n_freq=700)
    b = ss_inputs.config4(n_objects=4, n_freq=700)
    rng = np.random.default_rng(4242)
    n = 90
    td = np.sort(rng.integers(0, 30, size=n) + rng.uniform(0.0, 0.33, size=n))
    td[11] = td[10]
    ed = rng.uniform(0.02, 0.1, size=n)
    yd = 15 + 0.3 * np.sin(2 * np.pi * td / 0.61) + rng.normal(0, 1.0, size=n) * ed
    tz, yz, ez = np.array([0.1, 0.7, 1.9]), np.array([15.0, 15.1, 14.9]), np.array([0.05, 0.05, 0.05])
    times = np.concatenate([a.times, b.times, td, tz])
    mags = np.concatenate([a.mags, b.mags, yd, yz])
    errs = np.concatenate([a.errs, b.errs, ed, ez])
    sizes = np.concatenate([np.diff(a.offsets), np.diff(b.offsets), [n, 3]])
    off = np.zeros(len(sizes) + 1, dtype=np.int64)
    off[1:] = np.cumsum(sizes)
    return times, mags, errs, off


@pytest.mark.parametrize("mode", [CV, GV])
def test_static_entry_point_matches_the_pooled_path_twice(ss, mode):
    import torch
    dev = torch.device("cuda")
    times, mags, errs, off = _catalog()
    n_obj, n_freq, f_min, f_max = len(off) - 1, 700, 0.5, 24.0
    t, y, e, o = (torch.as_tensor(v, device=dev) for v in (times, mags, errs, off))

    ref_pg = torch.empty((n_obj, n_freq), dtype=torch.float64, device=dev)
    ref_bf = torch.empty(n_obj, dtype=torch.float64, device=dev)
    ref_bi = torch.empty(n_obj, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, o, n_obj, f_min, f_max, n_freq, mode, ref_pg, ref_bf, ref_bi)
    torch.cuda.synchronize()
    ref = ref_pg.cpu().numpy()
    assert np.isfinite(ref[:-1]).all() and np.isnan(ref[-1]).all()

    pg = torch.empty_like(ref_pg)
    bf = torch.empty_like(ref_bf)
    bi = torch.empty_like(ref_bi)
    ss.release_workspace()                       # the pooled buffers of the reference call go back to the driver
    torch.cuda.synchronize()
    for call in range(2):
        pg.fill_(-7.0); bf.fill_(-7.0); bi.fill_(-7)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        ss.ss_periodogram_static(t, y, e, o, off, n_obj, f_min, f_max, n_freq, mode, pg, bf, bi)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, f"call {call}: the device's free memory changed"
        assert ss.last_launch_count() > 0
        got = pg.cpu().numpy()
        both_nan = np.isnan(got) & np.isnan(ref)
        assert not (np.isnan(got) ^ np.isnan(ref)).any(), f"call {call}"
        d = np.abs(got - ref)
        assert (d[~both_nan] <= (RTOL * np.abs(ref) + ATOL)[~both_nan]).all(), (call, np.nanmax(d))
        assert torch.equal(bi, ref_bi), f"call {call}"
        assert torch.equal(bf.nan_to_num(nan=-1.0), ref_bf.nan_to_num(nan=-1.0)), f"call {call}"
        if call == 0:
            # a different catalog in between: the second call must not depend on what the first left behind
            c = ss_inputs.config3(n_objects=40, n_freq=300)
            tc, yc, ec, oc = (torch.as_tensor(v, device=dev) for v in (c.times, c.mags, c.errs, c.offsets))
            pgc = torch.empty((c.n_objects, c.n_freq), dtype=torch.float64, device=dev)
            ss.ss_periodogram_static(tc, yc, ec, oc, np.ascontiguousarray(c.offsets, dtype=np.int64), c.n_objects,
                                     c.f_min, c.f_max, c.n_freq, 1 - mode, pgc, None, None)
            torch.cuda.synchronize()


def test_static_entry_point_rejects_what_does_not_fit(ss):
    """Beyond the built-in scratch: a clear SS_ERR_UNSUPPORTED before anything is written."""
    import torch
    dev = torch.device("cuda")
    assert ss.STATIC_SCRATCH_BYTES == 32 << 20
    n = 3_000_000                                 # 72 MB of centred catalog copy alone
    off = np.arange(0, n + 1, 100, dtype=np.int64)
    n_obj = len(off) - 1
    t = torch.zeros(n, dtype=torch.float64, device=dev)
    o = torch.as_tensor(off, device=dev)
    pg = torch.full((4,), -7.0, dtype=torch.float64, device=dev)
    with pytest.raises(ss.SSError) as ei:
        ss.ss_periodogram_static(t, t, t, o, off, n_obj, 0.5, 24.0, 10, CV, None, pg, None)
    assert ei.value.status == 4 and "built-in scratch" in str(ei.value)      # SS_ERR_UNSUPPORTED
    assert bool((pg == -7.0).all())
    # one long light curve: the cluster path's staging fallback space is far beyond the scratch
    off1 = np.array([0, 20000], dtype=np.int64)
    with pytest.raises(ss.SSError) as ei:
        ss.ss_periodogram_static(t, t, t, torch.as_tensor(off1, device=dev), off1, 1, 0.5, 24.0, 10, CV, None, pg, None)
    assert ei.value.status == 4
    with pytest.raises(TypeError):
        ss.ss_periodogram_static(t, t, t, o, None, n_obj, 0.5, 24.0, 10, CV, None, pg, None)
