"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Bar (BASELINE.json north_star):
    |P_gpu - P_ref| <= 1e-9*|P_ref| + 1e-12   per periodogram value,
    identical best-frequency index except ties within 1e-12.
An eval that misses the bar is re-examined with the definition oracle (long double window sums);
if its closest span pick is a near-tie (relative margin < 1e-9) it is "branch-ambiguous" (R29) and
must match the oracle's re-evaluation with that pick forced the other way.
"""
import numpy as np
import pytest

import oracle
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


def _tol(ref):
    return RTOL * np.abs(ref) + ATOL


def check_parity(cat, pg, ref, mode, max_ambiguous=3, label="", oracle_opts=None):
    """pg, ref: [n_objects, n_freq].  Returns number of branch-ambiguous evals."""
    assert pg.shape == ref.shape
    both_nan = np.isnan(pg) & np.isnan(ref)
    d = np.abs(pg - ref)
    bad = (d > _tol(ref)) & ~both_nan
    bad |= np.isnan(pg) ^ np.isnan(ref)
    ambiguous = 0
    for o, k in zip(*np.nonzero(bad)):
        t, y, e = cat.obj(int(o))
        f = oracle.freq(cat.f_min, cat.f_max, cat.n_freq, int(k))
        r = oracle.eval_one(t, y, e, f, mode=mode, variant=oracle.DEFINITION, alt_threshold=1e-7,
                            **(oracle_opts or {}))
        if abs(pg[o, k] - r["P"]) <= _tol(r["P"]):
            continue            # the fast oracle was the inexact side; the definition oracle agrees
        if r["margin"] < 1e-9 and abs(pg[o, k] - r["P_alt"]) <= _tol(r["P_alt"]):
            ambiguous += 1
            continue
        raise AssertionError(f"{label} obj {o} k {k}: gpu {pg[o, k]!r} oracle {r['P']!r} "
                             f"(fast {ref[o, k]!r}) margin {r['margin']:.3e}")
    assert ambiguous <= max_ambiguous, f"{label}: {ambiguous} branch-ambiguous evals"
    return ambiguous


def check_best(pg_ref, bi_gpu, bf_gpu, cat):
    """Best index identical to the oracle's, except ties within 1e-12 (R15)."""
    for o in range(pg_ref.shape[0]):
        row = pg_ref[o]
        if np.all(np.isnan(row)):
            assert bi_gpu[o] == -1 and np.isnan(bf_gpu[o])
            continue
        kb = int(np.argmax(row))
        kg = int(bi_gpu[o])
        if kg != kb:
            assert abs(row[kg] - row[kb]) <= 1e-12 * max(1.0, abs(row[kb])), (o, kg, kb, row[kg], row[kb])
        assert bf_gpu[o] == oracle.freq(cat.f_min, cat.f_max, cat.n_freq, kg)


def run_both(ss, cat, mode, variant, **opts):
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                         mode, **opts)
    assert ss.last_launch_count() > 0
    ref, bf, bi = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max,
                                     cat.n_freq, mode=mode, variant=variant)
    return res, ref


# ------------------------------------------------------------------ the five configs (reduced)
@pytest.mark.parametrize("mode", [CV, GV])
def test_config1_full(ss, mode):
    cat = ss_inputs.make(1)
    res, ref = run_both(ss, cat, mode, oracle.DEFINITION)
    check_parity(cat, res.pgram, ref, mode, label="cfg1")
    check_best(ref, res.best_index, res.best_freq, cat)
    assert abs(res.best_freq[0] - 1 / 0.37) < 0.01 * (1 / 0.37)


@pytest.mark.parametrize("mode", [CV, GV])
def test_config2_reduced(ss, mode):
    cat = ss_inputs.make(2).with_grid(n_freq=3001)
    res, ref = run_both(ss, cat, mode, oracle.FAST)
    check_parity(cat, res.pgram, ref, mode, label="cfg2")
    check_best(ref, res.best_index, res.best_freq, cat)


@pytest.mark.parametrize("mode", [CV, GV])
def test_config3_reduced(ss, mode):
    """96 ragged objects (n = 50..200 incl. both extremes), 1,537 frequencies over the config's range."""
    full = ss_inputs.config3(n_objects=400, n_freq=1537)
    ns = np.diff(full.offsets)
    pick = sorted(set(list(range(90)) + [int(np.argmin(ns)), int(np.argmax(ns))]
                      + [int(i) for i in np.nonzero(ns % 32 == 0)[0][:4]]))
    cat = full.subset(pick)
    res, ref = run_both(ss, cat, mode, oracle.DEFINITION)
    check_parity(cat, res.pgram, ref, mode, label="cfg3")
    check_best(ref, res.best_index, res.best_freq, cat)


@pytest.mark.parametrize("mode", [CV, GV])
def test_config4_reduced_and_planner_tiling(ss, mode):
    """8 objects of config 4 (n = 500..2000, heteroscedastic, one pure-noise object), 301 frequencies;
    the host entry point is forced to tile frequencies (cap and freq_tile) and must return the same
    bits as the untiled run."""
    full = ss_inputs.config4(n_objects=30, n_freq=301)
    ns = np.diff(full.offsets)
    pick = sorted(set([0, 1, 2, 9, 19, int(np.argmin(ns)), int(np.argmax(ns)), 29]))
    cat = full.subset(pick)
    res, ref = run_both(ss, cat, mode, oracle.FAST)
    check_parity(cat, res.pgram, ref, mode, label="cfg4")
    check_best(ref, res.best_index, res.best_freq, cat)
    tiled = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                           mode, freq_tile=37)
    assert np.array_equal(tiled.pgram, res.pgram)
    assert np.array_equal(tiled.best_index, res.best_index)
    # shrink the cap until the planner must tile frequencies by itself
    n_max = int(ns[pick].max())
    cap = ss.plan(cat.n_points, n_max, cat.n_objects, cat.n_freq, mode, cap_bytes=1 << 40,
                  host_tiles=True).total_bytes
    while True:
        cap -= 8 * cat.n_objects * 16
        p = ss.plan(cat.n_points, n_max, cat.n_objects, cat.n_freq, mode, cap_bytes=cap, host_tiles=True)
        if p.n_freq_tiles >= 3:
            break
    assert p.total_bytes <= cap
    capped = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                            mode, workspace_cap=cap)
    assert np.array_equal(capped.pgram, res.pgram)
    assert np.array_equal(capped.best_index, res.best_index)


@pytest.mark.parametrize("mode", [CV, GV])
def test_config5_reduced_global_staging(ss, mode):
    """n = 20,000 (exceeds one SM's shared memory -> SS_PATH_STAGE), 40 frequencies."""
    cat = ss_inputs.make(5).with_grid(n_freq=40)
    assert ss.path_for_n(20000) == ss.PATH_CLUSTER
    res, ref = run_both(ss, cat, mode, oracle.FAST)
    check_parity(cat, res.pgram, ref, mode, label="cfg5")
    check_best(ref, res.best_index, res.best_freq, cat)
    staged = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                            force_path=ss.PATH_STAGE)
    check_parity(cat, staged.pgram, ref, mode, label="cfg5/stage")
    check_best(ref, staged.best_index, staged.best_freq, cat)
    # two evals against the definition oracle (long double direct window sums)
    t, y, e = cat.obj(0)
    for k in (3, 31):
        f = oracle.freq(cat.f_min, cat.f_max, cat.n_freq, k)
        r = oracle.eval_one(t, y, e, f, mode=mode, variant=oracle.DEFINITION)
        assert abs(res.pgram[0, k] - r["P"]) <= _tol(r["P"])


# ------------------------------------------------------------------ one eval, element by element
@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("n", [5, 6, 7, 33, 100, 257, 1000])
def test_smooth_values_and_permutation(ss, mode, n):
    rng = np.random.default_rng(100 + n)
    t = np.sort(rng.uniform(0, 30, size=n))
    y = 15 + 0.4 * np.sin(2 * np.pi * t / 0.61) + rng.normal(0, 0.05, size=n)
    e = rng.uniform(0.01, 0.2, size=n)
    for f in (0.5, 1.639, 7.77):
        P, smo, perm = ss.debug_eval(t, y, e, f, mode)
        r = oracle.eval_one(t, y, e, f, mode=mode, variant=oracle.DEFINITION, want_smo=True)
        assert np.array_equal(perm, r["perm"])              # bit-exact fold + stable order (R2, R13)
        if r["margin"] < 1e-9:
            continue
        assert np.abs(smo - r["smo"]).max() < 1e-10
        assert abs(P - r["P"]) <= _tol(r["P"])


# ------------------------------------------------------------------ paths agree
@pytest.mark.parametrize("mode", [CV, GV])
def test_forced_paths_agree(ss, mode):
    cat = ss_inputs.config3(n_objects=12, n_freq=257)
    ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max,
                                   cat.n_freq, mode=mode, variant=oracle.DEFINITION)
    for path in (ss.PATH_WARP, ss.PATH_GROUP, ss.PATH_BLOCK, ss.PATH_STAGE):
        res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                             mode, force_path=path)
        check_parity(cat, res.pgram, ref, mode, label=f"path{path}")
        check_best(ref, res.best_index, res.best_freq, cat)


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("mode", [CV, GV])
def test_degenerate_objects_and_ragged_catalog(ss, mode):
    """Empty object, n < 5 (NaN row, index -1), n = 5, constant magnitudes (zeros), unsorted times."""
    rng = np.random.default_rng(7)
    ns = [0, 3, 5, 40, 4, 64, 0, 9]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        t = rng.uniform(0, 20, size=n)                      # NOT sorted in time
        y = 15 + 0.3 * np.sin(2 * np.pi * t / 0.8) + rng.normal(0, 0.03, size=n)
        if i == 5:
            y = np.full(n, 15.25)                           # constant => chi0 = 0 => zeros
        T.append(t); Y.append(y); E.append(np.full(n, 0.03))
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("edge", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.2, 6.0, 97, np.full(len(ns), np.nan))
    res, ref = run_both(ss, cat, mode, oracle.DEFINITION)
    for i, n in enumerate(ns):
        if n < 5:
            assert np.all(np.isnan(res.pgram[i])) and res.best_index[i] == -1 and np.isnan(res.best_freq[i])
    assert np.all(res.pgram[5] == 0.0) and res.best_index[5] == 0
    check_parity(cat, res.pgram, ref, mode, label="edge")
    check_best(ref, res.best_index, res.best_freq, cat)
    # nothing to do
    empty = ss.periodogram(np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(1, dtype=np.int64), 0.2, 6.0, 10, mode)
    assert empty.pgram.shape == (0, 10)


@pytest.mark.parametrize("mode", [CV, GV])
def test_equal_phases_and_tied_runs(ss, mode):
    """Integer-day time stamps: at f = 1 every phase is 0 (Listing 1 lines 25-36, weighted mean);
    at f = 0.5 and 0.25 the phases fall into 2 / 4 exactly tied runs (equal-x averaging, R24);
    duplicated observation times give tied pairs at every frequency."""
    rng = np.random.default_rng(8)
    n = 48
    t1 = np.arange(n, dtype=np.float64) + 1000.0
    y1 = 15 + rng.normal(0, 0.1, size=n)
    t2 = np.sort(rng.uniform(0, 25, size=60)); t2[10] = t2[9]; t2[31] = t2[30]; t2[32] = t2[30]
    y2 = 15 + 0.5 * np.sin(2 * np.pi * t2 / 1.3) + rng.normal(0, 0.05, size=60)
    off = np.array([0, n, n + 60], dtype=np.int64)
    cat = ss_inputs.Catalog("ties", np.concatenate([t1, t2]), np.concatenate([y1, y2]),
                            np.concatenate([rng.uniform(0.05, 0.2, size=n), np.full(60, 0.05)]), off,
                            0.25, 1.25, 4, np.array([np.nan, 1 / 1.3]))      # f = 0.25, 0.5, 0.75, 1.0
    assert oracle.freq(cat.f_min, cat.f_max, cat.n_freq, 3) == 1.0
    for path in (ss.PATH_AUTO, ss.PATH_GROUP, ss.PATH_BLOCK, ss.PATH_STAGE):
        res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                             mode, force_path=path)
        ref, bf, bi = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max,
                                         cat.n_freq, mode=mode, variant=oracle.DEFINITION)
        assert abs(res.pgram[0, 3]) < 1e-12                      # all phases equal: chi2 == chi0
        check_parity(cat, res.pgram, ref, mode, label=f"ties/path{path}")


@pytest.mark.parametrize("mode", [CV, GV])
def test_phase_clusters_below_the_sort_key_resolution(ss, mode):
    """The CTA kernels sort 32-bit keys (20-22 phase bits | index) and repair the order inside a quantisation
    bucket on the full phases.  Observation times 1e-9 d apart fold into one bucket with DISTINCT phases.
    (a) a reversed triple and a reversed pair (repaired by odd-even transposition): full parity at the bar;
    (b) plus a 40-point burst in reverse time order (does not settle in 12 passes -> exact network): the
    permutation equals the oracle's bit for bit, and every CTA size gives the same values.  (With 40
    coincident abscissae the fits themselves are ill-conditioned -- a 7-point window holding 6 of them leaves
    the seventh a leave-one-out denominator of 0 up to rounding -- so (b) pins the ORDER, not the values.)"""
    rng = np.random.default_rng(77)
    for n, path_list in ((700, (ss.PATH_AUTO, ss.PATH_BLOCK, ss.PATH_STAGE)), (120, (ss.PATH_AUTO, ss.PATH_GROUP, ss.PATH_BLOCK))):
        t = np.sort(rng.uniform(0, 40, size=n))
        t[10:13] = t[10] + np.array([2e-9, 1e-9, 0.0])                # triple, reversed
        t[30:32] = t[30] + np.array([1e-9, 0.0])                      # pair, reversed
        y = 15 + 0.3 * np.sin(2 * np.pi * t / 0.7) + rng.normal(0, 0.05, size=n)
        e = rng.uniform(0.02, 0.1, size=n)
        off = np.array([0, n], dtype=np.int64)
        cat = ss_inputs.Catalog("clusters", t, y, e, off, 0.2, 3.0, 64, np.array([1 / 0.7]))
        ref, _, _ = oracle.periodogram(t, y, e, off, 0.2, 3.0, 64, mode=mode, variant=oracle.DEFINITION)
        for path in path_list:
            res = ss.periodogram(t, y, e, off, 0.2, 3.0, 64, mode, force_path=path)
            check_parity(cat, res.pgram, ref, mode, label=f"clusters n={n} path{path}")
        # (b) the burst
        tb = t.copy()
        tb[60:100] = tb[60] + 1e-9 * np.arange(40)[::-1]
        Pk = []
        for k in (3, 17, 40):
            f = oracle.freq(0.2, 3.0, 64, k)
            P, smo, perm = ss.debug_eval(tb, y, e, f, mode)            # 512-thread CTA
            r = oracle.eval_one(tb, y, e, f, mode=mode, variant=oracle.DEFINITION, want_smo=True)
            assert np.array_equal(perm, r["perm"])
            Pk.append(P)
        for path in path_list:                                        # 128- / 256-thread CTAs, deferred hand-over
            res = ss.periodogram(tb, y, e, off, 0.2, 3.0, 64, mode, force_path=path)
            assert np.allclose(res.pgram[0, [3, 17, 40]], Pk, rtol=1e-9, atol=1e-12), (n, path)


def test_invalid_arguments(ss):
    t = np.linspace(0, 10, 20); y = np.sin(t); e = np.full(20, 0.1)
    off = np.array([0, 20], dtype=np.int64)
    def call(**kw):
        a = dict(times=t, mags=y, errs=e, offsets=off, f_min=0.1, f_max=2.0, n_freq=16)
        a.update(kw)
        return ss.periodogram(a["times"], a["mags"], a["errs"], a["offsets"], a["f_min"], a["f_max"], a["n_freq"])
    call()
    for kw in (dict(f_min=0.0), dict(f_min=-1.0), dict(f_max=0.05), dict(n_freq=0),
               dict(errs=np.where(np.arange(20) == 3, 0.0, e)), dict(errs=-e),
               dict(mags=np.where(np.arange(20) == 5, np.nan, y)),
               dict(times=np.where(np.arange(20) == 5, np.inf, t)),
               dict(offsets=np.array([0, 25, 20], dtype=np.int64))):
        with pytest.raises(ss.SSError) as ei:
            call(**kw)
        assert ei.value.status == ss.SS_ERR_INVALID_ARG, kw
    for kw in (dict(span=-0.1), dict(span=1.5), dict(span=float("nan")), dict(iper=0), dict(iper=3),
               dict(alpha=float("inf"))):
        with pytest.raises(ss.SSError) as ei:
            ss.periodogram(t, y, e, off, 0.1, 2.0, 16, **kw)
        assert ei.value.status == ss.SS_ERR_INVALID_ARG, kw


def test_alpha_option(ss):
    """alpha in (0,10] switches the bass enhancement; alpha = 0 disables it."""
    cat = ss_inputs.config3(n_objects=3, n_freq=64)
    for alpha in (0.0, 5.0, 10.0):
        res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                             CV, alpha=alpha)
        ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max,
                                       cat.n_freq, mode=CV, variant=oracle.DEFINITION, alpha=alpha)
        check_parity(cat, res.pgram, ref, CV, label=f"alpha{alpha}")


# ------------------------------------------------------------------ the options Listing 1 has
LISTING_OPTIONS = [dict(iper=2), dict(span=0.3), dict(iper=2, span=0.3), dict(span=1.0), dict(iper=2, span=1.0),
                   dict(iper=2, span=0.01), dict(iper=2, alpha=0.0)]


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("opts", LISTING_OPTIONS, ids=lambda o: ",".join(f"{k}={v}" for k, v in o.items()))
def test_periodic_windows_and_fixed_span(ss, mode, opts):
    """iper = 2 (windows wrap around phase 0/1) and span > 0 (one smooth at a fixed span,
    PAPER.md:202-210), alone and combined, on every path class that serves them: config-3-sized objects
    (shared-memory CTA kernel), config-4-sized objects (both CTA sizes) and the global-staging kernel."""
    small = ss_inputs.config3(n_objects=40, n_freq=129)
    ns = np.diff(small.offsets)
    cat = small.subset(sorted(set(list(range(10)) + [int(np.argmin(ns)), int(np.argmax(ns))])))
    ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                   mode=mode, variant=oracle.DEFINITION, **opts)
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
    assert ss.last_launch_count() > 0
    check_parity(cat, res.pgram, ref, mode, label=f"cfg3 {opts}", oracle_opts=opts)
    check_best(ref, res.best_index, res.best_freq, cat)
    staged = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                            force_path=ss.PATH_STAGE, **opts)
    check_parity(cat, staged.pgram, ref, mode, label=f"cfg3/stage {opts}", oracle_opts=opts)
    big = ss_inputs.config4(n_objects=12, n_freq=41)
    nb = np.diff(big.offsets)
    cat = big.subset(sorted(set([0, 9, int(np.argmin(nb)), int(np.argmax(nb))])))
    ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                   mode=mode, variant=oracle.FAST, **opts)
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
    check_parity(cat, res.pgram, ref, mode, label=f"cfg4 {opts}", oracle_opts=opts)
    check_best(ref, res.best_index, res.best_freq, cat)
    blk = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                         force_path=ss.PATH_BLOCK, **opts)
    check_parity(cat, blk.pgram, ref, mode, label=f"cfg4/cta {opts}", oracle_opts=opts)


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("opts", LISTING_OPTIONS, ids=lambda o: ",".join(f"{k}={v}" for k, v in o.items()))
def test_listing_options_on_the_group_path(ss, mode, opts):
    """iper = 2 / span > 0 for 256 < n <= 3,584 are served by group_kernel<.., OPT> (the wrapped part of a periodic
    window as a second range with shifted abscissae, found by arithmetic): one object per (G, C) variant, one with a
    duplicated time stamp (handed over whole), one with integer-day times that tie at f = 1 / d, against the oracle,
    best index included."""
    rng = np.random.default_rng(919)
    ns = [257, 384, 500, 513, 600, 640, 700, 768, 850, 1000, 1280, 1400, 1536, 1700, 1792, 2048, 2055, 2560, 3072, 3584,
          300, 420]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        t = np.sort(rng.integers(0, 900, size=n) + rng.uniform(0.0, 0.33, size=n))
        if i == len(ns) - 2:
            t[11] = t[10]                                   # duplicated time stamp
        if i == len(ns) - 1:
            t = np.arange(n, dtype=np.float64) + 0.25 * (np.arange(n) % 3 == 0)      # ties at f = 1
        e = rng.uniform(0.02, 0.1, size=n)
        y = 15 + rng.uniform(0.2, 0.8) * np.sin(2 * np.pi * t / np.exp(rng.uniform(np.log(0.3), np.log(2.0))) + i) \
            + rng.normal(0, 1.0, size=n) * e
        T.append(t); Y.append(y); E.append(e)
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("gopts", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.25, 4.25, 64, np.full(len(ns), np.nan))
    assert oracle.freq(cat.f_min, cat.f_max, cat.n_freq, 12) == 1.0
    ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                   mode=mode, variant=oracle.FAST, **opts)
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
    check_parity(cat, res.pgram, ref, mode, label=f"group-opt {opts}", oracle_opts=opts, max_ambiguous=4)
    check_best(ref, res.best_index, res.best_freq, cat)


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("n", [5, 6, 7, 8, 33, 100, 257, 1000])
def test_smooth_values_with_listing_options(ss, mode, n):
    """One eval, element by element, under each option set; includes duplicated times (tied phases)."""
    rng = np.random.default_rng(300 + n)
    t = np.sort(rng.uniform(0, 30, size=n))
    if n >= 33:
        t[7] = t[6]
    y = 15 + 0.4 * np.sin(2 * np.pi * t / 0.61) + rng.normal(0, 0.05, size=n)
    e = rng.uniform(0.01, 0.2, size=n)
    for opts in LISTING_OPTIONS:
        for f in (0.5, 1.639):
            P, smo, perm = ss.debug_eval(t, y, e, f, mode, **opts)
            r = oracle.eval_one(t, y, e, f, mode=mode, variant=oracle.DEFINITION, want_smo=True, **opts)
            assert np.array_equal(perm, r["perm"])
            if r["margin"] < 1e-9:
                continue
            # element bar: 1e-9 mag (7e-11 relative).  A 5-point window (span = 0.01) of heteroscedastic points
            # can be near-singular in x; prefix-sum differences in fp64 then keep ~10 digits of the slope where
            # the long-double definition oracle keeps 13.  The north_star bar is the one on P, held exactly.
            assert np.abs(smo - r["smo"]).max() < 1e-9, (opts, f)
            assert abs(P - r["P"]) <= _tol(r["P"]), (opts, f)


def test_periodic_config5_staging(ss):
    """n = 20,000 on the global-staging kernel with periodic windows, and with a fixed span."""
    cat = ss_inputs.make(5).with_grid(n_freq=6)
    for mode, opts in ((CV, dict(iper=2)), (GV, dict(iper=2)), (CV, dict(iper=2, span=0.1))):
        ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                       mode=mode, variant=oracle.FAST, **opts)
        res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
        check_parity(cat, res.pgram, ref, mode, label=f"cfg5 {opts}", oracle_opts=opts)


# ------------------------------------------------------------------ device-tensor entry point
@pytest.mark.parametrize("mode", [CV, GV])
def test_device_entry_point_matches_host_entry_point(ss, mode):
    import torch
    cat = ss_inputs.config3(n_objects=20, n_freq=333)
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.full((cat.n_objects, cat.n_freq), -7.0, dtype=torch.float64, device=dev)
    bf = torch.empty(cat.n_objects, dtype=torch.float64, device=dev)
    bi = torch.empty(cat.n_objects, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, bf, bi)
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode)
    assert np.array_equal(pg.cpu().numpy(), res.pgram)
    assert np.array_equal(bi.cpu().numpy(), res.best_index)
    assert np.array_equal(bf.cpu().numpy(), res.best_freq)
    # pgram_out = NULL: only the best frequency is produced
    bi2 = torch.empty_like(bi)
    ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, None, None, bi2)
    assert torch.equal(bi, bi2)
    # on a side stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        pg3 = torch.empty_like(pg)
        ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg3, None, None)
    s.synchronize()
    assert torch.equal(pg, pg3)


# ------------------------------------------------------------------ full size, bench.py's launch configuration
@pytest.mark.parametrize("mode", [CV, GV])
def test_config3_full_size_sampled(ss, mode):
    """Config 3 at BASELINE.json's full size (10,000 objects x 50,000 frequencies, 4 GB of output), launched
    exactly as bench.py launches it (device pointers, default options).  Checked on sampled outputs the
    oracle computes one by one: 400 random (object, k) evals plus four whole rows (shortest, longest and
    two mid-size objects) with their best-frequency index."""
    import torch
    cat = ss_inputs.config3()
    assert cat.n_objects == 10000 and cat.n_freq == 50000
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev)
    bf = torch.empty(cat.n_objects, dtype=torch.float64, device=dev)
    bi = torch.empty(cat.n_objects, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, bf, bi)
    torch.cuda.synchronize()
    assert ss.last_launch_count() > 0
    # properties that hold at any size
    assert bool(torch.isfinite(pg).all()) and float(pg.max()) <= 1.0 + 1e-12
    rowmax, rowarg = pg.max(dim=1)
    assert torch.equal(rowarg, bi)                      # first maximum of every row (torch.max returns the first)
    k_t = bi.to(torch.float64)
    assert torch.equal(bf, cat.f_min + k_t * ((cat.f_max - cat.f_min) / cat.n_freq))
    # sampled evals
    rng = np.random.default_rng(12345)
    objs = rng.integers(0, cat.n_objects, size=400); ks = rng.integers(0, cat.n_freq, size=400)
    got = pg[torch.as_tensor(objs, device=dev), torch.as_tensor(ks, device=dev)].cpu().numpy()
    ambiguous = 0
    for o, k, g in zip(objs, ks, got):
        tt, yy, ee = cat.obj(int(o))
        r = oracle.eval_one(tt, yy, ee, oracle.freq(cat.f_min, cat.f_max, cat.n_freq, int(k)), mode=mode,
                            variant=oracle.DEFINITION, alt_threshold=1e-7)
        if abs(g - r["P"]) <= _tol(r["P"]):
            continue
        assert r["margin"] < 1e-9 and abs(g - r["P_alt"]) <= _tol(r["P_alt"]), (o, k, g, r["P"], r["margin"])
        ambiguous += 1
    assert ambiguous <= 2
    # whole rows
    ns = np.diff(cat.offsets)
    rows = [int(np.argmin(ns)), int(np.argmax(ns)), 1234, 7777]
    sub = cat.subset(rows)
    ref, _, _ = oracle.periodogram(sub.times, sub.mags, sub.errs, sub.offsets, sub.f_min, sub.f_max, sub.n_freq,
                                   mode=mode, variant=oracle.FAST)
    got_rows = pg[torch.as_tensor(rows, device=dev)].cpu().numpy()
    check_parity(sub, got_rows, ref, mode, max_ambiguous=4, label="cfg3-full")
    check_best(ref, bi[torch.as_tensor(rows, device=dev)].cpu().numpy(),
               bf[torch.as_tensor(rows, device=dev)].cpu().numpy(), sub)
    del pg
    torch.cuda.empty_cache()


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("cfg", [2, 5])
def test_single_object_configs_full_size_sampled(ss, cfg, mode):
    """Configs 2 (n = 1,000 x 100,000 frequencies, shared-memory CTA kernel) and 5 (n = 20,000 x 1,000,000
    frequencies, global-staging kernel) at BASELINE.json's full sizes through the device entry point; checked on
    properties that hold at any size and on sampled evals the oracle computes one by one (its fp64 variant, itself
    held to the long-double variant by the pins and by the reduced-size tests above)."""
    import torch
    cat = ss_inputs.make(cfg)
    assert cat.n_freq == {2: 100000, 5: 1000000}[cfg]
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.empty((1, cat.n_freq), dtype=torch.float64, device=dev)
    bf = torch.empty(1, dtype=torch.float64, device=dev); bi = torch.empty(1, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, 1, cat.f_min, cat.f_max, cat.n_freq, mode, pg, bf, bi)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(pg).all()) and float(pg.max()) <= 1.0 + 1e-12
    assert int(torch.argmax(pg[0])) == int(bi[0])
    kb = int(bi[0])
    assert float(bf[0]) == oracle.freq(cat.f_min, cat.f_max, cat.n_freq, kb)
    # the injected period (or a harmonic / the 1-day alias structure around it) carries the highest power
    f_true = {2: 1 / 2.71, 5: 1 / 0.853}[cfg]
    ratio = float(bf[0]) / f_true
    assert min(abs(ratio - r) for r in (0.5, 1.0, 2.0, 3.0, 4.0)) < 0.02, ratio
    rng = np.random.default_rng(cfg)
    ks = np.unique(np.concatenate([rng.integers(0, cat.n_freq, size=60 if cfg == 2 else 24), [0, cat.n_freq - 1, kb]]))
    got = pg[0, torch.as_tensor(ks, device=dev)].cpu().numpy()
    tt, yy, ee = cat.obj(0)
    ambiguous = 0
    for k, g in zip(ks, got):
        r = oracle.eval_one(tt, yy, ee, oracle.freq(cat.f_min, cat.f_max, cat.n_freq, int(k)), mode=mode,
                            variant=oracle.FAST, alt_threshold=1e-7)
        if abs(g - r["P"]) <= _tol(r["P"]):
            continue
        assert r["margin"] < 1e-9 and abs(g - r["P_alt"]) <= _tol(r["P_alt"]), (cfg, k, g, r["P"], r["margin"])
        ambiguous += 1
    assert ambiguous <= 2


def test_workspace_is_reused_between_calls_and_can_be_released(ss):
    """Steady-state calls allocate nothing (the per-thread pool serves the workspace, the host entry point's
    catalog copy and output tiles); ss_release_workspace gives the memory back; results do not change."""
    import torch
    cat = ss_inputs.config3(n_objects=50, n_freq=401)
    ss.release_workspace()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    first = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, CV)
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 < free0                                   # the pool now holds the buffers
    for _ in range(3):
        again = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, CV)
        assert torch.cuda.mem_get_info()[0] == free1       # nothing allocated, nothing freed
        assert np.array_equal(again.pgram, first.pgram) and np.array_equal(again.best_index, first.best_index)
    # a smaller and a different-shaped request are served from the same buffers
    sub = cat.subset(list(range(10)))
    ss.periodogram(sub.times, sub.mags, sub.errs, sub.offsets, sub.f_min, sub.f_max, 100, GV)
    assert torch.cuda.mem_get_info()[0] == free1
    ss.release_workspace()
    assert torch.cuda.mem_get_info()[0] >= free0 - (1 << 20)
    after = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, CV)
    assert np.array_equal(after.pgram, first.pgram)


# ------------------------------------------------------------------ round 2: gaps the round-1 review found
@pytest.mark.parametrize("mode", [CV, GV])
def test_warp_variants_upper_range(ss, mode):
    """n = 201..256 on the path the library picks by itself: warp_kernel<7,5> serves 193..219 and <8,6> 220..256
    (220..224 because the tweeter half-width 6 does not fit 7 points per lane).  Full parity against the
    definition oracle, best index included."""
    rng = np.random.default_rng(2024)
    ns = [201, 219, 220, 224, 225, 240, 255, 256]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        assert ss.path_for_n(n) == ss.PATH_WARP
        t = np.sort(rng.integers(0, 30, size=n) + rng.uniform(0.0, 0.33, size=n))
        P = np.exp(rng.uniform(np.log(0.1), np.log(2.0)))
        y = 15 + rng.uniform(0.1, 1.0) * np.sin(2 * np.pi * t / P + i) + rng.normal(0, 0.05, size=n)
        T.append(t); Y.append(y); E.append(rng.uniform(0.02, 0.1, size=n))
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("upper", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.5, 24.0, 193, np.full(len(ns), np.nan))
    res, ref = run_both(ss, cat, mode, oracle.DEFINITION)
    check_parity(cat, res.pgram, ref, mode, label="n=201..256")
    check_best(ref, res.best_index, res.best_freq, cat)


def _commensurate_catalog():
    """Quarter-day time stamps (no duplicates): at every frequency j/64 with even j many phases tie exactly, so
    the warp path hands those evals over one by one; the signal has period 1 d, so the PEAK (f = 1.0 = f_32) is
    one of them.  Second object: the same with duplicated time stamps (handed over as whole work items).  Third:
    an ordinary object."""
    rng = np.random.default_rng(99)
    m = np.sort(rng.choice(120, size=100, replace=False))
    t1 = m / 4.0
    y1 = 15 + 0.4 * np.sin(2 * np.pi * t1 / 1.0 + 0.3) + rng.normal(0, 0.02, size=100)
    t2 = t1.copy(); t2[17] = t2[16]; t2[60] = t2[58]
    y2 = 15 + 0.4 * np.sin(2 * np.pi * t2 / 1.0 + 1.1) + rng.normal(0, 0.02, size=100)
    t3 = np.sort(rng.uniform(0, 30, size=77))
    y3 = 15 + 0.3 * np.sin(2 * np.pi * t3 / 1.31) + rng.normal(0, 0.03, size=77)
    off = np.array([0, 100, 200, 277], dtype=np.int64)
    return ss_inputs.Catalog("commensurate", np.concatenate([t1, t2, t3]), np.concatenate([y1, y2, y3]),
                             np.concatenate([np.full(100, 0.02), np.full(100, 0.02), np.full(77, 0.03)]), off,
                             0.5, 1.5, 64, np.array([1.0, 1.0, 1 / 1.31]))


@pytest.mark.parametrize("mode", [CV, GV])
def test_best_index_when_the_peak_is_a_handed_over_eval(ss, mode):
    """The argmax has three sources on the warp path: the warp kernel's own partial maxima, single evals recomputed
    by the generic kernel (merged through atomics) and whole work items recomputed by it (objects with duplicated
    time stamps).  Here the true peak of objects 0 and 1 is a handed-over eval: values AND best index against the
    oracle, on both entry points and with forced frequency tiles."""
    import torch
    cat = _commensurate_catalog()
    assert oracle.freq(cat.f_min, cat.f_max, cat.n_freq, 32) == 1.0
    ref, _, bi_ref = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                        mode=mode, variant=oracle.DEFINITION)
    assert bi_ref[0] == 32 and bi_ref[1] == 32                  # the peak sits on the tied frequency
    for opts in (dict(), dict(freq_tile=16), dict(freq_tile=5)):
        res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
        check_parity(cat, res.pgram, ref, mode, label=f"handed-over {opts}")
        check_best(ref, res.best_index, res.best_freq, cat)
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    for want_pg in (True, False):
        pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev) if want_pg else None
        bf = torch.empty(cat.n_objects, dtype=torch.float64, device=dev)
        bi = torch.empty(cat.n_objects, dtype=torch.int64, device=dev)
        ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, bf, bi)
        if want_pg:
            check_parity(cat, pg.cpu().numpy(), ref, mode, label="handed-over/device")
        check_best(ref, bi.cpu().numpy(), bf.cpu().numpy(), cat)
    # the generic kernel serves the handed-over work with the code of the CTA path: identical bits
    blk = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                         force_path=ss.PATH_BLOCK)
    assert np.array_equal(res.pgram[1], blk.pgram[1])           # the object with duplicated time stamps, whole


@pytest.mark.parametrize("mode", [CV, GV])
def test_hand_over_list_overflow_repeats_the_call_on_the_cta_path(ss, mode):
    """With the list shrunk to 8 entries (test hook `defer_capacity`) the commensurate catalog overflows it: the
    call must then return exactly what the CTA path returns, periodogram and best index, on both entry points."""
    import torch
    cat = _commensurate_catalog()
    blk = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                         force_path=ss.PATH_BLOCK)
    n_block = ss.last_launch_count()
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                         defer_capacity=8)
    assert np.array_equal(res.pgram, blk.pgram) and np.array_equal(res.best_index, blk.best_index)
    assert np.array_equal(res.best_freq, blk.best_freq)
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev)
    bi = torch.empty(cat.n_objects, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, None, bi,
                      ss.default_options(defer_capacity=8))
    assert np.array_equal(pg.cpu().numpy(), blk.pgram) and np.array_equal(bi.cpu().numpy(), blk.best_index)
    # and a list that is long enough is not an overflow: the warp path's own values stand (parity, not bits)
    ok = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                        defer_capacity=4096)
    assert np.allclose(ok.pgram, blk.pgram, rtol=1e-9, atol=1e-12) and n_block > 0


@pytest.mark.parametrize("mode", [CV, GV])
def test_config4_full_size_sampled(ss, mode):
    """Config 4 at BASELINE.json's full size (1,000 objects of 500..2,000 points x 500,000 frequencies, 4 GB of
    output: the config whose frequency range the planner tiles), device entry point, default options -- the launch
    configuration of `bench.py --config 4`.  Checked on properties that hold at any size, on 300 random
    (object, k) evals the definition oracle computes one by one, and on two whole rows (shortest and longest
    object) with their best index."""
    import torch
    cat = ss_inputs.config4()
    assert cat.n_objects == 1000 and cat.n_freq == 500000
    dev = torch.device("cuda")
    t = torch.as_tensor(cat.times, device=dev); y = torch.as_tensor(cat.mags, device=dev)
    e = torch.as_tensor(cat.errs, device=dev); off = torch.as_tensor(cat.offsets, device=dev)
    pg = torch.empty((cat.n_objects, cat.n_freq), dtype=torch.float64, device=dev)
    bf = torch.empty(cat.n_objects, dtype=torch.float64, device=dev)
    bi = torch.empty(cat.n_objects, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, cat.n_objects, cat.f_min, cat.f_max, cat.n_freq, mode, pg, bf, bi)
    torch.cuda.synchronize()
    assert ss.last_launch_count() > 0
    assert bool(torch.isfinite(pg).all()) and float(pg.max()) <= 1.0 + 1e-12
    rowmax, rowarg = pg.max(dim=1)
    assert torch.equal(rowarg, bi)
    assert torch.equal(bf, cat.f_min + bi.to(torch.float64) * ((cat.f_max - cat.f_min) / cat.n_freq))
    rng = np.random.default_rng(4321)
    objs = rng.integers(0, cat.n_objects, size=300); ks = rng.integers(0, cat.n_freq, size=300)
    got = pg[torch.as_tensor(objs, device=dev), torch.as_tensor(ks, device=dev)].cpu().numpy()
    ambiguous = 0
    for o, k, g in zip(objs, ks, got):
        tt, yy, ee = cat.obj(int(o))
        r = oracle.eval_one(tt, yy, ee, oracle.freq(cat.f_min, cat.f_max, cat.n_freq, int(k)), mode=mode,
                            variant=oracle.DEFINITION, alt_threshold=1e-7)
        if abs(g - r["P"]) <= _tol(r["P"]):
            continue
        assert r["margin"] < 1e-9 and abs(g - r["P_alt"]) <= _tol(r["P_alt"]), (o, k, g, r["P"], r["margin"])
        ambiguous += 1
    assert ambiguous <= 2
    ns = np.diff(cat.offsets)
    rows = [int(np.argmin(ns)), int(np.argmax(ns))]
    sub = cat.subset(rows)
    ref, _, _ = oracle.periodogram(sub.times, sub.mags, sub.errs, sub.offsets, sub.f_min, sub.f_max, sub.n_freq,
                                   mode=mode, variant=oracle.FAST)
    got_rows = pg[torch.as_tensor(rows, device=dev)].cpu().numpy()
    check_parity(sub, got_rows, ref, mode, max_ambiguous=6, label="cfg4-full")
    check_best(ref, bi[torch.as_tensor(rows, device=dev)].cpu().numpy(),
               bf[torch.as_tensor(rows, device=dev)].cpu().numpy(), sub)
    del pg
    torch.cuda.empty_cache()


@pytest.mark.parametrize("mode", [CV, GV])
def test_group_kernel_every_variant(ss, mode):
    """The G-warps-per-eval kernels, one object per (G, C) variant at both ends of its range of n (capacities 384,
    512, 640, 768 = 4 warps x 6 points, 1,024, 1,280, 1,536 = 8 x 6, 2,048, 2,560, and the long variants 3,072 and
    3,584 = 16 x 7 that gather y and w from global memory; the path ends at n = 3,584), heteroscedastic errors,
    config-4 time sampling; against the definition oracle, best index included."""
    rng = np.random.default_rng(515)
    ns = [257, 384, 385, 512, 513, 640, 641, 700, 768, 769, 1024, 1025, 1280, 1281, 1400, 1536, 1537, 2048, 2049, 2055,
          2056, 2560, 2561, 3072, 3073, 3554, 3584]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        assert ss.path_for_n(n) == ss.PATH_GROUP
        kept = np.nonzero(np.mod(np.arange(1827), 365.25) < 243.5)[0]
        t = np.sort(rng.choice(kept, size=n, replace=True) + rng.uniform(0.0, 0.3, size=n))
        P = np.exp(rng.uniform(np.log(0.1), np.log(2.0)))
        e = rng.uniform(0.01, 0.2, size=n)
        y = 15 + rng.uniform(0.1, 1.0) * np.sin(2 * np.pi * t / P + i) + rng.normal(0, 1.0, size=n) * e
        T.append(t); Y.append(y); E.append(e)
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("group", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.01, 10.0, 67, np.full(len(ns), np.nan))
    res, ref = run_both(ss, cat, mode, oracle.DEFINITION)
    check_parity(cat, res.pgram, ref, mode, label="group variants")
    check_best(ref, res.best_index, res.best_freq, cat)
    # small objects forced onto the group path (n below one warp's worth, n = 5)
    small = ss_inputs.config3(n_objects=6, n_freq=65)
    tiny_t = np.array([0.1, 0.9, 1.7, 3.2, 4.4]); tiny_y = 15 + np.array([0.1, -0.2, 0.3, 0.0, -0.1])
    times = np.concatenate([small.times, tiny_t]); mags = np.concatenate([small.mags, tiny_y])
    errs = np.concatenate([small.errs, np.full(5, 0.05)])
    offs = np.concatenate([small.offsets, [small.offsets[-1] + 5]])
    cat2 = ss_inputs.Catalog("group-small", times, mags, errs, offs, 0.5, 24.0, 65, np.full(7, np.nan))
    ref2, _, _ = oracle.periodogram(times, mags, errs, offs, 0.5, 24.0, 65, mode=mode, variant=oracle.DEFINITION)
    res2 = ss.periodogram(times, mags, errs, offs, 0.5, 24.0, 65, mode, force_path=ss.PATH_GROUP)
    check_parity(cat2, res2.pgram, ref2, mode, label="group small")
    check_best(ref2, res2.best_index, res2.best_freq, cat2)


@pytest.mark.parametrize("mode", [CV, GV])
def test_cluster_kernel_every_cluster_size(ss, mode):
    """The cluster-per-eval kernels: R = 2, 4, 8, 16 CTAs x C = 3, 4, 5 points per thread, an object at both ends of
    several capacities (3,072 ... 40,960 points), decade-long nightly sampling, against the oracle (its fp64 variant,
    held to the long-double one by the pins; the smallest object also against the long-double variant).  One object
    has two duplicated time stamps: every one of its evals is handed over to the global-staging kernel."""
    rng = np.random.default_rng(616)
    ns = [2056, 3072, 3073, 5120, 6000, 10240, 12288, 16385, 20480, 24577, 40960]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        assert ss.path_for_n(n) == (ss.PATH_CLUSTER if n > 3584 else ss.PATH_GROUP)      # forced below: every (R, C)
        t = np.sort(rng.integers(0, 3652, size=n) + rng.uniform(0.0, 0.3, size=n))
        if n == 6000:
            t[100] = t[99]; t[4000] = t[3999]
        P = np.exp(rng.uniform(np.log(0.2), np.log(2.0)))
        e = rng.uniform(0.01, 0.1, size=n)
        y = 15 + rng.uniform(0.1, 0.5) * np.sin(2 * np.pi * t / P + i) + rng.normal(0, 1.0, size=n) * e
        T.append(t); Y.append(y); E.append(e)
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("cluster", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.01, 20.0, 9, np.full(len(ns), np.nan))
    res, ref = run_both(ss, cat, mode, oracle.FAST, force_path=ss.PATH_CLUSTER)
    check_parity(cat, res.pgram, ref, mode, label="cluster variants")
    check_best(ref, res.best_index, res.best_freq, cat)
    t, y, e = cat.obj(0)
    for k in (2, 7):
        r = oracle.eval_one(t, y, e, oracle.freq(cat.f_min, cat.f_max, cat.n_freq, k), mode=mode, variant=oracle.DEFINITION)
        assert abs(res.pgram[0, k] - r["P"]) <= _tol(r["P"])


@pytest.mark.parametrize("mode", [CV, GV])
def test_top_k_peaks(ss, mode):
    """ss_periodogram_peaks: on the library's OWN periodogram the peak indices must be bit-identical to
    the definition written out (oracle.peaks, a plain Python loop); against the oracle's periodogram they agree
    wherever the oracle's row separates its peaks by more than the parity tolerance.  Covers rows with fewer peaks
    than asked for, NaN rows (n < 5), a constant row (all zeros: one flat top at index 0), n_peaks = 1 = the argmax,
    a one-column grid, and both entry points."""
    import torch
    cat = ss_inputs.config3(n_objects=24, n_freq=2000)
    # add a degenerate object (NaN row) and a constant one (row of zeros)
    times = np.concatenate([cat.times, [0.0, 1.0, 2.5], np.linspace(0, 20, 30)])
    mags = np.concatenate([cat.mags, [15.0, 15.1, 15.2], np.full(30, 15.5)])
    errs = np.concatenate([cat.errs, [0.1, 0.1, 0.1], np.full(30, 0.05)])
    off = np.concatenate([cat.offsets, [cat.offsets[-1] + 3, cat.offsets[-1] + 33]])
    res = ss.periodogram(times, mags, errs, off, cat.f_min, cat.f_max, cat.n_freq, mode)
    ref, _, _ = oracle.periodogram(times, mags, errs, off, cat.f_min, cat.f_max, cat.n_freq, mode=mode, variant=oracle.FAST)
    n_obj = len(off) - 1
    for k in (1, 3, 8, 13, 32):
        pi, pv, pf = ss.peaks(res.pgram, cat.f_min, cat.f_max, k)
        for o in range(n_obj):
            ei, ev = oracle.peaks(res.pgram[o], k)
            assert np.array_equal(pi[o], ei), (k, o)
            assert np.array_equal(pv[o], ev, equal_nan=True)
            ok = ei >= 0
            assert np.array_equal(pf[o][ok], [oracle.freq(cat.f_min, cat.f_max, cat.n_freq, int(j)) for j in ei[ok]])
            assert np.all(np.isnan(pf[o][~ok]))
            # against the oracle's own row: same peaks where its leading peaks are separated by more than the tolerance
            ri, rv = oracle.peaks(ref[o], k + 1)
            gaps = np.abs(np.diff(rv[~np.isnan(rv)]))
            if len(gaps) == k and np.all(gaps > 1e-6):
                assert np.array_equal(pi[o], ri[:k]), (k, o)
        assert np.all(pi[n_obj - 2] == -1) and np.all(np.isnan(pv[n_obj - 2]))            # NaN row
        assert pi[n_obj - 1][0] == 0 and np.all(pi[n_obj - 1][1:] == -1)                   # row of zeros: one flat top
        if k == 1:
            real = res.best_index >= 0
            assert np.array_equal(pi[real, 0], res.best_index[real])
    # device entry point, strided rows, a sub-range of the columns
    dev = torch.device("cuda")
    pg = torch.as_tensor(res.pgram, device=dev)
    di = torch.empty((n_obj, 5), dtype=torch.int64, device=dev)
    dv = torch.empty((n_obj, 5), dtype=torch.float64, device=dev)
    ss.ss_periodogram_peaks(pg, n_obj, 700, cat.n_freq, cat.f_min, cat.f_min + 700 * cat.df, 5, di, dv, None)
    for o in range(n_obj):
        ei, ev = oracle.peaks(res.pgram[o, :700], 5)
        assert np.array_equal(di[o].cpu().numpy(), ei) and np.array_equal(dv[o].cpu().numpy(), ev, equal_nan=True)
    one_i, one_v, _ = ss.peaks(res.pgram[:3, :1], cat.f_min, cat.f_max, 2)
    assert np.all(one_i[:, 0] == 0) and np.all(one_i[:, 1] == -1)
    with pytest.raises(ss.SSError):
        ss.peaks(res.pgram, cat.f_min, cat.f_max, 33)


# ------------------------------------------------------------------ the paper's FP32 switch
MIXED_ATOL = 2e-2      # the worst value: an isolated eval where fp32 rounding flips a span pick (measured 1.3e-3 CV,
                       # 8.5e-3 GV -- the GV score is a difference Syy - ybar Sy - b Sxy of nearly equal fp32 numbers)
MIXED_P999 = 2e-4      # 99.9 % of the values (measured 3e-5): fp32 unit roundoff 6e-8 x (prefix magnitude / window sum ~ 20
                       # for the tweeter span) x the cancellation in Sxx = Swxx - xbar Swx (~100) ~ 1e-4 on a slope
MIXED_MEDIAN = 2e-6    # the typical value (measured 2e-7)


@pytest.mark.parametrize("mode", [CV, GV])
def test_mixed_precision_mode(ss, mode):
    """precision = SS_PRECISION_MIXED: fp64 fold / sort / prefix accumulation, fp32 smoother,
    for n <= 3,584 (warp and group paths).  (a) every periodogram value within MIXED_ATOL of the fp64 ORACLE; (b) the
    paper's criterion: the best period within 3 % of the fp64 one for at least 93 % of the objects (the
    paper reports 93.0-95.4 %); (c) longer objects are served in fp64 and keep the fp64 bits."""
    cat = ss_inputs.config4(n_objects=40, n_freq=3000)
    small = ss_inputs.config3(n_objects=60, n_freq=3000)
    rng = np.random.default_rng(99)
    nl = 3700
    tl = np.sort(rng.integers(0, 2500, size=nl) + rng.uniform(0.0, 0.3, size=nl))
    el = rng.uniform(0.01, 0.2, size=nl)
    yl = 15 + 0.3 * np.sin(2 * np.pi * tl / 1.37) + rng.normal(0, 1.0, size=nl) * el
    times = np.concatenate([cat.times, small.times, tl]); mags = np.concatenate([cat.mags, small.mags, yl])
    errs = np.concatenate([cat.errs, small.errs, el])
    off = np.concatenate([cat.offsets, cat.offsets[-1] + small.offsets[1:], [cat.offsets[-1] + small.offsets[-1] + nl]])
    both = ss_inputs.Catalog("mixed", times, mags, errs, off, 0.01, 10.0, 3000, np.full(len(off) - 1, np.nan))
    f64 = ss.periodogram(times, mags, errs, off, both.f_min, both.f_max, both.n_freq, mode)
    mix = ss.periodogram(times, mags, errs, off, both.f_min, both.f_max, both.n_freq, mode, precision=ss.PRECISION_MIXED)
    ref, bf_ref, _ = oracle.periodogram(times, mags, errs, off, both.f_min, both.f_max, both.n_freq, mode=mode,
                                        variant=oracle.FAST)
    n_big, n_f32 = cat.n_objects, cat.n_objects + small.n_objects
    for lo, hi in ((0, n_big), (n_big, n_f32)):            # group path, warp path
        err = np.abs(mix.pgram[lo:hi] - ref[lo:hi])
        assert err.max() <= MIXED_ATOL, err.max()
        assert np.quantile(err, 0.999) <= MIXED_P999, np.quantile(err, 0.999)
        assert np.median(err) <= MIXED_MEDIAN, np.median(err)
        assert not np.array_equal(mix.pgram[lo:hi], f64.pgram[lo:hi])           # the fp32 smoother really ran
        match = np.abs(1.0 / mix.best_freq[lo:hi] - 1.0 / bf_ref[lo:hi]) <= 0.03 / bf_ref[lo:hi]
        assert match.mean() >= 0.93, match.mean()
    assert np.array_equal(mix.pgram[n_f32:], f64.pgram[n_f32:])                  # n > 3,584: fp64, same bits
    # every (G, C) variant of the float kernel
    rng = np.random.default_rng(717)
    ns = [40, 64, 65, 96, 100, 128, 150, 160, 170, 192, 200, 224, 250, 256,      # every warp variant (C, IBW0)
          257, 384, 500, 640, 700, 768, 1000, 1280, 1400, 1536, 2048, 2055, 2560, 3072, 3584]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        t = np.sort(rng.integers(0, 1200, size=n) + rng.uniform(0.0, 0.3, size=n))
        e = rng.uniform(0.01, 0.2, size=n)
        y = 15 + 0.4 * np.sin(2 * np.pi * t / 0.77 + i) + rng.normal(0, 1.0, size=n) * e
        T.append(t); Y.append(y); E.append(e)
    off2 = np.zeros(len(ns) + 1, dtype=np.int64); off2[1:] = np.cumsum(ns)
    t2, y2, e2 = np.concatenate(T), np.concatenate(Y), np.concatenate(E)
    mix2 = ss.periodogram(t2, y2, e2, off2, 0.01, 10.0, 61, mode, precision=ss.PRECISION_MIXED)
    ref2, _, _ = oracle.periodogram(t2, y2, e2, off2, 0.01, 10.0, 61, mode=mode, variant=oracle.FAST)
    assert np.abs(mix2.pgram - ref2).max() <= MIXED_ATOL, np.abs(mix2.pgram - ref2).max()
    with pytest.raises(ss.SSError):
        ss.periodogram(t2, y2, e2, off2, 0.01, 10.0, 61, mode, precision=7)


# ------------------------------------------------------------------ shared time sampling
def _shared_times_catalog(n_objects, n, seed, dup=False):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.integers(0, 30, size=n) + rng.uniform(0.0, 0.33, size=n))
    if dup:
        t[7] = t[6]
    T, Y, E = [], [], []
    for i in range(n_objects):
        P = np.exp(rng.uniform(np.log(0.1), np.log(2.0)))
        e = rng.uniform(0.02, 0.1, size=n)
        T.append(t); E.append(e)
        Y.append(15 + rng.uniform(0.1, 1.0) * np.sin(2 * np.pi * t / P + i) + rng.normal(0, 1.0, size=n) * e)
    off = np.arange(n_objects + 1, dtype=np.int64) * n
    return np.concatenate(T), np.concatenate(Y), np.concatenate(E), off


@pytest.mark.parametrize("mode", [CV, GV])
def test_shared_time_sampling_reuses_the_sort(ss, mode):
    """shared_times = 1: one fold + sort per frequency for 4 objects at a time.  Equal to the ordinary call (to rounding),
    parity with the oracle, for group sizes that do not divide the catalog, every points-per-lane variant, a shared
    sampling with a duplicated time stamp (every eval handed over) and tied phases at f = 1 / d on integer times;
    a catalog whose time stamps differ is refused."""
    # n <= 256: warp_shared_kernel; beyond: group_kernel<.., 3> (one (G, C) variant per warp count, and the largest)
    for n_objects, n, dup in ((37, 150, False), (9, 64, False), (6, 200, False), (5, 256, False), (7, 90, True),
                              (9, 700, False), (6, 1100, False), (5, 2055, False), (7, 400, True), (3, 257, False),
                              (5, 3000, False), (3, 3584, False)):
        t, y, e, off = _shared_times_catalog(n_objects, n, seed=n, dup=dup)
        plain = ss.periodogram(t, y, e, off, 0.5, 24.0, 131, mode)
        shared = ss.periodogram(t, y, e, off, 0.5, 24.0, 131, mode, shared_times=1)
        # the same arithmetic in the same order; the compiler is free to contract a*b+c differently in the two kernels
        # (seen: 4e-16 on P for the 8-points-per-lane variant, 2.6e-14 on P = 0.06 -- one ulp of chi2 -- for the 4-warp x
        # 3-point group kernel, whose two instantiations differ in register budget), so equality is to rounding, not to
        # the bit: three orders inside the parity bar
        assert np.allclose(shared.pgram, plain.pgram, rtol=1e-12, atol=1e-13), (n_objects, n)
        assert np.array_equal(shared.best_index, plain.best_index) and np.array_equal(shared.best_freq, plain.best_freq)
        if n_objects == 9:
            cat = ss_inputs.Catalog("shared", t, y, e, off, 0.5, 24.0, 131, np.full(n_objects, np.nan))
            ref, _, _ = oracle.periodogram(t, y, e, off, 0.5, 24.0, 131, mode=mode,
                                           variant=oracle.DEFINITION if n <= 256 else oracle.FAST)
            check_parity(cat, shared.pgram, ref, mode, label="shared times")
            check_best(ref, shared.best_index, shared.best_freq, cat)
    # integer-day times: at f = 1 every phase ties (handed over for the whole group); warp and group path
    for n in (300, 40):
        t1 = np.arange(n, dtype=np.float64) + 0.25 * (np.arange(n) % 3 == 0)
        rng = np.random.default_rng(3)
        T = np.tile(t1, 5); Y = 15 + rng.normal(0, 0.1, size=5 * n); E = np.full(5 * n, 0.05)
        off = np.arange(6, dtype=np.int64) * n
        plain = ss.periodogram(T, Y, E, off, 0.25, 1.25, 4, mode)
        shared = ss.periodogram(T, Y, E, off, 0.25, 1.25, 4, mode, shared_times=1)
        assert np.allclose(shared.pgram, plain.pgram, rtol=1e-12, atol=1e-13) and np.array_equal(shared.best_index, plain.best_index)
    # not actually shared
    T2 = T.copy(); T2[3 * n + 5] += 1e-9
    with pytest.raises(ss.SSError) as ei:
        ss.periodogram(T2, Y, E, off, 0.25, 1.25, 4, mode, shared_times=1)
    assert ei.value.status == ss.SS_ERR_INVALID_ARG
    ragged = np.array([0, n, 2 * n, 3 * n, 4 * n, 5 * n - 1], dtype=np.int64)
    with pytest.raises(ss.SSError):
        ss.periodogram(T[:5 * n - 1], Y[:5 * n - 1], E[:5 * n - 1], ragged, 0.25, 1.25, 4, mode, shared_times=1)


# ------------------------------------------------------------------ boundary: asynchronous call, caller workspace
def test_async_call_and_caller_workspace(ss):
    """ss_periodogram_ex with async_mode = 1 (skip_validation + offsets_host: nothing is read back) returns before the
    work is done and ss_synchronize() completes it; a caller-supplied device workspace of ss_workspace_bytes() bytes
    is enough for the call (and nothing is allocated), a smaller one is refused; both give the bits of the plain call."""
    import torch
    a = ss_inputs.config3(n_objects=300, n_freq=2000)
    b = ss_inputs.config4(n_objects=3, n_freq=2000)
    times = np.concatenate([a.times, b.times]); mags = np.concatenate([a.mags, b.mags]); errs = np.concatenate([a.errs, b.errs])
    offsets = np.concatenate([a.offsets, a.offsets[-1] + b.offsets[1:]])
    n_obj, n_freq = len(offsets) - 1, 2000
    dev = torch.device("cuda")
    t = torch.as_tensor(times, device=dev); y = torch.as_tensor(mags, device=dev)
    e = torch.as_tensor(errs, device=dev); off = torch.as_tensor(offsets, device=dev)
    ref_pg = torch.empty((n_obj, n_freq), dtype=torch.float64, device=dev)
    ref_bi = torch.empty(n_obj, dtype=torch.int64, device=dev)
    ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, ref_pg, None, ref_bi)
    # asynchronous on a side stream
    s = torch.cuda.Stream()
    pg = torch.zeros((n_obj, n_freq), dtype=torch.float64, device=dev)
    bi = torch.zeros(n_obj, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        o = ss.default_options(async_mode=1, skip_validation=1, offsets_host=offsets.ctypes.data)
        ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, pg, None, bi, o)
        returned_early = not s.query()          # ~0.1 s of kernels are still running when the call is back
    ss.synchronize()
    assert s.query()
    assert torch.equal(pg, ref_pg) and torch.equal(bi, ref_bi)
    assert returned_early
    with pytest.raises(ss.SSError):             # async needs skip_validation and offsets_host
        ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, pg, None, bi, ss.default_options(async_mode=1))
    # the next call completes a pending one implicitly
    pg.zero_()
    ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, pg, None, bi,
                      ss.default_options(async_mode=1, skip_validation=1, offsets_host=offsets.ctypes.data))
    res = ss.periodogram(times[:a.offsets[5]], mags[:a.offsets[5]], errs[:a.offsets[5]], a.offsets[:6], 0.5, 24.0, 50, CV)
    assert res.pgram.shape == (5, 50) and torch.equal(pg, ref_pg)
    # caller-supplied workspace
    need = ss.workspace_bytes(len(times), int(np.diff(offsets).max()), n_obj, n_freq, CV)
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    assert ws.data_ptr() % 256 == 0
    ss.release_workspace()
    free0 = torch.cuda.mem_get_info()[0]
    pg.zero_()
    ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, pg, None, bi,
                      ss.default_options(workspace=ws.data_ptr(), workspace_bytes=need))
    assert torch.equal(pg, ref_pg) and torch.equal(bi, ref_bi)
    assert torch.cuda.mem_get_info()[0] == free0            # the library allocated nothing
    with pytest.raises(ss.SSError) as ei:
        ss.ss_periodogram(t, y, e, off, n_obj, 0.5, 24.0, n_freq, CV, pg, None, bi,
                          ss.default_options(workspace=ws.data_ptr(), workspace_bytes=1 << 20))
    assert ei.value.status == ss.SS_ERR_OUT_OF_MEMORY


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("opts", LISTING_OPTIONS, ids=lambda o: ",".join(f"{k}={v}" for k, v in o.items()))
def test_listing_options_on_the_warp_path(ss, mode, opts):
    """iper = 2 / span > 0 for n <= 256 are served by warp_opt_kernel (every window by prefix differences through a
    table of two ranges per point): objects of every points-per-lane class (n = 5 .. 256, incl. n = 32 C exactly), an
    object with duplicated time stamps (handed over whole) and integer-day times that tie at f = 1 / d, against the
    definition oracle, best index included; and against the generic CTA kernel (forced) within the parity bar."""
    rng = np.random.default_rng(818)
    ns = [5, 6, 9, 31, 64, 65, 96, 100, 128, 150, 160, 192, 200, 224, 255, 256, 120, 48]
    T, Y, E = [], [], []
    for i, n in enumerate(ns):
        t = np.sort(rng.integers(0, 30, size=n) + rng.uniform(0.0, 0.33, size=n))
        if i == len(ns) - 2:
            t[11] = t[10]                                   # duplicated time stamp
        if i == len(ns) - 1:
            t = np.arange(n, dtype=np.float64) + 0.25 * (np.arange(n) % 3 == 0)      # ties at f = 1
        e = rng.uniform(0.02, 0.1, size=n)
        y = 15 + rng.uniform(0.2, 0.8) * np.sin(2 * np.pi * t / np.exp(rng.uniform(np.log(0.3), np.log(2.0))) + i) \
            + rng.normal(0, 1.0, size=n) * e
        T.append(t); Y.append(y); E.append(e)
    off = np.zeros(len(ns) + 1, dtype=np.int64); off[1:] = np.cumsum(ns)
    cat = ss_inputs.Catalog("opts", np.concatenate(T), np.concatenate(Y), np.concatenate(E), off,
                            0.25, 4.25, 64, np.full(len(ns), np.nan))
    assert oracle.freq(cat.f_min, cat.f_max, cat.n_freq, 12) == 1.0
    ref, _, _ = oracle.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq,
                                   mode=mode, variant=oracle.DEFINITION, **opts)
    res = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode, **opts)
    check_parity(cat, res.pgram, ref, mode, label=f"warp-opt {opts}", oracle_opts=opts, max_ambiguous=4)
    check_best(ref, res.best_index, res.best_freq, cat)
    blk = ss.periodogram(cat.times, cat.mags, cat.errs, cat.offsets, cat.f_min, cat.f_max, cat.n_freq, mode,
                         force_path=ss.PATH_BLOCK, **opts)
    check_parity(cat, blk.pgram, ref, mode, label=f"cta-opt {opts}", oracle_opts=opts, max_ambiguous=4)
