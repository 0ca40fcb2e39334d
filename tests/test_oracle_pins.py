"""Pins for the CPU oracle (oracle/ss_oracle.c) against things OTHER than itself:
closed forms, textbook/library routines, brute force, invariants and the numbers
the paper prints (SURVEY.md 8(c) "Pins").  CPU only.
"""
import os

import numpy as np
import pytest

import oracle
import ss_inputs

CV, GV = oracle.CV, oracle.GV
DEF, FAST = oracle.DEFINITION, oracle.FAST
SPANS = (0.05, 0.2, 0.5)
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _sorted_xyw(rng, n, hetero=True):
    x = np.sort(rng.uniform(0.0, 1.0, size=n))
    y = rng.normal(0.0, 1.0, size=n)
    w = rng.uniform(0.5, 400.0, size=n) if hetero else np.ones(n)
    return x, y, w


# ---------------------------------------------------------------- grid, fold, sort
def test_grid_matches_table2():
    """half-open grid, df = (f_max-f_min)/N_f (R1)."""
    for line in open(os.path.join(GOLD, "table2_grid.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, fmin, fmax, df, nf = line.split()
        fmin, fmax, df, nf = float(fmin), float(fmax), float(df), int(nf)
        got = (oracle.freq(fmin, fmax, nf, 1) - oracle.freq(fmin, fmax, nf, 0))
        assert abs(got - df) / df < 0.02, name          # the paper prints 2 digits
        assert oracle.freq(fmin, fmax, nf, 0) == fmin
        assert oracle.freq(fmin, fmax, nf, nf - 1) < fmax   # f_max itself is excluded


def test_fold_is_frac_and_in_unit_interval():
    rng = np.random.default_rng(10)
    tt = np.concatenate([[0.0], rng.uniform(0, 3652, size=5000), np.arange(50.0)])
    for f in (0.01, 0.37, 1.0, 2.5, 24.0, 19.999987):
        phi = oracle.fold(tt, f)
        assert np.all(phi >= 0.0) and np.all(phi < 1.0)
        p = tt * f                       # numpy rounds the product once, like the oracle (R2)
        assert np.array_equal(phi, p - np.floor(p))
        # agrees with the paper's (tt mod p)/p to rounding
        per = 1.0 / f
        ref = np.mod(tt, per) / per
        d = np.abs(phi - ref)
        d = np.minimum(d, 1.0 - d)       # wrap-around at 0/1
        assert d.max() < 1e-9


def test_argsort_is_stable():
    rng = np.random.default_rng(11)
    # integer-day times at f = 1 give exact ties; plus random phases
    tt = np.concatenate([np.arange(40.0), rng.uniform(0, 30, size=200), np.arange(40.0) + 0.5])
    rng.shuffle(tt)
    for f in (1.0, 2.0, 0.731):
        phi = oracle.fold(tt, f)
        perm = oracle.argsort(phi)
        assert np.array_equal(perm, np.argsort(phi, kind="stable"))


# ---------------------------------------------------------------- windows
@pytest.mark.parametrize("span", SPANS)
def test_window_rule_brute_force(span):
    """O4: symmetric window of 2*ibw+1 points, pinned to the first/last K points at the ends."""
    for n in range(5, 41):
        ibw = max(2, int(np.floor(0.5 * span * n + 0.5)))
        K = min(2 * ibw + 1, n)
        for j in range(n):
            # brute force: among all runs of K consecutive indices in [0,n), the one whose centre is
            # closest to j (ties cannot happen: K is odd unless clamped to n)
            cands = [(abs((lo + (K - 1) / 2.0) - j), lo) for lo in range(0, n - K + 1)]
            lo_ref = min(cands)[1]
            assert oracle.window(n, span, j) == (lo_ref, K), (n, j)


# ---------------------------------------------------------------- the smooth primitive
@pytest.mark.parametrize("variant", [DEF, FAST])
def test_line_is_reproduced_exactly(variant):
    rng = np.random.default_rng(12)
    x, _, w = _sorted_xyw(rng, 137)
    y = 3.25 - 1.75 * x
    for span in SPANS + (0.9,):
        smo, acvr = oracle.smooth(x, y, w, span, cv=True, variant=variant)
        assert np.abs(smo - y).max() < 1e-12
        assert np.abs(acvr).max() < 1e-10      # end points have leverage near 1
    for mode in (CV, GV):
        smo = oracle.supsmu(x, y, w, mode=mode, variant=variant)
        assert np.abs(smo - y).max() < 1e-11


@pytest.mark.parametrize("variant", [DEF, FAST])
def test_full_window_is_weighted_least_squares(variant):
    """span large enough that K = n  ==> ordinary WLS line (numpy.polyfit)."""
    rng = np.random.default_rng(13)
    x, y, w = _sorted_xyw(rng, 60)
    smo, _ = oracle.smooth(x, y, w, 2.5, variant=variant)
    b, a = np.polyfit(x, y, 1, w=np.sqrt(w))
    assert np.abs(smo - (a + b * x)).max() < 1e-11


@pytest.mark.parametrize("variant", [DEF, FAST])
def test_moving_average_special_cases(variant):
    rng = np.random.default_rng(14)
    n = 101
    x = (np.arange(n) + 0.5) / n
    y = rng.normal(size=n)
    w1 = np.ones(n)
    for span in SPANS:
        ibw = max(2, int(np.floor(0.5 * span * n + 0.5)))
        K = 2 * ibw + 1
        smo, _ = oracle.smooth(x, y, w1, span, variant=variant)
        # interior, equal spacing + equal weights: the line's value at the window centre is the mean
        ref = np.convolve(y, np.ones(K) / K, mode="valid")
        assert np.abs(smo[ibw:n - ibw] - ref).max() < 1e-12
        # slope guard tripped (huge vsmlsq): weighted moving average everywhere, windows pinned at ends
        w = rng.uniform(0.5, 4.0, size=n)
        smo, _ = oracle.smooth(x, y, w, span, vsmlsq=1e30, variant=variant)
        for j in range(n):
            lo = min(max(j - ibw, 0), n - K)
            ref_j = np.sum(w[lo:lo + K] * y[lo:lo + K]) / np.sum(w[lo:lo + K])
            assert abs(smo[j] - ref_j) < 1e-12
        # periodic windows on equally spaced phases: circular moving average at EVERY point
        smo, _ = oracle.smooth(x, y, w1, span, jper=2, variant=variant)
        yy = np.concatenate([y[-ibw:], y, y[:ibw]])
        ref = np.convolve(yy, np.ones(K) / K, mode="valid")
        assert np.abs(smo - ref).max() < 1e-12


@pytest.mark.parametrize("variant", [DEF, FAST])
def test_cv_residual_is_brute_force_leave_one_out(variant):
    """acvr_j = |y_j - prediction at x_j of the WLS line fitted to the same window WITHOUT point j|."""
    rng = np.random.default_rng(15)
    for n in (8, 13, 20):
        x, y, w = _sorted_xyw(rng, n)
        for span in (0.3, 0.5, 0.8):
            smo, acvr = oracle.smooth(x, y, w, span, cv=True, variant=variant)
            for j in range(n):
                lo, K = oracle.window(n, span, j)
                idx = [m for m in range(lo, lo + K) if m != j]
                b, a = np.polyfit(x[idx], y[idx], 1, w=np.sqrt(w[idx]))
                ref = abs(y[j] - (a + b * x[j]))
                assert abs(acvr[j] - ref) <= 1e-9 * max(1.0, ref), (n, span, j)


@pytest.mark.parametrize("variant", [DEF, FAST])
def test_equal_x_runs_share_one_value(variant):
    rng = np.random.default_rng(16)
    x, y, w = _sorted_xyw(rng, 90)
    x[10:14] = x[10]
    x[40:42] = x[40]
    x[88:90] = x[88]
    for mode in (CV, GV):
        smo = oracle.supsmu(x, y, w, mode=mode, variant=variant)
        for a, b in ((10, 14), (40, 42), (88, 90)):
            assert np.all(smo[a:b] == smo[a])
    # the primitive: the shared value is the w-weighted mean of the un-averaged line values
    smo, _ = oracle.smooth(x, y, w, 0.2, variant=variant)
    xx = x.copy()
    for k in range(1, 4):                               # break ties by 1 ulp steps
        xx[10 + k] = np.nextafter(xx[10 + k - 1], 2.0)
    assert np.all(np.diff(xx[10:14]) > 0)
    raw, _ = oracle.smooth(xx, y, w, 0.2, variant=variant)
    assert raw[10] != raw[13]
    assert abs(smo[10] - np.sum(w[10:14] * raw[10:14]) / np.sum(w[10:14])) < 1e-12


# ---------------------------------------------------------------- supsmu, both modes
@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("variant", [DEF, FAST])
def test_shift_and_scale_equivariance(mode, variant):
    rng = np.random.default_rng(17)
    x, y, w = _sorted_xyw(rng, 125)
    y = np.sin(6.0 * x) + 0.1 * y
    s0 = oracle.supsmu(x, y, w, mode=mode, variant=variant)
    # power-of-two scale of y: bit-identical
    assert np.array_equal(oracle.supsmu(x, 4.0 * y, w, mode=mode, variant=variant), 4.0 * s0)
    # power-of-two scale of w: same smooth to rounding (vsmlsq guard scales with w: R22)
    s2 = oracle.supsmu(x, y, 8.0 * w, mode=mode, variant=variant)
    assert np.abs(s2 - s0).max() < 1e-12
    # general affine map of y
    s3 = oracle.supsmu(x, 2.5 * y + 15.0, w, mode=mode, variant=variant)
    assert np.abs(s3 - (2.5 * s0 + 15.0)).max() < 1e-9


@pytest.mark.parametrize("mode", [CV, GV])
def test_all_phases_equal_gives_weighted_mean(mode):
    """Listing 1 lines 25-36: x[n-1] <= x[0] ==> smo = sum(wy)/sum(w).
    Reached with integer-day times at f = 1 / day."""
    rng = np.random.default_rng(18)
    n = 30
    t = np.arange(n) * 1.0 + 100.0
    y = 15 + rng.normal(size=n)
    e = rng.uniform(0.01, 0.2, size=n)
    r = oracle.eval_one(t, y, e, 1.0, mode=mode, want_smo=True)
    w = 1 / e ** 2
    assert np.abs(r["smo"] - np.sum(w * y) / np.sum(w)).max() < 1e-12
    assert abs(r["P"]) < 1e-12      # chi2 == chi0


def test_alpha_outside_0_10_disables_bass_enhancement():
    """the enhancement runs only for 0 < alpha <= 10."""
    rng = np.random.default_rng(19)
    x, y, w = _sorted_xyw(rng, 125)
    a0 = oracle.supsmu(x, y, w, alpha=0.0)
    a11 = oracle.supsmu(x, y, w, alpha=11.0)
    a9 = oracle.supsmu(x, y, w, alpha=9.0)
    assert np.array_equal(a0, a11)
    assert not np.array_equal(a0, a9)
    # alpha = 10: exponent 0 => span jumps to the woofer wherever another span won
    a10 = oracle.supsmu(x, y, w, alpha=10.0)
    assert not np.array_equal(a10, a9)


def test_listing1_plumbing_rebuilt_from_the_primitive():
    """Rebuild Listing 1 in numpy on top of the oracle's smooth primitive:
    catches scratch-index slips in the C supsmu (the primitive itself is pinned above)."""
    rng = np.random.default_rng(20)
    x, y, w = _sorted_xyw(rng, 125)
    y = np.sin(9.0 * x) + 0.2 * y
    n = len(x)
    scale = x[3 * (n // 4) - 1] - x[n // 4 - 1]
    v = 1e-6 * scale * scale
    A, R = [], []
    for s in SPANS:
        a, r = oracle.smooth(x, y, w, s, vsmlsq=v, cv=True)
        A.append(a)
        R.append(oracle.smooth(x, r, w, SPANS[1], vsmlsq=v)[0])
    R = np.array(R)
    c = np.argmin(R, axis=0)                      # first minimum wins (strict '<')
    resmin = R[c, np.arange(n)]
    sp = np.array(SPANS)[c]
    on = (resmin < R[2]) & (resmin > 0)
    sp = np.where(on, sp + (SPANS[2] - sp) * np.maximum(resmin / R[2], 1e-7) ** (10.0 - 9.0), sp)
    sps = np.clip(oracle.smooth(x, sp, w, SPANS[1], vsmlsq=v)[0], SPANS[0], SPANS[2])
    f = sps - SPANS[1]
    B = np.where(f < 0,
                 (1 - f / (SPANS[0] - SPANS[1])) * A[1] + f / (SPANS[0] - SPANS[1]) * A[0],
                 (1 - f / (SPANS[2] - SPANS[1])) * A[1] + f / (SPANS[2] - SPANS[1]) * A[2])
    ref = oracle.smooth(x, B, w, SPANS[0], vsmlsq=v)[0]
    got = oracle.supsmu(x, y, w, mode=CV)
    assert np.abs(got - ref).max() < 1e-13


def test_gv_score_is_window_rms_over_dof():
    """O6 (R12): G = sqrt(RSS/Sw)/(1 - p/K) with RSS the window's own WLS residual sum; checked by
    brute force through numpy.polyfit, then the span pick/interpolation rebuilt in numpy."""
    rng = np.random.default_rng(21)
    x, y, w = _sorted_xyw(rng, 64)
    y = np.cos(5.0 * x) + 0.3 * y
    n = len(x)
    A = np.empty((3, n)); G = np.empty((3, n))
    for i, s in enumerate(SPANS):
        for j in range(n):
            lo, K = oracle.window(n, s, j)
            sl = slice(lo, lo + K)
            b, a = np.polyfit(x[sl], y[sl], 1, w=np.sqrt(w[sl]))
            A[i, j] = a + b * x[j]
            rss = np.sum(w[sl] * (y[sl] - a - b * x[sl]) ** 2)
            G[i, j] = np.sqrt(rss / np.sum(w[sl])) / (1 - 2.0 / K)
    c = np.argmin(G, axis=0)
    resmin = G[c, np.arange(n)]
    sp = np.array(SPANS)[c]
    on = (resmin < G[2]) & (resmin > 0)
    sp = np.where(on, sp + (SPANS[2] - sp) * np.maximum(resmin / G[2], 1e-7), sp)
    sp = np.clip(sp, SPANS[0], SPANS[2])
    f = sp - SPANS[1]
    ref = np.where(f < 0,
                   (1 - f / (SPANS[0] - SPANS[1])) * A[1] + f / (SPANS[0] - SPANS[1]) * A[0],
                   (1 - f / (SPANS[2] - SPANS[1])) * A[1] + f / (SPANS[2] - SPANS[1]) * A[2])
    for variant in (DEF, FAST):
        got = oracle.supsmu(x, y, w, mode=GV, variant=variant)
        assert np.abs(got - ref).max() < 1e-9


# ---------------------------------------------------------------- fast vs definition
@pytest.mark.parametrize("mode", [CV, GV])
def test_fast_variant_matches_definition(mode):
    rng = np.random.default_rng(22)
    worst = 0.0
    for n in (5, 6, 7, 9, 50, 125, 200, 777, 2000):
        t = np.sort(rng.uniform(0, 30, size=n))
        y = 15 + 0.4 * np.sin(2 * np.pi * t / 0.61) + rng.normal(0, 0.05, size=n)
        e = rng.uniform(0.01, 0.2, size=n)
        for f in (0.5, 1.639, 7.77):
            a = oracle.eval_one(t, y, e, f, mode=mode, variant=DEF)
            b = oracle.eval_one(t, y, e, f, mode=mode, variant=FAST)
            if a["margin"] < 1e-9:
                continue
            worst = max(worst, abs(a["chi2"] - b["chi2"]) / a["chi2"])
    assert worst < 1e-11, worst


# ---------------------------------------------------------------- periodogram level
@pytest.mark.parametrize("shape", ["sin", "saw"])
@pytest.mark.parametrize("mode", [CV, GV])
def test_noiseless_period_recovery(shape, mode):
    """north_star: exact recovery of injected periods on noiseless sinusoids and sawtooths."""
    c = ss_inputs.make(1)
    t = c.times
    ph = np.mod(t / 0.37, 1.0)
    y = 15 + (0.3 * np.sin(2 * np.pi * ph) if shape == "sin" else 0.3 * (2 * ph - 1))
    pg, bf, bi = oracle.periodogram(t, y, c.errs, c.offsets, c.f_min, c.f_max, c.n_freq,
                                    mode=mode, variant=FAST)
    k_true = (1 / 0.37 - c.f_min) / c.df
    # the peak is ~1/T = 20 grid steps wide; the paper's own match criterion is 1 %
    assert abs(bi[0] - k_true) <= 2.0, (bi[0], k_true)
    assert abs(bf[0] - 1 / 0.37) <= 0.005 * (1 / 0.37)
    assert abs(bf[0] - (c.f_min + bi[0] * c.df)) < 1e-12
    assert pg[0, bi[0]] > 0.99
    assert bi[0] == int(np.argmax(pg[0]))          # first maximum (R15)


def test_statistic_definition_and_bounds():
    """O7: P = (chi0 - chi2)/chi0 with chi0 about the weighted mean; constant data => P = 0 rows."""
    c = ss_inputs.make(1)
    t, y, e = c.obj(0)
    r = oracle.eval_one(t, y, e, 2.7, want_smo=True)
    w = 1 / e ** 2
    ys = y[r["perm"]]
    chi2 = np.sum(w * (ys - r["smo"]) ** 2)
    yb = np.sum(w * y) / np.sum(w)
    chi0 = np.sum(w * (y - yb) ** 2)
    assert abs(r["chi2"] - chi2) < 1e-9 * chi2
    assert abs(r["P"] - (chi0 - chi2) / chi0) < 1e-12
    pg, bf, bi = oracle.periodogram(t, np.full_like(y, 15.0), e, c.offsets, 0.1, 10.0, 50)
    assert np.all(pg == 0.0) and bi[0] == 0
    # n < 5: NaN row, index -1 (R17)
    off = np.array([0, 4], dtype=np.int64)
    pg, bf, bi = oracle.periodogram(t[:4], y[:4], e[:4], off, 0.1, 10.0, 7)
    assert np.all(np.isnan(pg)) and bi[0] == -1 and np.isnan(bf[0])


def test_cv_and_gv_agree_on_noisy_config3_like_objects():
    """the single-pass variant finds the same periods about as often."""
    c = ss_inputs.config3(n_objects=12, n_freq=4000)
    agree = 0
    for mode_pair in [(CV, GV)]:
        _, bf_cv, _ = oracle.periodogram(c.times, c.mags, c.errs, c.offsets, c.f_min, c.f_max,
                                         c.n_freq, mode=CV)
        _, bf_gv, _ = oracle.periodogram(c.times, c.mags, c.errs, c.offsets, c.f_min, c.f_max,
                                         c.n_freq, mode=GV)
        agree = np.sum(np.abs(bf_cv - bf_gv) <= 0.01 * bf_cv)
    assert agree >= 9, agree


def test_forced_branch_alternative_differs_only_when_asked():
    """O9/R29 hook: P_alt is NaN unless the closest span pick is within the threshold; with a huge
    threshold the forced re-evaluation runs and (generically) differs slightly from P."""
    c = ss_inputs.make(1)
    t, y, e = c.obj(0)
    r = oracle.eval_one(t, y, e, 3.3, alt_threshold=0.0)
    assert np.isnan(r["P_alt"]) and r["margin"] > 0
    r = oracle.eval_one(t, y, e, 3.3, alt_threshold=1e9)
    assert np.isfinite(r["P_alt"]) and r["P_alt"] != r["P"] and abs(r["P_alt"] - r["P"]) < 0.05


# ---------------------------------------------------------------- Listing 1's options
def _periodic_window(x, j, ibw):
    """indices and abscissae of the periodic window j-ibw .. j+ibw (x wraps by -1 / +1), written out."""
    n = len(x)
    idx, xs = [], []
    for m in range(j - ibw, j + ibw + 1):
        if m < 0:
            idx.append(m + n); xs.append(x[m + n] - 1.0)
        elif m >= n:
            idx.append(m - n); xs.append(x[m - n] + 1.0)
        else:
            idx.append(m); xs.append(x[m])
    return np.array(idx), np.array(xs)


@pytest.mark.parametrize("variant", [DEF, FAST])
def test_periodic_smooth_is_brute_force_wls_on_wrapped_windows(variant):
    """jper = 2: the value at x_j is the WLS line over the 2*ibw+1 cyclic neighbours with wrapped
    abscissae, and the CV residual is the leave-one-out refit on that same window (numpy.polyfit)."""
    rng = np.random.default_rng(31)
    for n in (9, 14, 20, 37):
        x, y, w = _sorted_xyw(rng, n)
        for span in (0.3, 0.5, 0.8, 1.0):
            ibw = max(2, int(np.floor(0.5 * span * n + 0.5)))
            if 2 * ibw + 1 > n:
                ibw = (n - 1) // 2
            smo, acvr = oracle.smooth(x, y, w, span, jper=2, cv=True, variant=variant)
            for j in range(n):
                idx, xs = _periodic_window(x, j, ibw)
                b, a = np.polyfit(xs, y[idx], 1, w=np.sqrt(w[idx]))
                assert abs(smo[j] - (a + b * x[j])) < 1e-9, (n, span, j)
                keep = idx != j
                b, a = np.polyfit(xs[keep], y[idx][keep], 1, w=np.sqrt(w[idx][keep]))
                ref = abs(y[j] - (a + b * x[j]))
                assert abs(acvr[j] - ref) <= 1e-8 * max(1.0, ref), (n, span, j)


@pytest.mark.parametrize("mode", [CV, GV])
@pytest.mark.parametrize("variant", [DEF, FAST])
def test_periodic_supsmu_is_rotation_equivariant(mode, variant):
    """With iper = 2 the phase origin is arbitrary: x -> (x + c) mod 1 (re-sorted) rotates the smooth.
    (vsmlsq depends on the origin through the quartile points, but only as a threshold.)  The
    non-periodic smoother does NOT have this property -- checked too, so the pin can fail."""
    rng = np.random.default_rng(32)
    n = 120
    x, y, w = _sorted_xyw(rng, n)
    y = np.sin(2 * np.pi * x) + 0.1 * rng.normal(size=n)
    c = 0.37
    xr = (x + c) % 1.0
    order = np.argsort(xr, kind="stable")
    for opts in (dict(), dict(span=0.25), dict(alpha=0.0)):
        a = oracle.supsmu(x, y, w, mode=mode, iper=2, variant=variant, **opts)
        b = oracle.supsmu(xr[order], y[order], w[order], mode=mode, iper=2, variant=variant, **opts)
        assert np.abs(b - a[order]).max() < 1e-9, opts
    a = oracle.supsmu(x, y, w, mode=mode, iper=1, variant=variant)
    b = oracle.supsmu(xr[order], y[order], w[order], mode=mode, iper=1, variant=variant)
    assert np.abs(b - a[order]).max() > 1e-4


@pytest.mark.parametrize("mode", [CV, GV])
def test_fixed_span_is_one_smooth_in_both_modes(mode):
    """span > 0: supsmu returns S(y; span) with ties averaged, whatever the mode, and
    the periodogram's eval_one uses it; the whole-window span gives the global WLS line."""
    rng = np.random.default_rng(33)
    x, y, w = _sorted_xyw(rng, 80)
    q1 = 80 // 4 - 1; q3 = 3 * (q1 + 1) - 1
    vs = 1e-6 * (x[q3] - x[q1]) ** 2
    for iper in (1, 2):
        for span in (0.1, 0.45):
            full = oracle.supsmu(x, y, w, mode=mode, iper=iper, span=span)
            one, _ = oracle.smooth(x, y, w, span, jper=iper, vsmlsq=vs)
            assert np.array_equal(full, one)
    smo = oracle.supsmu(x, y, w, mode=mode, span=1.0)          # K clamps to n, window = everything
    b, a = np.polyfit(x, y, 1, w=np.sqrt(w))
    assert np.abs(smo - (a + b * x)).max() < 1e-11
    # fast variant agrees with the definition under the options too
    for opts in (dict(iper=2), dict(span=0.3), dict(iper=2, span=0.3)):
        d = oracle.supsmu(x, y, w, mode=mode, variant=DEF, **opts)
        f = oracle.supsmu(x, y, w, mode=mode, variant=FAST, **opts)
        assert np.abs(d - f).max() < 1e-10, opts
