"""ctypes binding of the CPU oracle (oracle/ss_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import build as _build

CV, GV = 0, 1
DEFINITION, FAST = 0, 1

_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.sso_window.argtypes = [C.c_int, C.c_double, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.sso_smooth.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp, C.c_double, C.c_int, C.c_double,
                                 C.c_int, _dp, _dp]
        L.sso_supsmu.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, C.c_int, C.c_double,
                                 C.c_double, _dp]
        L.sso_prep.argtypes = [C.c_int, _dp, _dp, _dp, _dp, _dp, C.POINTER(C.c_double),
                               C.POINTER(C.c_double)]
        L.sso_freq.argtypes = [C.c_double, C.c_double, C.c_int64, C.c_int64]
        L.sso_freq.restype = C.c_double
        L.sso_fold.argtypes = [C.c_int, _dp, C.c_double, _dp]
        L.sso_argsort.argtypes = [C.c_int, _dp, _ip]
        L.sso_eval.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, C.c_double, C.c_int,
                               C.c_double, C.c_double, C.c_double, _dp, C.c_void_p, C.c_void_p]
        L.sso_periodogram.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp, _lp, C.c_int64,
                                      C.c_double, C.c_double, C.c_int64,
                                      C.c_int64, C.c_int64, C.c_int64,
                                      C.c_int, C.c_double, C.c_double, C.c_int,
                                      _dp, _dp, _lp]
        L.sso_periodogram.restype = C.c_int
        L.sso_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def window(n, span, j):
    lo, K = C.c_int(), C.c_int()
    lib().sso_window(int(n), float(span), int(j), C.byref(lo), C.byref(K))
    return lo.value, K.value


def smooth(x, z, w, span, *, jper=1, vsmlsq=0.0, cv=False, variant=DEFINITION):
    """O4: S(z; span, cv).  Returns (smo, acvr or None)."""
    x, z, w = _f64(x), _f64(z), _f64(w)
    n = len(x)
    smo = np.empty(n)
    acvr = np.zeros(n)
    lib().sso_smooth(variant, n, x, z, w, float(span), int(jper), float(vsmlsq), int(bool(cv)), smo, acvr)
    return smo, (acvr if cv else None)


def supsmu(x, y, w, *, mode=CV, iper=1, span=0.0, alpha=9.0, variant=DEFINITION):
    """O5/O6 on sorted x."""
    x, y, w = _f64(x), _f64(y), _f64(w)
    smo = np.empty(len(x))
    lib().sso_supsmu(variant, mode, len(x), x, y, w, int(iper), float(span), float(alpha), smo)
    return smo


def prep(t, y, e):
    t, y, e = _f64(t), _f64(y), _f64(e)
    n = len(t)
    tt, w = np.empty(n), np.empty(n)
    yb, c0 = C.c_double(), C.c_double()
    lib().sso_prep(n, t, y, e, tt, w, C.byref(yb), C.byref(c0))
    return tt, w, yb.value, c0.value


def freq(f_min, f_max, n_freq, k):
    return lib().sso_freq(float(f_min), float(f_max), int(n_freq), int(k))


def fold(tt, f):
    tt = _f64(tt)
    phi = np.empty(len(tt))
    lib().sso_fold(len(tt), tt, float(f), phi)
    return phi


def argsort(phi):
    phi = _f64(phi)
    perm = np.empty(len(phi), dtype=np.int32)
    lib().sso_argsort(len(phi), phi, perm)
    return perm


def eval_one(t, y, e, f, *, mode=CV, variant=DEFINITION, iper=1, span=0.0, alpha=9.0,
             alt_threshold=1e-6, want_smo=False):
    """One (object, frequency) eval with diagnostics.
    Returns dict(P, chi2, margin, P_alt, guard_margin[, smo, perm])."""
    t, y, e = _f64(t), _f64(y), _f64(e)
    n = len(t)
    out = np.empty(5)
    smo = np.empty(n) if want_smo else None
    perm = np.empty(n, dtype=np.int32) if want_smo else None
    lib().sso_eval(variant, mode, n, t, y, e, float(f), int(iper), float(span), float(alpha),
                   float(alt_threshold), out,
                   smo.ctypes.data if want_smo else None, perm.ctypes.data if want_smo else None)
    r = dict(P=out[0], chi2=out[1], margin=out[2], P_alt=out[3], guard_margin=out[4])
    if want_smo:
        r["smo"], r["perm"] = smo, perm
    return r


def periodogram(times, mags, errs, offsets, f_min, f_max, n_freq, *, mode=CV, variant=FAST,
                k0=0, k_stride=1, k_count=None, iper=1, span=0.0, alpha=9.0, n_threads=None):
    """Algorithm 1 over a CSR catalog.  Returns (pgram[n_objects, k_count], best_freq, best_index)."""
    times, mags, errs = _f64(times), _f64(mags), _f64(errs)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n_obj = len(offsets) - 1
    if k_count is None:
        k_count = (int(n_freq) - k0 + k_stride - 1) // k_stride
    if n_threads is None:
        n_threads = max_threads()
    pg = np.empty((n_obj, k_count))
    bf = np.empty(n_obj)
    bi = np.empty(n_obj, dtype=np.int64)
    rc = lib().sso_periodogram(variant, mode, times, mags, errs, offsets, n_obj,
                               float(f_min), float(f_max), int(n_freq), int(k0), int(k_stride),
                               int(k_count), int(iper), float(span), float(alpha), int(n_threads),
                               pg, bf, bi)
    if rc != 0:
        raise RuntimeError("oracle failed")
    return pg, bf, bi


def max_threads():
    return min(lib().sso_max_threads(), os.cpu_count() or 1)


def peaks(row, n_peaks):
    """The n_peaks highest PEAKS of one periodogram row, written out (include/ss_periodogram.h, ss_periodogram_peaks;
    motivation PAPER.md:67, Fig. 1): k is a peak if P[k] > P[k-1] and P[k] >= P[k+1], a neighbour outside the grid
    does not disqualify, NaN never qualifies; ordered by falling power, equal powers by rising index; padded with
    index -1 / power NaN.  Plain Python loop: test infrastructure."""
    row = np.asarray(row, dtype=np.float64)
    n = len(row)
    found = []
    for k in range(n):
        left = row[k - 1] if k > 0 else -np.inf
        right = row[k + 1] if k + 1 < n else -np.inf
        if row[k] > left and row[k] >= right:
            found.append((-row[k], k))
    found.sort()
    idx = np.full(n_peaks, -1, dtype=np.int64)
    val = np.full(n_peaks, np.nan)
    for j, (nv, k) in enumerate(found[:n_peaks]):
        idx[j], val[j] = k, -nv
    return idx, val
