"""Seeded synthetic light-curve catalogs for the five BASELINE.json configs.

This module holds NO SuperSmoother arithmetic: it only draws times, magnitudes
and errors.  It is the single thing the CPU oracle's tests and the CUDA path's
tests/bench share (the same numpy arrays are handed to both sides), so no
cross-language RNG matching is needed.

The catalogs stand in for the paper's ObjSmall / ObjLarge / Stripe82 / TESS /
LINEAR data, none of which is available; the recipes are
SURVEY.md §8(d)'s concretisation of BASELINE.json `configs`, restated in
DESIGN.md.  Times are in days, magnitudes are semi-amplitudes around 15 mag.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

TWO_PI = 2.0 * np.pi


@dataclass
class Catalog:
    """CSR catalog + the frequency grid of one config (half-open [f_min, f_max))."""
    name: str
    times: np.ndarray      # float64[offsets[-1]]
    mags: np.ndarray       # float64[offsets[-1]]
    errs: np.ndarray       # float64[offsets[-1]]
    offsets: np.ndarray    # int64[n_objects + 1]
    f_min: float
    f_max: float
    n_freq: int
    true_freq: np.ndarray  # float64[n_objects], injected frequency (NaN = pure noise)

    @property
    def n_objects(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_points(self) -> int:
        return int(self.offsets[-1])

    @property
    def df(self) -> float:
        return (self.f_max - self.f_min) / self.n_freq

    def obj(self, i: int):
        a, b = int(self.offsets[i]), int(self.offsets[i + 1])
        return self.times[a:b], self.mags[a:b], self.errs[a:b]

    def subset(self, idx) -> "Catalog":
        """A new catalog holding only the objects in idx (same grid)."""
        idx = [int(i) for i in idx]
        t = [self.obj(i)[0] for i in idx]
        y = [self.obj(i)[1] for i in idx]
        e = [self.obj(i)[2] for i in idx]
        off = np.zeros(len(idx) + 1, dtype=np.int64)
        off[1:] = np.cumsum([len(a) for a in t])
        cat = lambda xs: (np.concatenate(xs) if xs else np.zeros(0))
        return Catalog(self.name + "/subset", cat(t), cat(y), cat(e), off,
                       self.f_min, self.f_max, self.n_freq,
                       self.true_freq[idx].copy())

    def with_grid(self, n_freq: int | None = None, k0: int = 0, k1: int | None = None) -> "Catalog":
        """Same objects, a sub-range [k0, k1) of the original grid (exact same f_k values
        cannot be guaranteed for a sub-range, so tests use this only to shrink work)."""
        if n_freq is not None:
            return Catalog(self.name, self.times, self.mags, self.errs, self.offsets,
                           self.f_min, self.f_max, int(n_freq), self.true_freq)
        k1 = self.n_freq if k1 is None else k1
        df = self.df
        return Catalog(self.name, self.times, self.mags, self.errs, self.offsets,
                       self.f_min + k0 * df, self.f_min + k1 * df, k1 - k0, self.true_freq)


def _shape(kind: int, phase: np.ndarray) -> np.ndarray:
    """Unit semi-amplitude light-curve shapes on phase in [0,1)."""
    if kind == 0:      # sinusoid
        return np.sin(TWO_PI * phase)
    if kind == 1:      # sawtooth
        return 2.0 * phase - 1.0
    # two Gaussian dips (eclipse-like), depths 1 and 0.6, sigma_phi = 0.03
    d1 = np.minimum(np.abs(phase - 0.25), 1.0 - np.abs(phase - 0.25))
    d2 = np.minimum(np.abs(phase - 0.75), 1.0 - np.abs(phase - 0.75))
    return 1.0 * np.exp(-0.5 * (d1 / 0.03) ** 2) + 0.6 * np.exp(-0.5 * (d2 / 0.03) ** 2)


def _kept_nights(rng, n_nights: int, dropout: float) -> np.ndarray:
    nights = np.arange(n_nights)
    in_season = np.mod(nights, 365.25) < 243.5          # 8-month season, 4-month gap
    up = rng.uniform(size=n_nights) >= dropout
    return nights[in_season & up]


def config1(seed: int = 0) -> Catalog:
    rng = np.random.default_rng(seed)
    n = 100
    night = rng.integers(0, 10, size=n)
    t = np.sort(night + rng.uniform(0.0, 0.25, size=n))
    y = 15.0 + 0.3 * np.sin(TWO_PI * t / 0.37) + rng.normal(0.0, 0.02, size=n)
    e = np.full(n, 0.02)
    return Catalog("cfg1", t, y, e, np.array([0, n], dtype=np.int64), 0.1, 10.0, 2000,
                   np.array([1.0 / 0.37]))


def config2(seed: int = 1) -> Catalog:
    rng = np.random.default_rng(seed)
    n = 1000
    kept = _kept_nights(rng, 1096, 0.3)
    t = np.sort(rng.choice(kept, size=n, replace=True) + rng.uniform(0.0, 0.3, size=n))
    ph = np.mod(t / 2.71, 1.0)
    y = 15.0 + 0.5 * (2.0 * ph - 1.0) + rng.normal(0.0, 0.03, size=n)
    e = np.full(n, 0.03)
    return Catalog("cfg2", t, y, e, np.array([0, n], dtype=np.int64), 0.05, 20.0, 100000,
                   np.array([1.0 / 2.71]))


def config3(seed: int = 2, n_objects: int = 10000, n_freq: int = 50000) -> Catalog:
    rng = np.random.default_rng(seed)
    ns = rng.integers(50, 201, size=n_objects)
    off = np.zeros(n_objects + 1, dtype=np.int64)
    off[1:] = np.cumsum(ns)
    T = np.empty(off[-1]); Y = np.empty(off[-1]); E = np.empty(off[-1])
    ftrue = np.empty(n_objects)
    for i in range(n_objects):
        n = int(ns[i])
        night = rng.integers(0, 30, size=n)
        t = np.sort(night + rng.uniform(0.0, 0.33, size=n))
        P = np.exp(rng.uniform(np.log(0.1), np.log(2.0)))
        amp = rng.uniform(0.1, 1.0)
        sig = rng.uniform(0.02, 0.1)
        y = 15.0 + amp * _shape(i % 3, np.mod(t / P, 1.0)) + rng.normal(0.0, sig, size=n)
        a, b = off[i], off[i + 1]
        T[a:b] = t; Y[a:b] = y; E[a:b] = sig
        ftrue[i] = 1.0 / P
    return Catalog("cfg3", T, Y, E, off, 0.5, 24.0, n_freq, ftrue)


def config4(seed: int = 3, n_objects: int = 1000, n_freq: int = 500000) -> Catalog:
    rng = np.random.default_rng(seed)
    ns = rng.integers(500, 2001, size=n_objects)
    off = np.zeros(n_objects + 1, dtype=np.int64)
    off[1:] = np.cumsum(ns)
    T = np.empty(off[-1]); Y = np.empty(off[-1]); E = np.empty(off[-1])
    ftrue = np.empty(n_objects)
    for i in range(n_objects):
        n = int(ns[i])
        kept = _kept_nights(rng, 1827, 0.3)
        t = np.sort(rng.choice(kept, size=n, replace=True) + rng.uniform(0.0, 0.3, size=n))
        P = np.exp(rng.uniform(np.log(0.1), np.log(2.0)))
        amp = rng.uniform(0.1, 1.0)
        e = rng.uniform(0.01, 0.2, size=n)
        noise = rng.normal(0.0, 1.0, size=n) * e
        if i % 10 == 9:
            y = 15.0 + noise
            ftrue[i] = np.nan
        else:
            y = 15.0 + amp * _shape(i % 3, np.mod(t / P, 1.0)) + noise
            ftrue[i] = 1.0 / P
        a, b = off[i], off[i + 1]
        T[a:b] = t; Y[a:b] = y; E[a:b] = e
    return Catalog("cfg4", T, Y, E, off, 0.01, 10.0, n_freq, ftrue)


def config5(seed: int = 4, n: int = 20000, n_freq: int = 1000000) -> Catalog:
    rng = np.random.default_rng(seed)
    t = np.sort(rng.integers(0, 3652, size=n) + rng.uniform(0.0, 0.3, size=n))
    amps = (0.3, 0.15, 0.08, 0.04)
    psi = rng.uniform(0.0, TWO_PI, size=4)
    y = np.full(n, 15.0)
    for h in range(4):
        y += amps[h] * np.sin(TWO_PI * (h + 1) * t / 0.853 + psi[h])
    y += 0.05 * np.sin(TWO_PI * t / 1.0) + rng.normal(0.0, 0.02, size=n)
    e = np.full(n, 0.02)
    return Catalog("cfg5", t, y, e, np.array([0, n], dtype=np.int64), 0.01, 20.0, n_freq,
                   np.array([1.0 / 0.853]))


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make(cfg: int, **kw) -> Catalog:
    return CONFIGS[cfg](**kw)
