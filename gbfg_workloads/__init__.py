"""Seeded synthetic workloads for libgbfg (BASELINE.json:configs[0..4]).

This module is the ONLY code shared by the oracle-side tests and the CUDA-side
tests/bench.  It holds workload *parameters* and seeded generators of raw
inputs (hand-made edge-case catalogs, the config-4 population table).  It holds
none of the method's arithmetic: no Philox, no binning rule, no deposit, no
median, no SNR.  Bin counts, catalogs drawn from the population and every
derived quantity are computed separately by `oracle/` and by the CUDA library.

Citations: BASELINE.json:configs[0..4]; PAPER.md:151
(T_obs = 4 yr), :166 (rho_th = 7), :552 (window ~2000), :549 (C = 729/512).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List

import numpy as np

YEAR_S = 3.15581e7            # BASELINE.json:configs[0] "T_obs = 1 yr (3.15581e7 s)"
MEDIAN_NORM_PAPER = 729.0 / 512.0   # PAPER.md:549 eq. (D3), nu = 2, exactly (1-1/9)^-3
SCALE_LOG2 = -140             # BASELINE.json:configs[0] "fixed scale of 2^-140 strain^2"


@dataclass(frozen=True)
class Population:
    """Lambda of BASELINE.json's generator (configs[0], configs[4])."""
    slope: float = 1.5          # p(f) ∝ f^-slope
    logA_offset: float = -22.5  # log10 A mean at 1 mHz
    logA_sigma: float = 0.4
    logMc_mean: float = float(np.log10(0.3))
    logMc_sigma: float = 0.2
    n_src: int = 0


@dataclass(frozen=True)
class Workload:
    name: str
    t_obs: float
    f_min: float
    f_max: float
    window: int
    rho_th: float
    max_iter: int
    seed: int
    pops: List[Population] = field(default_factory=list)
    median_norm: float = MEDIAN_NORM_PAPER
    scale_log2: int = SCALE_LOG2

    @property
    def n_cat(self) -> int:
        return len(self.pops)

    @property
    def n_src_total(self) -> int:
        return sum(p.n_src for p in self.pops)

    def offsets(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum([p.n_src for p in self.pops])]).astype(np.int64)


def _single(name, n, years, f_max, window, seed) -> Workload:
    return Workload(name=name, t_obs=years * YEAR_S, f_min=1e-4, f_max=f_max, window=window,
                    rho_th=7.0, max_iter=30, seed=seed, pops=[Population(n_src=int(n))])


def config4_population_table(n_cat: int = 64, seed: int = 4) -> List[Population]:
    """configs[4]: per-catalog Lambda drawn from the uniform prior box (harness-side,
    SURVEY.md §8(c) C1 last row).  numpy default_rng(seed); order of draws fixed here."""
    rng = np.random.default_rng(seed)
    pops = []
    for _ in range(n_cat):
        slope = rng.uniform(1.0, 2.0)
        off = rng.uniform(-23.0, -22.0)
        sig = rng.uniform(0.2, 0.6)
        mc = rng.uniform(-0.8, -0.2)
        n = int(np.floor(10.0 ** rng.uniform(6.0, 7.0)))
        pops.append(Population(slope=float(slope), logA_offset=float(off), logA_sigma=float(sig),
                               logMc_mean=float(mc), logMc_sigma=0.2, n_src=n))
    return pops


def config(i: int) -> Workload:
    """BASELINE.json:configs[i]."""
    if i == 0:
        return _single("cfg0_1e4_1yr", 1e4, 1, 10e-3, 1001, 0)
    if i == 1:
        return _single("cfg1_1e5_1yr", 1e5, 1, 10e-3, 1001, 1)
    if i == 2:
        return _single("cfg2_1e6_4yr", 1e6, 4, 30e-3, 2001, 2)
    if i == 3:
        return _single("cfg3_1e7_4yr", 1e7, 4, 30e-3, 2001, 3)
    if i == 4:
        w = _single("cfg4_batch64_4yr", 0, 4, 30e-3, 2001, 4)
        return replace(w, pops=config4_population_table(64, 4))
    raise ValueError(i)


def dense_case(kind: str = "short") -> Workload:
    """Extra parity cases on a narrow 1-yr band where the source density per bin is high, so the
    loop really iterates (configs 0-1 converge in 2-3 iterations; SURVEY.md §8(d) cfg-1 note).
    'short': 2e5 sources on 0.1-3 mHz (about 6 iterations); 'long': 3e5 louder sources on
    0.1-2 mHz (about 28 iterations, long tail)."""
    if kind == "short":
        w = _single("dense_short", 2e5, 1, 3e-3, 1001, 11)
        return w
    if kind == "long":
        w = _single("dense_long", 3e5, 1, 2e-3, 1001, 12)
        return replace(w, pops=[replace(w.pops[0], logA_offset=-22.3)])
    raise ValueError(kind)


def scaled(w: Workload, n_src: int | None = None, n_cat: int | None = None, name: str | None = None,
           **kw) -> Workload:
    """A reduced copy of a workload (fewer sources / catalogs) for parity cases and CPU samples."""
    pops = list(w.pops)
    if n_cat is not None:
        pops = pops[:n_cat]
    if n_src is not None:
        pops = [replace(p, n_src=int(n_src)) for p in pops]
    return replace(w, pops=pops, name=name or f"{w.name}_scaled", **kw)


def handmade_catalog(kind: str, w: Workload, n: int = 256, seed: int = 1234):
    """Raw (A, f, fdot) arrays for edge cases; plain numpy draws, no method arithmetic.

    kinds: 'narrow'  – fdot = 0 (one bin each), loud and quiet mixed
           'wide'    – very wide chirps incl. some running off the top of the band
           'bad'     – NaN / negative A / negative fdot / out-of-band f mixed with good ones
           'edges'   – sources at the first and last representable in-band frequencies
           'dupes'   – many identical sources in a handful of bins (contention, equal keys)
    """
    rng = np.random.default_rng(seed)
    span = w.f_max - w.f_min
    f = w.f_min + span * rng.random(n)
    A = 10.0 ** rng.uniform(-23.5, -20.5, n)
    fdot = np.zeros(n)
    if kind == "narrow":
        pass
    elif kind == "wide":
        fdot = 10.0 ** rng.uniform(-14.0, -10.5, n)
        f[: n // 8] = w.f_max - span * 1e-4 * rng.random(n // 8)   # clip at the top edge
    elif kind == "bad":
        fdot = 10.0 ** rng.uniform(-18.0, -13.0, n)
        bad = rng.integers(0, 6, n)
        A = np.where(bad == 1, -A, A)
        A = np.where(bad == 2, np.nan, A)
        fdot = np.where(bad == 3, -fdot, fdot)
        f = np.where(bad == 4, w.f_max + span * rng.random(n), f)
        f = np.where(bad == 5, w.f_min * 0.5, f)
        f[0] = np.nan
        fdot[1] = np.nan
        f[2] = w.f_max          # exactly f_max is outside [f_min, f_max)
        A[3] = 1e30             # quantised power overflows the int64 headroom
        fdot[4] = 1e300         # width overflows
    elif kind == "edges":
        f[0::4] = w.f_min
        f[1::4] = np.nextafter(w.f_max, 0.0)
        f[2::4] = np.nextafter(w.f_min, 1.0)
        fdot = 10.0 ** rng.uniform(-17.0, -13.0, n)
    elif kind == "dupes":
        f = w.f_min + span * rng.integers(1, 6, n) / 7.0
        A = np.full(n, 3e-22)
        fdot = np.where(rng.random(n) < 0.5, 0.0, 2.5e-14)
    else:
        raise ValueError(kind)
    return (np.ascontiguousarray(A, dtype=np.float64), np.ascontiguousarray(f, dtype=np.float64),
            np.ascontiguousarray(fdot, dtype=np.float64))


def random_spectrum(n: int, seed: int, kind: str = "lognormal") -> np.ndarray:
    """Raw int64 arrays to exercise the running median on its own."""
    rng = np.random.default_rng(seed)
    if kind == "lognormal":
        return np.floor(np.exp(rng.normal(10.0, 2.0, n))).astype(np.int64)
    if kind == "dupes":
        return rng.integers(0, 4, n).astype(np.int64)
    if kind == "zeros":
        x = rng.integers(0, 1 << 30, n).astype(np.int64)
        x[rng.random(n) < 0.7] = 0
        return x
    if kind == "full64":
        return rng.integers(-(1 << 62), 1 << 62, n, dtype=np.int64)
    if kind == "ramp":
        return np.arange(n, dtype=np.int64) * 3 - n
    if kind == "const":
        return np.full(n, 42, dtype=np.int64)
    if kind == "plateaus":          # what wide chirps leave: runs of equal values on a slowly drifting level
        runs = rng.integers(1, 60, n)
        vals = np.cumsum(rng.integers(-50, 51, n)) + 10_000
        return np.repeat(vals, runs)[:n].astype(np.int64)
    if kind == "straddle32":        # values on both sides of 2^32: the 32-bit-key path must hand the tile over
        return ((1 << 32) + rng.integers(-5000, 5000, n)).astype(np.int64)
    if kind == "negative":
        return rng.integers(-(1 << 20), 1 << 20, n).astype(np.int64)
    raise ValueError(kind)


def log_bin_edges(w: Workload, n_coarse: int = 100, f_lo: float | None = None, f_hi: float | None = None) -> np.ndarray:
    """Fine-bin index edges of n_coarse logarithmically spaced coarse bins over [f_lo, f_hi] (100 bins
    over 0.1-10 mHz; default: the workload's band).  Harness-side, handed to both the oracle and the library:
    coarse bin k holds the fine bins whose centre f_min + (i + 1/2)/T lies in [e_k, e_{k+1})."""
    f_lo = w.f_min if f_lo is None else f_lo
    f_hi = w.f_max if f_hi is None else f_hi
    n_bins = int(np.ceil((w.f_max - w.f_min) * w.t_obs))
    e = np.geomspace(f_lo, f_hi, n_coarse + 1)
    idx = np.ceil((e - w.f_min) * w.t_obs - 0.5).astype(np.int64)      # first bin whose centre is >= e_k
    return np.clip(idx, 0, n_bins)


@dataclass(frozen=True)
class PaperPopulation:
    """Lambda of the paper's own population model, eq. (9) PAPER.md:126 (Table I).  Defaults: the
    parameters of Fig. 1."""
    alpha_pl: float = -2.9
    alpha_gamma: float = 1.96
    beta_gamma: float = 1.8
    mu_gamma: float = -21.0
    mu: float = -22.0
    sigma: float = 0.18
    rho: float = 0.99
    n_src: int = 0


def paper_prior_draw(seed: int, n_src: int | None = None) -> PaperPopulation:
    """One draw of Lambda from the priors of Table I (harness-side, numpy default_rng)."""
    rng = np.random.default_rng(seed)
    return PaperPopulation(alpha_pl=float(rng.uniform(-4, -2)), alpha_gamma=float(rng.uniform(1, 3)),
                           beta_gamma=float(rng.uniform(1, 3)), mu_gamma=float(rng.uniform(-22, -20)),
                           mu=float(rng.uniform(-23, -21)), sigma=float(rng.uniform(0.1, 0.3)),
                           rho=float(rng.uniform(0, 1)),
                           n_src=int(rng.uniform(5e6, 30e6)) if n_src is None else int(n_src))
