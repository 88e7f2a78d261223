"""Pins for the oracle's stages (ii) deposit and (iii) running median + PSD."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import ndimage

import gbfg_workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def _grid(orc, i=0):
    w = W.config(i)
    return w, orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)


def test_n_bins_of_the_configs(orc):
    # 312 426 bins (configs 0-1), 3 774 349 bins (configs 2-4); ~3.1e5 per BASELINE.json:configs[0]
    assert _grid(orc, 0)[1].n_bins == 312426
    assert _grid(orc, 2)[1].n_bins == 3774349
    assert orc.make_grid(0.0, 1.0, 10.0).n_bins == 10          # exact product: no extra bin


def test_worked_examples(orc):
    w, g = _grid(orc, 0)
    s_instr = orc.instrument_noise(g)
    for row in _rows("worked_sources.txt"):
        A, f, fd = map(float, row[:3])
        k0, wid = int(row[3]), int(row[4])
        P, p, q, s_at, r2 = float(row[5]), float(row[6]), int(row[7]), float(row[8]), float(row[9])
        st, gk0, gw, gwe, gp, gq = orc.source_bins(g, A, f, fd)
        assert st == 0 and gk0 == k0 and gw == wid and gwe == wid
        assert abs(gp * gw / P - 1) < 1e-6 and abs(gp / p - 1) < 1e-6
        assert abs(gq - q) <= 1                              # q tabulated from a 7-digit p
        assert abs(s_instr[k0] / s_at - 1) < 1e-9
        assert abs(orc.rho2(g, A, f, fd, s_instr) / r2 - 1) < 1e-6


def _exact_triple(g, A, f, fd):
    """Independent statement of DESIGN.md R2 with exact rationals for the quantisation."""
    T = g.t_obs
    k0 = math.floor((f - g.f_min) * T)
    w = max(1, math.ceil(fd * (T * T)))
    p = ((A * A) * (0.5 * T)) / float(w)
    x = Fraction(p) * (1 << (-g.scale_log2))
    q = int(x)
    rem = x - q
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and q % 2 == 1):
        q += 1
    return k0, w, p, q


def test_deposit_brute_force_and_identities(orc):
    w, g = _grid(orc, 0)
    from dataclasses import replace
    pop = replace(w.pops[0], n_src=3000)
    A, f, fd = orc.sample_catalog(g, pop, 0, 42)
    A2, f2, fd2 = W.handmade_catalog("wide", w, 300)
    A, f, fd = np.concatenate([A, A2]), np.concatenate([f, f2]), np.concatenate([fd, fd2])
    spec = np.zeros(g.n_bins, dtype=np.int64)
    assert orc.deposit(g, A, f, fd, spec) == 0
    brute = {}
    diff = np.zeros(g.n_bins + 1, dtype=np.int64)
    total = 0
    clipped = 0
    for a, ff, d in zip(A, f, fd):
        k0, wid, p, q = _exact_triple(g, float(a), float(ff), float(d))
        w_eff = min(wid, g.n_bins - k0)
        clipped += w_eff < wid
        for k in range(k0, k0 + w_eff):
            brute[k] = brute.get(k, 0) + q
        diff[k0] += q
        diff[k0 + w_eff] -= q
        total += q * w_eff
        st, gk0, gw, gwe, gp, gq = orc.source_bins(g, float(a), float(ff), float(d))
        assert (st, gk0, gw, gwe, gp, gq) == (0, k0, wid, w_eff, p, q)
    assert clipped > 0                                         # the 'wide' set runs off the top of the band
    dense = np.zeros(g.n_bins, dtype=np.int64)
    for k, v in brute.items():
        dense[k] = v
    assert np.array_equal(spec, dense)
    assert np.array_equal(spec, np.cumsum(diff)[:-1])          # range-update form == per-bin adds
    assert int(spec.sum()) == total
    # subtracting the same set returns exactly zero; a selection list addresses sources by index
    sel = np.arange(0, A.size, 3, dtype=np.int64)
    part = np.zeros_like(spec)
    orc.deposit(g, A, f, fd, part, sel=sel)
    only = np.zeros_like(spec)
    orc.deposit(g, A[sel], f[sel], fd[sel], only)
    assert np.array_equal(part, only)
    orc.deposit(g, A, f, fd, spec, sign=-1)
    assert not spec.any()


def test_deposit_rejects_bad_sources(orc):
    w, g = _grid(orc, 0)
    A, f, fd = W.handmade_catalog("bad", w, 600)
    spec = np.zeros(g.n_bins, dtype=np.int64)
    rejected = orc.deposit(g, A, f, fd, spec)
    good = (A >= 0) & (fd >= 0) & (f >= w.f_min) & (f < w.f_max)
    good[3] = False      # range: quantised power too large
    good[4] = False      # range: width too large
    assert rejected == int((~good).sum()) and 0 < rejected < 600
    ref = np.zeros_like(spec)
    orc.deposit(g, A[good], f[good], fd[good], ref)
    assert np.array_equal(spec, ref)
    assert orc.source_bins(g, 1e-22, w.f_max, 0.0)[0] == 1
    assert orc.source_bins(g, float("nan"), 1e-3, 0.0)[0] == 1
    assert orc.source_bins(g, 1e30, 1e-3, 0.0)[0] == 2
    assert orc.source_bins(g, 1e-22, 1e-3, 1e300)[0] == 2
    st, k0, wd, we, p, q = orc.source_bins(g, 0.0, w.f_min, 0.0)
    assert (st, k0, wd, we, p, q) == (0, 0, 1, 1, 0.0, 0)


# ----------------------------------------------------------------------------------------------------
# running median
# ----------------------------------------------------------------------------------------------------

KINDS = ["lognormal", "dupes", "zeros", "full64", "ramp", "const"]


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("window", [1, 3, 5, 101, 1001])
def test_sliding_median_equals_definition_and_scipy(orc, kind, window):
    n = 2500 if window > 101 else 700
    x = W.random_spectrum(n, seed=hash((kind, window)) % 1000, kind=kind)
    slid = orc.running_median(x, window)
    assert np.array_equal(slid, orc.running_median_sort(x, window))
    # library routine: half-sample-symmetric reflection == scipy mode='reflect' == numpy pad 'symmetric'
    assert np.array_equal(slid, ndimage.median_filter(x, size=window, mode="reflect"))
    h = window // 2
    xp = np.pad(x, h, mode="symmetric")
    ks = [0, 1, h, n // 2, n - 1 - h, n - 2, n - 1]
    for k in ks:
        if 0 <= k < n:
            assert slid[k] == np.sort(xp[k:k + window])[h]


def test_median_properties(orc):
    x = W.random_spectrum(4000, 7, "lognormal")
    m = orc.running_median(x, 201)
    assert np.array_equal(orc.running_median(np.full(500, 42, dtype=np.int64), 201), np.full(500, 42))
    y = x + W.random_spectrum(4000, 8, "dupes")          # x <= y elementwise  =>  med(x) <= med(y)
    assert np.all(m <= orc.running_median(y, 201))
    z = np.full(3000, 1000, dtype=np.int64)
    z[1000:1100] = 1 << 40                                 # a spike narrower than h+1 bins is invisible
    assert np.array_equal(orc.running_median(z, 201), np.full(3000, 1000))
    z[1000:1101] = 1 << 40                                 # h+1 bins wide: seen by the windows that contain all of it
    out = orc.running_median(z, 201)
    assert np.array_equal(np.flatnonzero(out == (1 << 40)), np.arange(1000, 1101))
    big = np.array([(1 << 62) + 1, (1 << 62) + 3, (1 << 62) + 2] * 50, dtype=np.int64)   # beyond 2^53
    assert np.array_equal(orc.running_median(big, 3), ndimage.median_filter(big, size=3, mode="reflect"))


def test_median_size_limits(orc):
    x = W.random_spectrum(6, 1, "lognormal")
    assert np.array_equal(orc.running_median(x, 11), orc.running_median_sort(x, 11))      # n == h + 1
    with pytest.raises(ValueError):
        orc.running_median(x, 13)                           # n < h + 1
    with pytest.raises(ValueError):
        orc.running_median(x, 4)                            # even window
    with pytest.raises(ValueError):
        orc.running_median_sort(x, 0)


def test_psd_formation(orc):
    # psd = s_instr + C * med * 2^-140 ; C = 729/512 is exact in binary ((1 - 2/(9 nu))^-3, nu = 2)
    assert Fraction(W.MEDIAN_NORM_PAPER) == Fraction(1, (1 - Fraction(2, 18)) ** 3) == Fraction(729, 512)
    assert abs(W.MEDIAN_NORM_PAPER - 1.4237) < 2e-4         # the paper prints "~1.4237"
    med = np.array([0, 1, 219928, (1 << 53) + 1, 7], dtype=np.int64)
    s = np.array([1e-40, 0.0, 2e-38, 0.0, 3e-41])
    out = orc.psd_from_median(med, s, W.MEDIAN_NORM_PAPER, -140)
    for k in range(5):
        exact = Fraction(float(med[k])) * Fraction(729, 512) / (1 << 140)
        if k != 3:
            exact_sum = Fraction(float(s[k])) + exact
            assert abs(Fraction(float(out[k])) - exact_sum) <= Fraction(math.ulp(float(out[k]))) / 2
        else:
            assert abs(Fraction(float(out[k])) / exact - 1) < Fraction(1, 1 << 51)
    assert out[0] == 1e-40 and out[1] == 729.0 / 512.0 * 2.0 ** -140
