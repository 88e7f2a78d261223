"""Pins for the oracle's stages (iv) SNR + selection and (v) the subtraction loop."""
import math
from dataclasses import replace
from fractions import Fraction

import numpy as np
import pytest

import gbfg_workloads as W


def _setup(orc, i=0, n=4000, seed=None):
    w = W.config(i)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pop = replace(w.pops[0], n_src=n)
    A, f, fd = orc.sample_catalog(g, pop, 0, w.seed if seed is None else seed)
    return w, g, A, f, fd, orc.instrument_noise(g)


def test_snr_closed_form_isolated_source(orc):
    """An isolated source (median 0 around it) has rho^2 = (4P/w) sum_k 1/S_instr[k]: exact rationals."""
    w, g, A, f, fd, s = _setup(orc, 0, 10)
    for a, ff, d in [(1e-22, 1e-3, 1e-17), (3e-22, 8e-3, 2.5e-14), (5e-23, 9.99e-3, 4e-13), (2e-21, 1.0001e-4, 0.0)]:
        st, k0, wid, we, p, q = orc.source_bins(g, a, ff, d)
        assert st == 0
        exact = sum(Fraction(4.0 * p) / Fraction(float(s[k])) for k in range(k0, k0 + we))
        got = orc.rho2(g, a, ff, d, s)
        assert abs(Fraction(got) / exact - 1) <= Fraction(we + 1, 1 << 52)
        assert abs(orc.rho2(g, a, ff, d, s, long_double=True) / got - 1) <= (we + 1) * 2.0 ** -52
        if we == 1:
            assert got == (4.0 * p) / s[k0]                  # w = 1: a single correctly rounded division


def test_snr_scalings(orc):
    w, g, A, f, fd, s = _setup(orc, 0, 300)
    wideA, widef, widefd = W.handmade_catalog("wide", w, 50)
    A, f, fd = np.concatenate([A, wideA]), np.concatenate([f, widef]), np.concatenate([fd, widefd])
    for i in range(0, A.size, 7):
        r = orc.rho2(g, A[i], f[i], fd[i], s)
        assert orc.rho2(g, 2.0 * A[i], f[i], fd[i], s) == 4.0 * r      # rho^2 ∝ A^2, exactly for a factor 2
        assert orc.rho2(g, A[i], f[i], fd[i], 4.0 * s) == 0.25 * r      # rho^2 ∝ 1/PSD
        assert orc.rho2(g, A[i], f[i], fd[i], 1.5 * s) < r              # monotone in the PSD
    assert math.isnan(orc.rho2(g, -1.0, 1e-3, 0.0, s))


def test_selection_is_strict_and_counts_near_threshold(orc):
    w, g, *_ = _setup(orc, 0, 10)
    A, f, fd = np.array([1e-22, 2e-22, 1e-22]), np.array([1e-3, 2e-3, 3e-3]), np.zeros(3)
    psd = np.ones(g.n_bins)
    trip = [orc.source_bins(g, A[i], f[i], fd[i]) for i in range(3)]
    for i in range(3):
        psd[trip[i][1]] = (4.0 * trip[i][4]) / 64.0             # rho^2 = 64 exactly (power-of-two scaling)
    res = np.zeros(3, dtype=np.uint8)
    sel, r2, near = orc.snr_select(g, A, f, fd, psd, 8.0, res)
    assert list(r2) == [64.0, 64.0, 64.0] and sel.size == 0 and not res.any() and near == 3   # rho == rho_th: not resolved
    sel, r2, near = orc.snr_select(g, A, f, fd, psd, math.nextafter(8.0, 0.0), res)
    assert list(sel) == [0, 1, 2] and res.all()
    res[:] = [0, 1, 0]                                           # already-resolved sources are not tested again
    sel, r2, near = orc.snr_select(g, A, f, fd, psd, 7.0, res)
    assert list(sel) == [0, 2] and math.isnan(r2[1]) and near == 0
    res[:] = 0
    sel, r2, near = orc.snr_select(g, A, f, fd, psd, 8.0 * (1 + 0.9e-9), res)
    assert sel.size == 0 and near == 3                           # within 1e-9 relative in rho
    sel, r2, near = orc.snr_select(g, A, f, fd, psd, 8.0 * (1 + 1.2e-9), res)
    assert near == 0


def test_selection_skips_rejected_sources(orc):
    w, g, *_ = _setup(orc, 0, 10)
    A, f, fd = W.handmade_catalog("bad", w, 200)
    s = orc.instrument_noise(g)
    res = np.zeros(200, dtype=np.uint8)
    sel, r2, near = orc.snr_select(g, A * 100, f, fd, s * 1e-6, 7.0, res)
    good = (A >= 0) & (fd >= 0) & (f >= w.f_min) & (f < w.f_max)
    good[[3, 4]] = False
    assert np.all(np.isnan(r2[~good])) and not res[~good].any() and res[good].any()


def _stepwise(orc, g, A, f, fd, s, w, rho_th, max_iter):
    """The loop composed from the stage functions in Python (R6), recording each median."""
    spec = np.zeros(g.n_bins, dtype=np.int64)
    orc.deposit(g, A, f, fd, spec)
    total = spec.copy()
    res = np.zeros(A.size, dtype=np.uint8)
    meds, news, conv, it = [], [], 0, 0
    for it in range(max_iter):
        med = orc.running_median(spec, w.window)
        psd = orc.psd_from_median(med, s, w.median_norm, w.scale_log2)
        meds.append(med)
        sel, _, _ = orc.snr_select(g, A, f, fd, psd, rho_th, res)
        news.append(sel.size)
        if sel.size == 0:
            conv = 1
            break
        orc.deposit(g, A, f, fd, spec, sel=sel, sign=-1)
    if not conv:
        med = orc.running_median(spec, w.window)
        psd = orc.psd_from_median(med, s, w.median_norm, w.scale_log2)
        meds.append(med)
    return dict(total=total, residual=spec, resolved=res, meds=meds, news=news, converged=conv,
                n_iter=(it + 1) if max_iter else 0, psd=psd, median=med)


@pytest.fixture(scope="module")
def multi_iter_case(orc):
    """2e5 sources on a narrow 1-yr band: several subtraction iterations."""
    w = W.dense_case("short")
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = orc.sample_catalog(g, orc.make_pop(w.pops[0]), 0, w.seed)
    s = orc.instrument_noise(g)
    return w, g, A, f, fd, s


def test_loop_matches_stage_composition_and_invariants(orc, multi_iter_case):
    w, g, A, f, fd, s = multi_iter_case
    ref = _stepwise(orc, g, A, f, fd, s, w, w.rho_th, w.max_iter)
    assert ref["converged"] == 1 and ref["n_iter"] >= 4          # really iterates
    spec = ref["total"].copy()
    out = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, w.rho_th, w.max_iter, spec)
    assert out["n_iter"] == ref["n_iter"] and out["converged"] == 1
    assert list(out["n_new_per_iter"][:ref["n_iter"]]) == ref["news"]
    assert np.array_equal(spec, ref["residual"]) and np.array_equal(out["resolved"], ref["resolved"])
    assert np.array_equal(out["median"], ref["median"]) and np.array_equal(out["psd"], ref["psd"])
    assert out["n_resolved"] == int(ref["resolved"].sum()) == sum(ref["news"])
    # power conservation, exactly in fixed point: residual + subtracted = total
    sub = np.zeros_like(spec)
    orc.deposit(g, A, f, fd, sub, sel=np.flatnonzero(out["resolved"]))
    assert np.array_equal(spec + sub, ref["total"])
    assert spec.min() >= 0
    # the foreground never grows from one iteration to the next
    for a, b in zip(ref["meds"][:-1], ref["meds"][1:]):
        assert np.all(b <= a)
    assert np.all(out["psd"] >= s)
    # idempotence: run again on the residual with the same flags -> nothing new, one iteration
    again = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, w.rho_th, w.max_iter,
                                         spec, resolved=out["resolved"].copy())
    assert again["n_iter"] == 1 and again["converged"] == 1 and again["n_resolved"] == 0
    assert np.array_equal(again["psd"], out["psd"])


def test_loop_cap_branch(orc, multi_iter_case):
    w, g, A, f, fd, s = multi_iter_case
    for cap in (1, 2):
        ref = _stepwise(orc, g, A, f, fd, s, w, w.rho_th, cap)
        spec = ref["total"].copy()
        out = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, w.rho_th, cap, spec)
        assert out["converged"] == 0 and out["n_iter"] == cap
        assert np.array_equal(spec, ref["residual"])
        # the returned median / PSD belong to the returned residual, not to the previous iterate
        assert np.array_equal(out["median"], orc.running_median(spec, w.window))
        assert np.array_equal(out["psd"], orc.psd_from_median(out["median"], s, w.median_norm, w.scale_log2))


def test_loop_threshold_limits(orc):
    w, g, A, f, fd, s = _setup(orc, 0, 3000, seed=21)
    spec = np.zeros(g.n_bins, dtype=np.int64)
    orc.deposit(g, A, f, fd, spec)
    total = spec.copy()
    out = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, math.inf, w.max_iter, spec)
    assert out["n_iter"] == 1 and out["converged"] == 1 and out["n_resolved"] == 0
    assert np.array_equal(spec, total)
    assert np.array_equal(out["psd"], orc.psd_from_median(orc.running_median(total, w.window), s, w.median_norm, w.scale_log2))
    # rho_th -> 0+: every source with p > 0 goes at iteration 0, residual exactly 0, PSD = S_instr exactly
    out = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, 1e-300, w.max_iter, spec)
    assert out["n_iter"] == 2 and out["n_resolved"] == 3000 and not spec.any()
    assert np.array_equal(out["psd"], s)


def test_foreground_grows_with_number_and_flatter_slope(orc):
    """PAPER.md:136 (Fig. 2): the foreground increases with N_b and with a flatter power law."""
    w = W.dense_case("short")
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s = orc.instrument_noise(g)

    def level(n, slope):
        A, f, fd = orc.sample_catalog(g, orc.make_pop(replace(w.pops[0], n_src=n, slope=slope)), 0, 3)
        spec = np.zeros(g.n_bins, dtype=np.int64)
        orc.deposit(g, A, f, fd, spec)
        out = orc.subtract_until_converged(g, A, f, fd, s, w.window, w.median_norm, w.rho_th, w.max_iter, spec)
        band = slice(int((5e-4 - w.f_min) * w.t_obs), int((1e-3 - w.f_min) * w.t_obs))
        return float(np.mean(out["psd"][band] - s[band]))
    assert level(200000, 1.5) > level(100000, 1.5) > 0
    assert level(200000, 1.2) > level(200000, 1.8)
