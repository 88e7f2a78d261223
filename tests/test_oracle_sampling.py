"""Pins for the oracle's stage (i): Philox, u01, elementary functions, population draws.

None of these tests re-types the oracle's formula and compares it with itself: Philox is held to
the published known-answer vectors, the elementary functions to mpmath at 40 digits and to glibc,
the draws to closed-form CDFs (KS), and eq. (4) to mpmath and to tabulated values.
"""
import math
import os
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest
from scipy import stats

import gbfg_workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
mp.mp.dps = 40


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def _ulps(got, exact):
    return abs((mp.mpf(got) - exact) / math.ulp(float(exact)))


def test_philox_known_answers(orc):
    for row in _rows("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        assert orc.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_u01_exact_and_open_interval(orc):
    # u = (x + 1/2) 2^-52 with x the top 52 bits of (hi:lo): exact rational check
    rng = np.random.default_rng(1)
    cases = [(0, 0), (0xFFFFFFFF, 0xFFFFFFFF), (0xFFF, 0), (0x1000, 0)]
    cases += [tuple(int(v) for v in rng.integers(0, 1 << 32, 2)) for _ in range(200)]
    for lo, hi in cases:
        x = ((hi << 32) | lo) >> 12
        u = orc.u01(lo, hi)
        assert Fraction(u) == Fraction(2 * x + 1, 1 << 53)
        assert 0.0 < u < 1.0
    assert orc.u01(0, 0) == 2.0 ** -53
    assert orc.u01(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53


def test_log_against_mpmath_and_glibc(orc):
    rng = np.random.default_rng(2)
    xs = np.concatenate([rng.random(1500), 10.0 ** rng.uniform(-300, 300, 1500),
                         1.0 + 1e-3 * rng.standard_normal(1500), [2.0 ** -53, 1 - 2.0 ** -53, 1.0, 2.0, 0.5,
                                                                    math.sqrt(0.5), math.sqrt(2.0)]])
    worst = 0
    for x in xs:
        x = float(abs(x))
        got = orc.log(x)
        if x == 1.0:
            assert got == 0.0
            continue
        worst = max(worst, _ulps(got, mp.log(mp.mpf(x))))
        assert abs(got - math.log(x)) <= 4 * math.ulp(math.log(x))
    assert worst <= 3.0


def test_exp10_against_mpmath_and_glibc(orc):
    rng = np.random.default_rng(3)
    worst = 0
    for y in np.concatenate([rng.uniform(-60, 60, 3000), rng.uniform(-300, 300, 500), [0.0, 1.0, -1.0, 22.0, -22.5]]):
        y = float(y)
        got = orc.exp10(y)
        worst = max(worst, _ulps(got, mp.mpf(10) ** mp.mpf(y)))
    assert worst <= 3.0
    assert orc.exp10(0.0) == 1.0
    assert abs(orc.exp10(3.0) - 1000.0) <= 2 * math.ulp(1000.0)


def test_sincos_against_mpmath(orc):
    rng = np.random.default_rng(4)
    worst = 0
    for u in np.concatenate([rng.random(3000), [0.0, 0.125, 0.25, 0.5, 0.75, 2.0 ** -53, 1 - 2.0 ** -53]]):
        u = float(u)
        s, c = orc.sincos2pi(u)
        es, ec = mp.sin(2 * mp.pi * mp.mpf(u)), mp.cos(2 * mp.pi * mp.mpf(u))
        for got, ex in ((s, es), (c, ec)):
            if abs(ex) < mp.mpf(2) ** -60:          # exact zeros of the function on the grid of quarter turns
                assert got == 0.0
            else:
                worst = max(worst, _ulps(got, ex))
    assert worst <= 3.0
    worst = 0
    for x in rng.uniform(-3.0, 3.0, 3000):
        s, c = orc.sincos(float(x))
        worst = max(worst, _ulps(s, mp.sin(mp.mpf(float(x)))), _ulps(c, mp.cos(mp.mpf(float(x)))))
    assert worst <= 3.0
    assert orc.sincos2pi(0.0) == (0.0, 1.0)
    assert orc.sincos2pi(0.25) == (1.0, 0.0)
    assert orc.sincos2pi(0.5)[1] == -1.0


def _grid_pop(orc, w, **kw):
    from dataclasses import replace
    pop = replace(w.pops[0], **kw)
    return orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2), pop


@pytest.mark.parametrize("slope", [1.5, 1.0, 2.0, 1.25])
def test_frequency_draw_matches_power_law_cdf(orc, slope):
    w = W.config(0)
    g, pop = _grid_pop(orc, w, slope=slope, n_src=40000)
    A, f, fd = orc.sample_catalog(g, pop, 0, 12345)
    assert np.all(f >= w.f_min) and np.all(f < w.f_max)
    if abs(slope - 1.0) < 1e-12:
        cdf = lambda x: np.log(x / w.f_min) / np.log(w.f_max / w.f_min)
    else:
        q = 1.0 - slope
        cdf = lambda x: (x ** q - w.f_min ** q) / (w.f_max ** q - w.f_min ** q)
    assert stats.kstest(f, cdf).pvalue > 1e-3


def test_normals_amplitude_and_chirp_relations(orc):
    w = W.config(0)
    g, pop = _grid_pop(orc, w, n_src=40000)
    A, f, fd = orc.sample_catalog(g, pop, 0, 777)
    lf = np.log10(f)
    z_a = (np.log10(A) - pop.logA_offset - (2.0 / 3.0) * (lf + 3.0)) / pop.logA_sigma
    K = float(mp.mpf(96) / 5 * mp.pi ** (mp.mpf(8) / 3))
    tsun = 4.925490947641267e-6
    # invert eq. (4): Mc = (fdot / (K f^(11/3)))^(3/5) / Tsun
    mc = (fd / (K * f ** (11.0 / 3.0))) ** 0.6 / tsun
    z_m = (np.log10(mc) - pop.logMc_mean) / pop.logMc_sigma
    assert stats.kstest(z_a, "norm").pvalue > 1e-3
    assert stats.kstest(z_m, "norm").pvalue > 1e-3
    assert abs(np.corrcoef(z_a, z_m)[0, 1]) < 0.02
    assert abs(np.corrcoef(z_a, lf)[0, 1]) < 0.02
    assert abs(np.corrcoef(z_m, lf)[0, 1]) < 0.02


def test_box_muller_identity_and_counter_layout(orc):
    """z_A^2 + z_M^2 = -2 ln u_1 with u_1 from words (2,3) of block 0 of counter (i, 0, b, cat);
    u_f from words (0,1) reproduces f through the closed-form inverse CDF (R1)."""
    w = W.config(0)
    seed, cat = 0xDEADBEEF12345, 3
    g, pop = _grid_pop(orc, w, n_src=64)
    A, f, fd = orc.sample_catalog(g, pop, cat, seed)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    K = mp.mpf(96) / 5 * mp.pi ** (mp.mpf(8) / 3)
    tsun = mp.mpf("4.925490947641267e-6")
    for i in range(64):
        b0 = orc.philox4x32_10([i, 0, 0, cat], key)
        b1 = orc.philox4x32_10([i, 0, 1, cat], key)
        u_f, u_1, u_2 = orc.u01(b0[0], b0[1]), orc.u01(b0[2], b0[3]), orc.u01(b1[0], b1[1])
        a, b = mp.mpf(w.f_min) ** mp.mpf(-0.5), mp.mpf(w.f_max) ** mp.mpf(-0.5)
        f_exact = (a + mp.mpf(u_f) * (b - a)) ** -2
        assert abs(mp.mpf(float(f[i])) / f_exact - 1) < mp.mpf("1e-13")
        lf = mp.log10(mp.mpf(float(f[i])))
        z_a = (mp.log10(mp.mpf(float(A[i]))) - mp.mpf(pop.logA_offset) - mp.mpf(2) / 3 * (lf + 3)) / mp.mpf(pop.logA_sigma)
        mc = (mp.mpf(float(fd[i])) / (K * mp.mpf(float(f[i])) ** (mp.mpf(11) / 3))) ** (mp.mpf(3) / 5) / tsun
        z_m = (mp.log10(mc) - mp.mpf(pop.logMc_mean)) / mp.mpf(pop.logMc_sigma)
        r2 = -2 * mp.log(mp.mpf(u_1))
        assert abs((z_a ** 2 + z_m ** 2) / r2 - 1) < mp.mpf("1e-10")
        # the angle is 2 pi u_2: z_A = r cos, z_M = r sin
        assert abs(z_a - mp.sqrt(r2) * mp.cos(2 * mp.pi * mp.mpf(u_2))) < mp.mpf("1e-10")
        assert abs(z_m - mp.sqrt(r2) * mp.sin(2 * mp.pi * mp.mpf(u_2))) < mp.mpf("1e-10")


def test_chirp_is_eq4_and_amplitude_trend(orc):
    """sigma = 0 removes the randomness: fdot = (96/5) pi^(8/3) (Tsun Mc)^(5/3) f^(11/3),
    A = 10^(offset + (2/3) log10(f / 1 mHz)) (BASELINE.json:configs[0])."""
    w = W.config(2)
    g, pop = _grid_pop(orc, w, n_src=2000, logA_sigma=0.0, logMc_sigma=0.0)
    A, f, fd = orc.sample_catalog(g, pop, 0, 5)
    K = mp.mpf(96) / 5 * mp.pi ** (mp.mpf(8) / 3)
    tm = mp.mpf("4.925490947641267e-6") * mp.mpf(10) ** mp.mpf(pop.logMc_mean)
    for i in range(0, 2000, 37):
        fi = mp.mpf(float(f[i]))
        assert abs(mp.mpf(float(fd[i])) / (K * tm ** (mp.mpf(5) / 3) * fi ** (mp.mpf(11) / 3)) - 1) < mp.mpf("2e-13")
        assert abs(mp.mpf(float(A[i])) / (mp.mpf(10) ** (mp.mpf(pop.logA_offset) + mp.mpf(2) / 3 * mp.log10(fi / mp.mpf("1e-3")))) - 1) < mp.mpf("2e-13")


def test_eq4_tabulated_values():
    """The tabulated eq. (4) values (tests/golden/fdot_gw.txt) against mpmath; the sampler is tied to
    eq. (4) by test_chirp_is_eq4_and_amplitude_trend."""
    K = mp.mpf(96) / 5 * mp.pi ** (mp.mpf(8) / 3)
    tm = mp.mpf("4.925490947641267e-6") * mp.mpf("0.3")
    for f, val in _rows("fdot_gw.txt"):
        got = K * tm ** (mp.mpf(5) / 3) * mp.mpf(f) ** (mp.mpf(11) / 3)
        assert abs(got / mp.mpf(val) - 1) < mp.mpf("1e-6")


def test_counter_based_streams(orc):
    w = W.config(0)
    g, pop = _grid_pop(orc, w, n_src=5000)
    full = orc.sample_catalog(g, pop, 0, 9)
    part = orc.sample_catalog(g, pop, 0, 9, 1234, 2345)
    for a, b in zip(full, part):
        assert np.array_equal(a[1234:2345], b)
    again = orc.sample_catalog(g, pop, 0, 9)
    other_cat = orc.sample_catalog(g, pop, 1, 9)
    other_seed = orc.sample_catalog(g, pop, 0, 10)
    assert all(np.array_equal(a, b) for a, b in zip(full, again))
    assert not np.array_equal(full[1], other_cat[1]) and not np.array_equal(full[1], other_seed[1])


def test_instrument_noise_robson_curve(orc):
    # tabulated values (5 digits)
    for f, val in _rows("robson_curve.txt"):
        assert abs(orc.robson_sn(float(f)) / float(val) - 1) < 1e-4
    # independent 40-digit evaluation of the same published curve
    L, fs = mp.mpf("2.5e9"), mp.mpf("19.09e-3")
    rng = np.random.default_rng(6)
    for f in 10.0 ** rng.uniform(-4, -1.5, 300):
        x = mp.mpf(float(f))
        poms = mp.mpf("1.5e-11") ** 2 * (1 + (mp.mpf("2e-3") / x) ** 4)
        pacc = mp.mpf("3e-15") ** 2 * (1 + (mp.mpf("0.4e-3") / x) ** 2) * (1 + (x / mp.mpf("8e-3")) ** 4)
        sn = mp.mpf(10) / (3 * L ** 2) * (poms + 2 * (1 + mp.cos(x / fs) ** 2) * pacc / (2 * mp.pi * x) ** 4) * (1 + mp.mpf("0.6") * (x / fs) ** 2)
        assert abs(mp.mpf(orc.robson_sn(float(f))) / sn - 1) < mp.mpf("3e-15")
    # array form: bin centres f_min + (k + 1/2)/T
    w = W.config(0)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs)
    s = orc.instrument_noise(g)
    for k in (0, 1, 28402, g.n_bins - 1):
        assert s[k] == orc.robson_sn(w.f_min + (k + 0.5) / w.t_obs)
