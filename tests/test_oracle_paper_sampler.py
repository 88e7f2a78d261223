"""Pins of the oracle's version of the paper's population sampler (Table I, eqs. 7-9, Gaussian
copula of Appendix A; R12): the special functions against mpmath / scipy, the marginals
against their closed-form CDFs, the copula's defining properties."""
import numpy as np
import pytest

import gbfg_workloads as wl

mp = pytest.importorskip("mpmath")
stats = pytest.importorskip("scipy.stats")


def test_erfc_and_normal_tail_against_40_digits(orc):
    mp.mp.dps = 40
    for t in np.concatenate([np.linspace(0, 2, 41), np.linspace(2, 6.2, 43)]):
        got = orc.erfc_pos(float(t))
        assert abs(mp.mpf(got) / mp.erfc(mp.mpf(float(t))) - 1) < mp.mpf("3e-13")
    for z in np.linspace(-8.5, 8.5, 69):
        ref = mp.ncdf(-abs(mp.mpf(float(z))))
        assert abs(mp.mpf(orc.norm_tail(float(z))) / ref - 1) < mp.mpf("3e-13")
    assert orc.norm_tail(0.0) == 0.5


def test_incomplete_gamma_against_40_digits(orc):
    mp.mp.dps = 40
    for a in [1.0, 1.3, 1.96, 2.5, 3.0]:
        for x in np.concatenate([np.geomspace(1e-9, a + 3, 40), np.linspace(a + 3, 70, 40)]):
            P, Q = orc.gamma_pq(a, float(x))
            Pm = mp.gammainc(a, 0, float(x), regularized=True)
            Qm = mp.gammainc(a, float(x), mp.inf, regularized=True)
            if x < a + 3:
                assert abs(mp.mpf(P) / Pm - 1) < mp.mpf("1e-13")
            else:
                assert abs(mp.mpf(Q) / Qm - 1) < mp.mpf("1e-13")
            assert abs(P + Q - 1) < 1e-15
    # a = 1 is the exponential distribution: P = 1 - e^-x
    for x in [0.1, 1.0, 2.5]:
        assert abs(orc.gamma_pq(1.0, x)[0] - (1 - np.exp(-x))) < 1e-15


def test_gamma_quantile_inverts_the_cdf_in_both_tails(orc):
    mp.mp.dps = 40
    for a in [1.0, 1.3, 1.96, 2.5, 3.0]:
        for z in np.linspace(-8.5, 8.5, 35):
            x = orc.gamma_quantile(a, float(z))
            tail = mp.ncdf(-abs(mp.mpf(float(z))))
            back = mp.gammainc(a, 0, x, regularized=True) if z <= 0 else mp.gammainc(a, x, mp.inf, regularized=True)
            assert abs(back / tail - 1) < mp.mpf("1e-12"), (a, z, x)
    # scipy's quantile function (a library routine) in the bulk
    for a in [1.2, 2.0, 2.9]:
        for z in [-3.0, -1.0, 0.0, 0.7, 2.5]:
            assert abs(orc.gamma_quantile(a, z) / stats.gamma.ppf(stats.norm.cdf(z), a) - 1) < 1e-10


def _draw(orc, pop, seed=7):
    w = wl.config(1)                                  # band 0.1-10 mHz: the paper's (Table I)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    return w, orc.sample_catalog_paper(g, pop, 0, seed)


def test_marginals_follow_table_I(orc):
    pop = wl.PaperPopulation(n_src=40_000)
    w, (A, f, fd) = _draw(orc, pop)
    # power law p(f) ∝ f^alpha on [f_min, f_max]
    a1 = 1 + pop.alpha_pl
    cdf_f = lambda x: (x ** a1 - w.f_min ** a1) / (w.f_max ** a1 - w.f_min ** a1)
    assert stats.kstest(f, cdf_f).pvalue > 1e-3
    # eq. (7): log10 fdot - mu_Gamma ~ Gamma(alpha, rate beta)
    ft = np.log10(fd) - pop.mu_gamma
    assert stats.kstest(ft, stats.gamma(pop.alpha_gamma, scale=1 / pop.beta_gamma).cdf).pvalue > 1e-3
    # eq. (8): A~ = log10[(f/Hz)^(-2/3) A] - mu is log-normal: ln A~ ~ N(0, sigma)
    At = np.log10(f ** (-2.0 / 3.0) * A) - pop.mu
    assert np.all(At > 0)
    assert stats.kstest(np.log(At) / pop.sigma, "norm").pvalue > 1e-3


def test_copula_properties(orc):
    """the marginals do not depend on rho; rho = 0 leaves f and fdot independent, rho -> 1 makes
    fdot an increasing function of f (rank correlation -> 1); the normal scores have correlation rho."""
    base = wl.PaperPopulation(n_src=20_000)
    out = {}
    for rho in [0.0, 0.6, 0.99]:
        pop = wl.replace(base, rho=rho)
        w, (A, f, fd) = _draw(orc, pop, seed=3)
        out[rho] = (A, f, fd)
        zs_f = stats.norm.ppf(stats.rankdata(f) / (f.size + 1))
        zs_d = stats.norm.ppf(stats.rankdata(fd) / (fd.size + 1))
        assert abs(np.corrcoef(zs_f, zs_d)[0, 1] - rho) < 0.02
    # same seed, same first normal: f does not depend on rho at all; fdot keeps its marginal
    assert np.array_equal(out[0.0][1], out[0.99][1])
    assert stats.ks_2samp(out[0.0][2], out[0.99][2]).pvalue > 1e-3
    assert np.array_equal(out[0.0][0], out[0.6][0])           # amplitudes use their own normal
    assert stats.spearmanr(out[0.99][1], out[0.99][2])[0] > 0.98
    assert abs(stats.spearmanr(out[0.0][1], out[0.0][2])[0]) < 0.03


def test_counter_layout_and_pieces(orc):
    pop = wl.PaperPopulation(n_src=5_000)
    w = wl.config(1)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = orc.sample_catalog_paper(g, pop, 2, 11)
    A2, f2, fd2 = orc.sample_catalog_paper(g, pop, 2, 11, 1000, 3000)      # a piece of the same catalog
    assert np.array_equal(A[1000:3000], A2) and np.array_equal(f[1000:3000], f2) and np.array_equal(fd[1000:3000], fd2)
    B = orc.sample_catalog_paper(g, pop, 3, 11)[1]
    assert not np.array_equal(f, B)                                        # another catalog id, another stream
    assert np.all((f >= w.f_min) & (f < w.f_max)) and np.all(fd > 0) and np.all(A > 0)


# ---------------------------------------------------------------------------------------------------------------
# DESIGN.md R12: the lengths of the fixed recurrences (erfc: 80 terms / depth 40; P, Q: 48 terms / depth 40; quantile:
# 10 Newton steps) and the domain they are stated for (0.25 <= alpha_Gamma <= 16, |z| <= 8.6: every z a binary64
# uniform in [2^-53, 1 - 2^-53] can give through Box-Muller).  The pins below sit on the corners of that domain, on both
# sides of the series / continued-fraction switches, and the SAME oracle source built one notch shorter fails them.
# ---------------------------------------------------------------------------------------------------------------
A_DOMAIN = [0.25, 1.0, 3.0, 8.0, 16.0]
Z_DOMAIN = [-8.6, -8.0, -5.0, -2.0, -0.3, 0.0, 0.3, 2.0, 5.0, 8.0, 8.6]


def _pins_of_the_recurrences(L):
    """Worst relative errors against mpmath of erfc, (P, Q) and the quantile, through the C functions of library L."""
    import ctypes as C
    import math
    mp.mp.dps = 40
    L.orc_erfc_pos.restype = C.c_double
    L.orc_erfc_pos.argtypes = [C.c_double]
    L.orc_gamma_pq.argtypes = [C.c_double] * 3 + [C.POINTER(C.c_double)] * 3
    L.orc_gamma_quantile.restype = C.c_double
    L.orc_gamma_quantile.argtypes = [C.c_double] * 4
    w_erfc = 0
    for t in [0.0, 0.5, 1.0, 1.5, np.nextafter(2.0, 0.0), 2.0, 2.05, 2.5, 4.0, 8.6 / np.sqrt(2.0)]:
        w_erfc = max(w_erfc, abs(mp.mpf(L.orc_erfc_pos(float(t))) / mp.erfc(mp.mpf(float(t))) - 1))
    w_pq = 0
    for a in A_DOMAIN:
        sw = a + 3.0
        for x in [1e-9, 0.1 * a, a, np.nextafter(sw, 0.0), sw, sw + 0.5, 2 * sw, sw + 40.0, sw + 80.0]:
            P, Q, pref = C.c_double(), C.c_double(), C.c_double()
            L.orc_gamma_pq(a, float(x), math.lgamma(a), C.byref(P), C.byref(Q), C.byref(pref))
            if x < sw:
                w_pq = max(w_pq, abs(mp.mpf(P.value) / mp.gammainc(a, 0, float(x), regularized=True) - 1))
            else:
                w_pq = max(w_pq, abs(mp.mpf(Q.value) / mp.gammainc(a, float(x), mp.inf, regularized=True) - 1))
    w_q = 0
    for a in A_DOMAIN:
        # the Wilson-Hilferty start hands over to the far-tail start where w = (1 - c) + z sqrt(c) reaches 0, c = 1 / (9 a):
        # both starts are at their worst next to that point, which is where the number of Newton steps is decided
        c = 1.0 / (9.0 * a)
        z_sw = -(1.0 - c) / np.sqrt(c)
        for z in Z_DOMAIN + [float(z_sw + d) for d in (-0.2, -0.05, 0.0, 0.05, 0.2, 0.5) if abs(z_sw + d) <= 8.6]:
            x = L.orc_gamma_quantile(a, math.lgamma(a), math.lgamma(a + 1.0), z)
            tail = mp.ncdf(-abs(mp.mpf(z)))
            back = mp.gammainc(a, 0, x, regularized=True) if z <= 0 else mp.gammainc(a, x, mp.inf, regularized=True)
            w_q = max(w_q, abs(back / tail - 1))
    return float(w_erfc), float(w_pq), float(w_q)


def _build_variant(tmp_path, name, **macros):
    import ctypes as C
    import os
    import subprocess
    import oracle
    so = os.path.join(tmp_path, f"liboracle_{name}.so")
    defs = [f"-D{k}={v}" for k, v in macros.items()]
    subprocess.check_call(["gcc", *oracle.GCC_FLAGS, *defs, "-o", so, oracle._SRC, "-lm"])
    return C.CDLL(so)


def test_recurrence_lengths_cover_the_stated_domain_and_a_notch_shorter_fails(orc, tmp_path):
    TOL_ERFC, TOL_PQ, TOL_Q = 3e-13, 3e-13, 1e-12
    e, pq, q = _pins_of_the_recurrences(_build_variant(tmp_path, "default"))
    assert e < TOL_ERFC and pq < TOL_PQ and q < TOL_Q, (e, pq, q)
    # one notch shorter, one recurrence at a time: the pin of that recurrence fails, so a cut that is too deep is seen
    e, _, _ = _pins_of_the_recurrences(_build_variant(tmp_path, "erfc_cf32", ORC_ERFC_CF_DEPTH=32))
    assert e > TOL_ERFC, e
    e, _, _ = _pins_of_the_recurrences(_build_variant(tmp_path, "erfc_s20", ORC_ERFC_SERIES_TERMS=20))
    assert e > TOL_ERFC, e
    _, pq, _ = _pins_of_the_recurrences(_build_variant(tmp_path, "gamma_cf16", ORC_GAMMA_CF_DEPTH=16))
    assert pq > TOL_PQ, pq
    _, pq, _ = _pins_of_the_recurrences(_build_variant(tmp_path, "gamma_s24", ORC_GAMMA_SERIES_TERMS=24))
    assert pq > TOL_PQ, pq
    _, _, q = _pins_of_the_recurrences(_build_variant(tmp_path, "newton8", ORC_QUANTILE_NEWTON_STEPS=8))
    assert q > TOL_Q, q
    # and the lengths the oracle had before commit 60b0425 (100 terms, depth 120, 14 steps) change nothing the pins see:
    # the shorter recurrences lose no accuracy on the domain
    e2, pq2, q2 = _pins_of_the_recurrences(_build_variant(tmp_path, "long", ORC_GAMMA_SERIES_TERMS=100, ORC_GAMMA_CF_DEPTH=120,
                                                          ORC_QUANTILE_NEWTON_STEPS=14, ORC_ERFC_CF_DEPTH=120))
    assert pq2 < TOL_PQ and q2 < TOL_Q and e2 < TOL_ERFC
