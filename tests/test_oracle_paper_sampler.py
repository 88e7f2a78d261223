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
