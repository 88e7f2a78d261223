"""The CUDA path's stage (i), noise curves and paper sampler against MATHEMATICS, not against the oracle.

DESIGN.md section 4 fixes the elementary functions as text, and oracle and kernel both type that text, so their bit
equality (test_gpu_parity.py) shows that the two transcriptions agree, not that either is right.  The oracle's side is
pinned to mpmath / KS / known-answer vectors in tests/test_oracle_*.py.  This file does the same for the GPU's OWN
outputs: nothing here calls the oracle.  Philox4x32-10 is restated below in Python integers (the published round function,
Salmon et al. SC'11) and held to the Random123 known-answer vectors before it is used.
"""
import math
import os

import numpy as np
import pytest

import gbfg_workloads as wl

pytestmark = pytest.mark.gpu

mp = pytest.importorskip("mpmath")
stats = pytest.importorskip("scipy.stats")
mp.mp.dps = 40

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M32 = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M32, p1 & M32, ((p0 >> 32) ^ c3 ^ k1) & M32, p0 & M32
        k0, k1 = (k0 + 0x9E3779B9) & M32, (k1 + 0xBB67AE85) & M32
    return [c0, c1, c2, c3]


def u01(lo, hi):
    """(x + 1/2) 2^-52 with x the top 52 bits of (hi:lo), as an exact mpmath number (R1)."""
    return (mp.mpf(((hi << 32) | lo) >> 12) + mp.mpf(1) / 2) / mp.mpf(2) ** 52


def test_python_philox_is_the_published_one():
    with open(os.path.join(GOLD, "philox4x32_10_kat.txt")) as fh:
        rows = [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        assert philox4x32_10(v[0:4], v[4:6]) == v[6:10]


@pytest.fixture(scope="module")
def torch():
    import torch as t
    return t


def _draw(gb, torch, w, pop, seed, cat):
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n = pop.n_src
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    gb.sample_catalog(g, [pop], [0, n], seed, A, f, fd, first_cat_id=cat)
    return A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()


K_EQ4 = mp.mpf(96) / 5 * mp.pi ** (mp.mpf(8) / 3)             # eq. (4)
T_SUN = mp.mpf("4.925490947641267e-6")                      # G Msun / c^3 in seconds (R1)


@pytest.mark.parametrize("slope", [1.5, 1.0, 1.73])
def test_gpu_catalog_is_the_inverse_cdf_box_muller_and_eq4_of_the_philox_words(gb, torch, slope):
    """Every GPU-drawn (f, A, fdot) is rebuilt at 40 digits from the raw Philox words of counter (i, 0, block, cat):
    f by the inverse CDF of p(f) ∝ f^-s, (z_A, z_M) by Box-Muller, A by BASELINE's amplitude relation, fdot by eq. (4).
    A wrong constant, counter layout, sign, quadrant or series coefficient in the kernel fails here."""
    w = wl.config(0)
    seed, cat = 0xDEADBEEF12345, 3
    pop = wl.replace(w.pops[0], slope=slope, n_src=96)
    A, f, fd = _draw(gb, torch, w, pop, seed, cat)
    key = [seed & M32, seed >> 32]
    fmin, fmax = mp.mpf(w.f_min), mp.mpf(w.f_max)
    worst = 0
    for i in range(pop.n_src):
        b0 = philox4x32_10([i, 0, 0, cat], key)
        b1 = philox4x32_10([i, 0, 1, cat], key)
        u_f, u_1, u_2 = u01(b0[0], b0[1]), u01(b0[2], b0[3]), u01(b1[0], b1[1])
        if slope == 1.0:
            f_ex = fmin * (fmax / fmin) ** u_f
        else:
            q = 1 - mp.mpf(slope)
            f_ex = (fmin ** q + u_f * (fmax ** q - fmin ** q)) ** (1 / q)
        r = mp.sqrt(-2 * mp.log(u_1))
        z_a, z_m = r * mp.cos(2 * mp.pi * u_2), r * mp.sin(2 * mp.pi * u_2)
        a_ex = mp.mpf(10) ** (mp.mpf(pop.logA_offset) + mp.mpf(2) / 3 * mp.log10(f_ex / mp.mpf("1e-3")) + mp.mpf(pop.logA_sigma) * z_a)
        mc = mp.mpf(10) ** (mp.mpf(pop.logMc_mean) + mp.mpf(pop.logMc_sigma) * z_m)
        fd_ex = K_EQ4 * (T_SUN * mc) ** (mp.mpf(5) / 3) * f_ex ** (mp.mpf(11) / 3)
        for got, ex in ((f[i], f_ex), (A[i], a_ex), (fd[i], fd_ex)):
            worst = max(worst, abs(mp.mpf(float(got)) / ex - 1))
    # log/exp10/sincos are each good to <= 3 ulp (6.7e-16); the chain multiplies arguments of size <= 60 by ln 10 and
    # adds a handful of roundings: 1e-13 leaves a factor ~10 of room and is far below any formula error
    assert worst < mp.mpf("1e-13"), worst


def test_gpu_chirp_is_eq4_and_amplitude_trend(gb, torch):
    """sigma = 0 removes the randomness (the mpmath counterpart of test_chirp_is_eq4_and_amplitude_trend, on GPU output)."""
    w = wl.config(2)
    pop = wl.replace(w.pops[0], n_src=2000, logA_sigma=0.0, logMc_sigma=0.0)
    A, f, fd = _draw(gb, torch, w, pop, 5, 0)
    tm = T_SUN * mp.mpf(10) ** mp.mpf(pop.logMc_mean)
    assert np.all((f >= w.f_min) & (f < w.f_max))
    for i in range(0, 2000, 37):
        fi = mp.mpf(float(f[i]))
        assert abs(mp.mpf(float(fd[i])) / (K_EQ4 * tm ** (mp.mpf(5) / 3) * fi ** (mp.mpf(11) / 3)) - 1) < mp.mpf("2e-13")
        assert abs(mp.mpf(float(A[i])) / (mp.mpf(10) ** (mp.mpf(pop.logA_offset) + mp.mpf(2) / 3 * mp.log10(fi / mp.mpf("1e-3")))) - 1) < mp.mpf("2e-13")


def test_gpu_draws_follow_their_distributions(gb, torch):
    """KS of the GPU's own draws against closed-form CDFs; normal scores recovered by inverting the relations."""
    w = wl.config(0)
    for slope in (1.5, 1.0, 2.0):
        pop = wl.replace(w.pops[0], slope=slope, n_src=40_000)
        A, f, fd = _draw(gb, torch, w, pop, 12345, 0)
        if slope == 1.0:
            cdf = lambda x: np.log(x / w.f_min) / np.log(w.f_max / w.f_min)
        else:
            q = 1.0 - slope
            cdf = lambda x: (x ** q - w.f_min ** q) / (w.f_max ** q - w.f_min ** q)
        assert stats.kstest(f, cdf).pvalue > 1e-3
    lf = np.log10(f)
    z_a = (np.log10(A) - pop.logA_offset - (2.0 / 3.0) * (lf + 3.0)) / pop.logA_sigma
    mc = (fd / (float(K_EQ4) * f ** (11.0 / 3.0))) ** 0.6 / float(T_SUN)
    z_m = (np.log10(mc) - pop.logMc_mean) / pop.logMc_sigma
    assert stats.kstest(z_a, "norm").pvalue > 1e-3 and stats.kstest(z_m, "norm").pvalue > 1e-3
    assert abs(np.corrcoef(z_a, z_m)[0, 1]) < 0.02 and abs(np.corrcoef(z_a, lf)[0, 1]) < 0.02


def _robson_mp(x):
    L, fs = mp.mpf("2.5e9"), mp.mpf("19.09e-3")
    poms = mp.mpf("1.5e-11") ** 2 * (1 + (mp.mpf("2e-3") / x) ** 4)
    pacc = mp.mpf("3e-15") ** 2 * (1 + (mp.mpf("0.4e-3") / x) ** 2) * (1 + (x / mp.mpf("8e-3")) ** 4)
    return mp.mpf(10) / (3 * L ** 2) * (poms + 2 * (1 + mp.cos(x / fs) ** 2) * pacc / (2 * mp.pi * x) ** 4) * (1 + mp.mpf("0.6") * (x / fs) ** 2)


@pytest.mark.parametrize("cfg", [0, 2])
def test_gpu_instrument_noise_is_the_robson_curve_at_bin_centres(gb, torch, cfg):
    w = wl.config(cfg)
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s = torch.empty(g.n_bins, dtype=torch.float64, device="cuda")
    gb.instrument_noise(g, s)
    s = s.cpu().numpy()
    assert np.all(s > 0) and np.all(np.isfinite(s))
    rng = np.random.default_rng(6 + cfg)
    ks = np.concatenate([[0, 1, g.n_bins - 1], rng.integers(0, g.n_bins, 300)])
    for k in ks:
        fk = mp.mpf(w.f_min) + (mp.mpf(int(k)) + mp.mpf(1) / 2) / mp.mpf(w.t_obs)
        # 3e-15 for the formula in binary64 (as the oracle's pin) + the rounding of the bin centre itself (<= 2^-53
        # relative in f, amplified by the curve's steepest logarithmic slope, ~5 below 0.4 mHz)
        assert abs(mp.mpf(float(s[k])) / _robson_mp(fk) - 1) < mp.mpf("4e-15"), k


@pytest.mark.parametrize("tdi2", [True, False])
def test_gpu_aet_noise_is_eqs_C1_C5_B2_B5(gb, torch, tdi2):
    from test_oracle_aet_noise import _mp_formulas            # the formulas as the paper prints them, at 40 digits
    w = wl.config(2)
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    outs = [torch.empty(g.n_bins, dtype=torch.float64, device="cuda") for _ in range(4)]
    gb.instrument_noise_aet(g, *outs, tdi2=tdi2)
    outs = [o.cpu().numpy() for o in outs]
    rng = np.random.default_rng(11)
    for k in np.concatenate([[0, g.n_bins - 1], rng.integers(0, g.n_bins, 120)]):
        fk = mp.mpf(w.f_min) + (mp.mpf(int(k)) + mp.mpf(1) / 2) / mp.mpf(w.t_obs)
        want = _mp_formulas(fk, tdi2=tdi2)
        # next to the zero of the TDI 2.0 factor 4 sin^2(2x) at 2x = pi (29.98 mHz, the top of the band) a rounding of x
        # is amplified by 2 / |tan 2x|: the tolerance follows the condition number there
        s2x = abs(mp.sin(2 * fk / (mp.mpf(299792458) / (2 * mp.pi * mp.mpf("2.5e9")))))
        for j, (o, w_) in enumerate(zip(outs, want)):
            tol = mp.mpf("3e-14") * (max(1, mp.mpf("0.05") / s2x) if (tdi2 and j < 2) else 1)
            assert abs(mp.mpf(float(o[k])) / w_ - 1) < tol, (k, tdi2, j)


def test_gpu_paper_sampler_marginals_follow_table_I(gb, torch):
    """KS of the GPU's draws from the paper's own population model against Table I's closed-form CDFs,
    the copula's normal-score correlation (App. A) and PAPER.md:459 (marginals independent of rho)."""
    w = wl.config(1)                                  # 0.1-10 mHz: the band of Table I
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)

    def draw(pop, seed):
        n = pop.n_src
        A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        gb.sample_catalog_paper(g, [pop], [0, n], seed, A, f, fd)
        return A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()

    for pop in (wl.PaperPopulation(n_src=40_000), wl.paper_prior_draw(3, n_src=40_000), wl.paper_prior_draw(8, n_src=40_000)):
        A, f, fd = draw(pop, 7)
        a1 = 1 + pop.alpha_pl
        cdf_f = lambda x: (x ** a1 - w.f_min ** a1) / (w.f_max ** a1 - w.f_min ** a1)
        assert stats.kstest(f, cdf_f).pvalue > 1e-3
        ft = np.log10(fd) - pop.mu_gamma                               # eq. (7)
        assert stats.kstest(ft, stats.gamma(pop.alpha_gamma, scale=1 / pop.beta_gamma).cdf).pvalue > 1e-3
        At = np.log10(f ** (-2.0 / 3.0) * A) - pop.mu                  # eq. (8)
        assert np.all(At > 0)
        assert stats.kstest(np.log(At) / pop.sigma, "norm").pvalue > 1e-3
        zs_f = stats.norm.ppf(stats.rankdata(f) / (f.size + 1))
        zs_d = stats.norm.ppf(stats.rankdata(fd) / (fd.size + 1))
        assert abs(np.corrcoef(zs_f, zs_d)[0, 1] - pop.rho) < 0.02
    base = wl.PaperPopulation(n_src=20_000)
    lo, hi = draw(wl.replace(base, rho=0.0), 3), draw(wl.replace(base, rho=0.99), 3)
    assert np.array_equal(lo[1], hi[1])                                # f does not depend on rho at all
    assert stats.ks_2samp(lo[2], hi[2]).pvalue > 1e-3                  # fdot keeps its marginal


def test_gpu_paper_sampler_is_the_copula_of_the_philox_words(gb, torch):
    """The paper's sampler rebuilt at 40 digits from the raw Philox words (counter blocks 2 and 3, R12):
    (n1, n2) by Box-Muller, z2 = rho n1 + sqrt(1 - rho^2) n2, u' = Phi(z1), v' = Phi(z2) (App. A steps iii-iv,
    PAPER.md:456-457), f by the inverse power-law CDF at u', x = beta (log10 fdot - mu_Gamma) must sit at probability v'
    of Gamma(alpha) (eq. 7; checked on z2's own tail), A = 10^(mu + exp(sigma z3) + (2/3) log10 f) (eq. 8).  The GPU's
    erfc, incomplete gamma function and Newton iteration are checked through the sampler's own output."""
    w = wl.config(1)
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    seed, cat = 0x1234567890ABC, 5
    key = [seed & M32, seed >> 32]
    for pop in (wl.replace(wl.PaperPopulation(n_src=48), rho=0.6), wl.paper_prior_draw(2, n_src=48),
                wl.replace(wl.PaperPopulation(n_src=48), alpha_gamma=1.0, beta_gamma=3.0, rho=0.0)):
        n = pop.n_src
        A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        gb.sample_catalog_paper(g, [pop], [0, n], seed, A, f, fd, first_cat_id=cat)
        A, f, fd = A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()
        a1 = 1 + mp.mpf(pop.alpha_pl)
        rho = mp.mpf(pop.rho)
        for i in range(n):
            b2 = philox4x32_10([i, 0, 2, cat], key)
            b3 = philox4x32_10([i, 0, 3, cat], key)
            u1, u2, u3, u4 = u01(b2[0], b2[1]), u01(b2[2], b2[3]), u01(b3[0], b3[1]), u01(b3[2], b3[3])
            r = mp.sqrt(-2 * mp.log(u1))
            n1, n2 = r * mp.cos(2 * mp.pi * u2), r * mp.sin(2 * mp.pi * u2)
            z3 = mp.sqrt(-2 * mp.log(u3)) * mp.cos(2 * mp.pi * u4)
            z1, z2 = n1, rho * n1 + mp.sqrt(1 - rho * rho) * n2
            up = mp.ncdf(z1)
            f_ex = (mp.mpf(w.f_min) ** a1 + up * (mp.mpf(w.f_max) ** a1 - mp.mpf(w.f_min) ** a1)) ** (1 / a1)
            assert abs(mp.mpf(float(f[i])) / f_ex - 1) < mp.mpf("1e-12"), (i, "f")
            x = mp.mpf(pop.beta_gamma) * (mp.log10(mp.mpf(float(fd[i]))) - mp.mpf(pop.mu_gamma))
            if z2 <= 0:
                back, tail = mp.gammainc(pop.alpha_gamma, 0, x, regularized=True), mp.ncdf(z2)
            else:
                back, tail = mp.gammainc(pop.alpha_gamma, x, mp.inf, regularized=True), mp.ncdf(-z2)
            assert abs(back / tail - 1) < mp.mpf("1e-10"), (i, "fdot", back, tail)
            a_ex = mp.mpf(10) ** (mp.mpf(pop.mu) + mp.exp(mp.mpf(pop.sigma) * z3) + mp.mpf(2) / 3 * mp.log10(f_ex))
            assert abs(mp.mpf(float(A[i])) / a_ex - 1) < mp.mpf("1e-12"), (i, "A")
