"""Pins of the oracle's coarse-graining (eqs. 13-14) and characteristic strain (eq. B1,
PAPER.md:465): closed forms, numpy's reduceat, the structure of the logarithmic bins."""
import numpy as np

import gbfg_workloads as wl


def test_log_bin_edges_are_logarithmic_and_cover_the_band():
    w = wl.config(2)
    e = wl.log_bin_edges(w, 100, 1e-4, 1e-2)               # the paper's 100 bins over 0.1-10 mHz
    assert e.size == 101 and e[0] == 0 and np.all(np.diff(e) >= 1)
    centres = w.f_min + (e[:-1] + 0.5) / w.t_obs
    ratio = centres[2:] / centres[1:-1]
    assert np.allclose(ratio, 10 ** (2 / 100), rtol=2e-3)   # each coarse bin starts a factor 10^(2/100) higher
    full = wl.log_bin_edges(w, 64)
    n_bins = int(np.ceil((w.f_max - w.f_min) * w.t_obs))
    assert full[0] == 0 and full[-1] == n_bins             # default: the whole band, every fine bin in one coarse bin


def test_coarse_grain_closed_forms(orc):
    w = wl.config(0)
    T, f_min = w.t_obs, w.f_min
    e = wl.log_bin_edges(w, 50)
    n = int(e[-1])
    S, fk, hc = orc.coarse_grain(np.full(n, 2.0 ** -131), e, f_min, T)
    assert np.all(S == 2.0 ** -131)                         # mean of a constant power of two, exactly
    S, fk, hc = orc.coarse_grain(np.full(n, 3.25e-40), e, f_min, T)
    assert np.allclose(S, 3.25e-40, rtol=3e-16, atol=0)     # any constant: two roundings
    mid = f_min + ((e[:-1] + e[1:] - 1) / 2.0 + 0.5) / T   # mean of an arithmetic progression
    assert np.allclose(fk, mid, rtol=1e-15, atol=0)
    assert np.allclose(hc, np.sqrt(fk * 3.25e-40), rtol=1e-15)
    # against numpy's segmented sum
    rng = np.random.default_rng(5)
    psd = 10.0 ** rng.uniform(-41, -36, n)
    S, fk, hc = orc.coarse_grain(psd, e, f_min, T)
    ref = np.add.reduceat(psd, e[:-1]) / np.diff(e)
    assert np.allclose(S, ref, rtol=1e-13)
    # the mean lies between the extremes of its bin; N_k adds up
    for k in (0, 10, 49):
        seg = psd[e[k]:e[k + 1]]
        assert seg.min() <= S[k] <= seg.max()
    assert np.diff(e).sum() == n
    # an empty coarse bin is NaN
    e2 = np.array([0, 5, 5, 9], dtype=np.int64)
    S2, f2, h2 = orc.coarse_grain(psd, e2, f_min, T)
    assert np.isnan(S2[1]) and np.isnan(f2[1]) and np.isnan(h2[1]) and not np.isnan(S2[2])


def test_coarse_grained_foreground_trends(orc):
    """PAPER.md:136 (Fig. 2): the foreground grows with the number of binaries; in coarse-grained form."""
    w1 = wl.scaled(wl.config(1), n_src=30_000)
    w2 = wl.scaled(wl.config(1), n_src=100_000)
    e = wl.log_bin_edges(w1, 20, 2e-4, 2e-3)
    out = []
    for w in (w1, w2):
        r = orc.simulate(w)
        S, fk, hc = orc.coarse_grain(r["psd"] - r["s_instr"], e, w.f_min, w.t_obs)
        out.append(S)
    assert np.all(out[1] >= out[0]) and np.sum(out[1] > out[0]) >= 5
