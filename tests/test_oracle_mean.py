"""Pins of the oracle's running-mean estimator (eq. D1; R8) against things
other than itself: numpy on a symmetric-padded array, exact rationals, closed forms, and the paper's
qualitative statements about mean vs median."""
from fractions import Fraction

import numpy as np
import pytest

import gbfg_workloads as wl


def _numpy_window_sum(x, window):
    """Library pin: numpy's 'symmetric' padding is the half-sample reflection; cumulative sums in
    Python integers (object dtype) are exact for any int64 input."""
    h = window // 2
    xp = np.pad(np.asarray(x, dtype=object), h, mode="symmetric")
    c = np.concatenate([[0], np.cumsum(xp)])
    return np.array([c[k + window] - c[k] for k in range(len(x))], dtype=object)


@pytest.mark.parametrize("kind", ["lognormal", "dupes", "zeros", "ramp", "const"])
@pytest.mark.parametrize("n,window", [(4000, 1001), (3001, 2001), (700, 3), (1200, 1), (501, 1001)])
def test_running_sum_matches_numpy_and_the_definition(orc, kind, n, window):
    x = wl.random_spectrum(n, seed=n + window, kind=kind)
    got = orc.running_sum(x, window)
    assert np.array_equal(got.astype(object), _numpy_window_sum(x, window))
    ks = sorted(set([0, 1, window // 2, n // 2, n - 2, n - 1]))
    for k in ks:
        assert orc.running_sum_def(x, window, k, k + 1)[0] == got[k]


def test_running_sum_closed_forms(orc):
    c = np.full(5000, 12345678901, dtype=np.int64)
    assert np.all(orc.running_sum(c, 2001) == 2001 * 12345678901)           # constant -> W c
    # a spike of height a is seen by exactly W outputs, once each (twice next to an end, by reflection)
    x = np.zeros(6000, dtype=np.int64)
    x[3000] = 7
    s = orc.running_sum(x, 1001)
    assert s.sum() == 1001 * 7 and s[2500] == 7 and s[3500] == 7 and s[2499] == 0 and s[3501] == 0
    y = np.zeros(6000, dtype=np.int64)
    y[10] = 5
    sy = orc.running_sum(y, 1001)
    assert sy[0] == 10 and sy[489] == 10 and sy[490] == 5 and sy[510] == 5 and sy[511] == 0   # the reflected image of bin 10 is bin -11: in the window of k <= 489
    # linearity, exactly
    a = wl.random_spectrum(3000, seed=5, kind="lognormal")
    b = wl.random_spectrum(3000, seed=6, kind="dupes")
    assert np.array_equal(orc.running_sum(a + b, 501), orc.running_sum(a, 501) + orc.running_sum(b, 501))
    # values above 2^53 stay exact
    big = np.full(100, (1 << 55) + 1, dtype=np.int64)
    assert np.all(orc.running_sum(big, 11) == 11 * ((1 << 55) + 1))
    with pytest.raises(ValueError):
        orc.running_sum(a, 1000)
    with pytest.raises(ValueError):
        orc.running_sum(a[:100], 1001)


def test_psd_from_sum_is_the_correctly_rounded_composition(orc):
    rng = np.random.default_rng(3)
    wsum = rng.integers(0, 1 << 50, 200, dtype=np.int64)
    s_instr = 10.0 ** rng.uniform(-41, -33, 200)
    got = orc.psd_from_sum(wsum, s_instr, 2001, -140)
    for k in range(200):
        e = Fraction(int(wsum[k])) / Fraction(2) ** 140           # exact (sum < 2^53)
        m = float(e / 2001)                                      # one correctly rounded division
        want = float(Fraction(s_instr[k]) + Fraction(m))         # one correctly rounded addition
        assert got[k] == want


def _run(orc, w, estimator):
    return orc.simulate(w, estimator=estimator)


def test_loop_with_the_mean_estimator(orc):
    w = wl.dense_case("short")
    ref = _run(orc, w, 1)
    g = ref["grid"]
    # the loop is the composition of the stages
    assert np.array_equal(ref["median"], orc.running_sum(ref["residual"], w.window))
    assert np.array_equal(ref["psd"].view(np.int64),
                          orc.psd_from_sum(ref["median"], ref["s_instr"], w.window, w.scale_log2).view(np.int64))
    # power conservation, residual >= 0
    spec = np.zeros(g.n_bins, dtype=np.int64)
    sel = np.nonzero(ref["resolved"])[0].astype(np.int64)
    orc.deposit(g, ref["A"], ref["f"], ref["fdot"], spec, sel=sel)
    assert np.array_equal(ref["total"] - ref["residual"], spec)
    assert ref["residual"].min() >= 0
    assert ref["n_iter"] >= 3 and ref["n_resolved"] == sel.size


def test_mean_against_median_as_the_paper_describes(orc):
    """PAPER.md:577 / Table III: the median estimator resolves more sources than the mean and leaves a
    lower foreground estimate (the mean is pulled up by the loud lines it has not yet subtracted)."""
    w = wl.dense_case("short")
    mean, med = _run(orc, w, 1), _run(orc, w, 0)
    assert med["n_resolved"] >= mean["n_resolved"]
    fg_mean = mean["psd"] - mean["s_instr"]
    fg_med = med["psd"] - med["s_instr"]
    assert np.median(fg_med) <= np.median(fg_mean)
