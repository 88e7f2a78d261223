"""Pins of the oracle's SciRDv1 A/E/T noise (eqs. C1-C5) and TDI response (eqs. B2-B5,
PAPER.md:475-487): a 40-digit re-evaluation of the formulas as the paper prints them, their low-frequency
limits, and the sky-averaged curve of Robson et al. 2019 (the paper's ref. [70]) they must reduce to."""
import numpy as np
import pytest

mp = pytest.importorskip("mpmath")


def _mp_formulas(f, P=15, A=3, L=2.5e9, tdi2=True):
    mp.mp.dps = 40
    f = mp.mpf(f); c = mp.mpf(299792458); L = mp.mpf(L)
    fstar = c / (2 * mp.pi * L)
    x = f / fstar
    p_oms = (P * mp.mpf("1e-12")) ** 2 * (1 + (mp.mpf("2e-3") / f) ** 4) * (2 * mp.pi * f / c) ** 2                    # (C1)
    p_tm = ((A * mp.mpf("1e-15")) ** 2 * (1 + (mp.mpf("0.4e-3") / f) ** 2) * (1 + (f / mp.mpf("8e-3")) ** 4)
            * (1 / (2 * mp.pi * f)) ** 4 * (2 * mp.pi * f / c) ** 2)                                                     # (C2)
    s_aa = 8 * mp.sin(x) ** 2 * (4 * (1 + mp.cos(x) + mp.cos(x) ** 2) * p_tm + (2 + mp.cos(x)) * p_oms)                # (C3)
    s_tt = 16 * mp.sin(x) ** 2 * (2 * (1 - mp.cos(x)) ** 2 * p_tm + (1 - mp.cos(x)) * p_oms)                           # (C4)
    pre = 16 * mp.sin(x) ** 2 * x ** 2                                                                                  # (B3)
    r_aa = pre * mp.mpf(9) / 20 / (1 + mp.mpf("0.7") * x ** 2)                                                          # (B4)
    r_tt = pre * mp.mpf(9) / 20 * x ** 6 / (mp.mpf("1.8e3") + mp.mpf("0.7") * x ** 8)                                   # (B5)
    fac = 4 * mp.sin(2 * x) ** 2 if tdi2 else 1                                                                         # (C5)
    return fac * s_aa, fac * s_tt, s_aa / r_aa, s_tt / r_tt


@pytest.mark.parametrize("tdi2", [True, False])
def test_aet_noise_against_40_digits(orc, tdi2):
    for f in [1e-4, 3.3e-4, 1e-3, 2.5e-3, 8e-3, 1.9e-2, 2.9e-2]:
        got = orc.aet_noise(f, tdi2=tdi2)
        want = _mp_formulas(f, tdi2=tdi2)
        for g, w_ in zip(got, want):
            assert abs(mp.mpf(g) / w_ - 1) < mp.mpf("2e-14"), (f, g, w_)


def test_aet_noise_reduces_to_the_sky_averaged_curve(orc):
    """S_AA / R_AA is the sky-averaged strain sensitivity of one channel: below ~3 mHz it is the curve of
    Robson et al. 2019 (10 / (3 L^2)) (P_oms + 2 (1 + cos^2 x) P_acc / (2 pi f)^4) (1 + 0.6 x^2) to a percent
    (different f*: c / (2 pi L) against the literal 19.09 mHz; approximate response)."""
    for f in [1e-4, 3e-4, 1e-3, 3e-3]:
        assert abs(orc.aet_noise(f)[2] / orc.robson_sn(f) - 1) < 0.02
    # the T channel is insensitive at low frequency: its strain-equivalent noise is orders of magnitude higher
    assert orc.aet_noise(1e-3)[3] > 1e4 * orc.aet_noise(1e-3)[2]


def test_aet_noise_scalings(orc):
    f = 2e-3
    a = orc.aet_noise(f, P=15, A=3)
    b = orc.aet_noise(f, P=30, A=6)
    for x, y in zip(a, b):
        assert abs(y / x - 4) < 1e-14                       # quadratic in the two amplitudes together
    c = 299792458.0
    fstar = c / (2 * np.pi * 2.5e9)
    t1, t2 = orc.aet_noise(f, tdi2=False), orc.aet_noise(f, tdi2=True)
    assert abs(t2[0] / t1[0] / (4 * np.sin(2 * f / fstar) ** 2) - 1) < 1e-13     # (C5)
    assert t1[2] == t2[2] and t1[3] == t2[3]                 # the ratio to the response does not see the TDI generation


def test_instrument_noise_aet_array(orc):
    import gbfg_workloads as wl
    w = wl.config(0)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    arrs = orc.instrument_noise_aet(g)
    for k in (0, 1, 1000, g.n_bins - 1):
        want = orc.aet_noise(w.f_min + (k + 0.5) / w.t_obs)
        assert tuple(a[k] for a in arrs) == want
    assert all(np.all(a > 0) and np.all(np.isfinite(a)) for a in arrs)


# ------------------------------------------------------------------------------------------------------------------
# The SNR summed over the TDI channels, eq. (11), in the power domain (R14)
# ------------------------------------------------------------------------------------------------------------------
def test_channel_sum_noise_is_the_harmonic_sum_of_the_channels(orc):
    """1 / S_sum = 1 / S_h^AA + 1 / S_h^EE + 1 / S_h^TT with E = A (C3), against exact rationals of the inputs."""
    from fractions import Fraction
    rng = np.random.default_rng(3)
    a = 10.0 ** rng.uniform(-41, -36, 500)
    t = 10.0 ** rng.uniform(-38, -20, 500)
    s = orc.channel_sum_noise(a, t)
    for ai, ti, si in zip(a, t, s):
        exact = 1 / (2 / Fraction(ai) + 1 / Fraction(ti))
        assert abs(Fraction(si) / exact - 1) < Fraction(4, 2 ** 52)          # four roundings
    assert np.all(s < a / 2 * (1 + 1e-15))                                   # three channels never do worse than two


def test_channel_summed_snr_of_an_isolated_source_is_eq_11(orc):
    """An isolated one-bin source: rho^2 against S_sum equals the sum over A, E, T of 4 p R_XX / S^XX with the noises and
    responses of eqs. (C3)-(C4), (B4)-(B5) evaluated at 40 digits as the paper prints them; and the T channel adds next to
    nothing below a few mHz."""
    import gbfg_workloads as wl
    w = wl.config(0)
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    _, _, sh_aa, sh_tt = orc.instrument_noise_aet(g)
    s_sum = orc.channel_sum_noise(sh_aa, sh_tt)
    for f0, A0 in [(3.3e-4, 2e-21), (1.2e-3, 4e-22), (4.7e-3, 1e-22), (9.1e-3, 3e-22)]:
        st, k0, wdt, we, p, q = orc.source_bins(g, A0, f0, 0.0)
        assert st == 0 and we == 1
        got = orc.rho2(g, A0, f0, 0.0, s_sum)
        fk = mp.mpf(w.f_min) + (mp.mpf(k0) + mp.mpf(1) / 2) / mp.mpf(w.t_obs)
        s_aa, s_tt, shaa, shtt = _mp_formulas(fk)                            # S^XX and S^XX / R_XX at 40 digits
        want = 4 * mp.mpf(p) * (2 / shaa + 1 / shtt)                          # = sum_X 4 p R_XX / S^XX, A = E
        assert abs(mp.mpf(got) / want - 1) < mp.mpf("5e-14"), (f0, got, want)
        two = orc.rho2(g, A0, f0, 0.0, sh_aa / 2)                             # A and E alone
        assert 0 <= got / two - 1 < (1e-3 if f0 < 5e-3 else 0.2)
