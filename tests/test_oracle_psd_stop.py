"""Pins of the oracle's second stop rule, "convergence in S_n is reached" (R13):
its limits, its consistency with a replay of the stages, and monotonicity in the tolerance."""
import numpy as np

import gbfg_workloads as wl


def _replay_deltas(orc, w, n_iter):
    """Relative PSD change between consecutive iterations, recomputed stage by stage (no loop code)."""
    g = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = orc.sample_catalog(g, w.pops[0], 0, w.seed)
    s_instr = orc.instrument_noise(g)
    spec = np.zeros(g.n_bins, dtype=np.int64)
    orc.deposit(g, A, f, fd, spec)
    resolved = np.zeros(A.size, dtype=np.uint8)
    deltas, prev = [], None
    for it in range(n_iter):
        psd = orc.psd_from_median(orc.running_median(spec, w.window), s_instr, w.median_norm, w.scale_log2)
        if prev is not None:
            deltas.append(float(np.max(np.abs(psd - prev) / prev)))
        prev = psd
        sel, _, _ = orc.snr_select(g, A, f, fd, psd, w.rho_th, resolved)
        if sel.size == 0:
            break
        orc.deposit(g, A, f, fd, spec, sel=sel, sign=-1)
    return deltas


def test_psd_stop_rule(orc):
    w = wl.dense_case("short")
    base = orc.simulate(w)                                   # rule off
    assert base["converged"] == 1 and base["n_iter"] >= 4
    deltas = _replay_deltas(orc, w, base["n_iter"])
    assert len(deltas) == base["n_iter"] - 1 and min(deltas) >= 0.0
    # a tolerance above every change stops at the second iteration, before its SNR test
    big = orc.simulate(w, psd_rtol=1e300)
    assert (big["n_iter"], big["converged"]) == (2, 2)
    assert big["n_resolved"] == base["n_new_per_iter"][0]
    # a tolerance between two consecutive changes stops exactly where the replay says
    for j in range(len(deltas) - 1):
        if deltas[j] > deltas[j + 1] > 0:
            tol = 0.5 * (deltas[j] + deltas[j + 1])
            first = next(i for i, d in enumerate(deltas) if d <= tol)
            r = orc.simulate(w, psd_rtol=tol)
            assert (r["n_iter"], r["converged"]) == (first + 2, 2)
            assert r["n_resolved"] == int(np.sum(base["n_new_per_iter"][: first + 1]))
            # the PSD returned is that of the returned residual
            assert np.array_equal(r["psd"].view(np.int64),
                                  orc.psd_from_median(orc.running_median(r["residual"], w.window), r["s_instr"],
                                                      w.median_norm, w.scale_log2).view(np.int64))
            break
    else:
        raise AssertionError("no decreasing pair of PSD changes in this case")
    # a tolerance below every non-zero change never fires before the source rule does
    tiny = orc.simulate(w, psd_rtol=1e-300)
    assert tiny["n_resolved"] == base["n_resolved"] and np.array_equal(tiny["residual"], base["residual"])
    # looser tolerance, earlier stop, fewer sources subtracted
    n_res = [orc.simulate(w, psd_rtol=t)["n_resolved"] for t in (1e-6, 1e-2, 1.0)]
    assert n_res[0] >= n_res[1] >= n_res[2]
