"""oracle/pool.py runs the unchanged single-threaded oracle in several processes: same results as in-process calls,
and its element-by-element comparison against stored arrays reports what differs and where."""
import os

import numpy as np

import gbfg_workloads as wl


def _small_batch():
    w = wl.scaled(wl.config(4), n_cat=3)
    w = wl.replace(w, t_obs=wl.YEAR_S, f_max=3e-3, window=501,
                   pops=[wl.replace(p, n_src=n) for p, n in zip(w.pops, (20_000, 0, 7_001))])
    return w


def test_pool_equals_in_process_calls_and_reports_differences(orc, tmp_path):
    from oracle import pool
    w = _small_batch()
    refs = {c: orc.simulate(w, cat=c) for c in range(w.n_cat)}
    for c, ref in refs.items():
        for name in pool.ROW_NAMES:
            a = ref[name].copy()
            if c == 2 and name == "median":
                a[5] += 1                                     # one planted difference
            np.save(os.path.join(tmp_path, f"{name}_{c}.npy"), a)
    out = pool.simulate_many(w, range(w.n_cat), n_proc=2, compare_dir=str(tmp_path))
    assert out["n_proc"] == 2 and sorted(out["results"]) == [0, 1, 2]
    for c, ref in refs.items():
        r = out["results"][c]
        assert (r["n_iter"], r["converged"], r["n_resolved"]) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
        assert r["n_new_per_iter"] == [int(v) for v in ref["n_new_per_iter"]]
        for name in pool.ROW_NAMES:
            want = 1 if (c == 2 and name == "median") else 0
            assert r["diff"][name]["n_diff"] == want, (c, name, r["diff"][name])
        assert set(r["stage_s"]) == {"sample", "noise", "deposit", "estimator_passes", "snr_passes", "subtract"}
    assert out["results"][2]["diff"]["median"]["first"] == 5
    # one process: the same path without a pool
    one = pool.simulate_many(w, [0], n_proc=1)
    assert one["results"][0]["n_resolved"] == refs[0]["n_resolved"]
