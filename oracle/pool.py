"""The oracle over several independent catalogs at once, one process per catalog.  TEST INFRASTRUCTURE ONLY.

configs[4] is 64 independent catalogs (the SBI training set); each runs through the plain
single-threaded oracle (oracle.simulate) unchanged, here merely in several processes side by side so that the
host cores of the box check (tests/test_gpu_parity.py::test_loop_config4_full) or time (bench.py's config-4 leg,
SURVEY.md 8(d)) all of them in minutes.  Nothing of the method is parallelised: a worker is `oracle.simulate(w, cat=c)`.

Comparison with another implementation's arrays happens inside the workers, element by element, against .npy files
the caller wrote (`compare_dir`): `<name>_<cat>.npy` for name in ROW_NAMES.  The oracle never reads an expected
value from them; it only reports where the two differ.
"""
from __future__ import annotations

import multiprocessing as mp
import os
import time
from typing import Dict, List, Optional, Sequence

import numpy as np

ROW_NAMES = ("total", "residual", "median", "psd", "resolved")


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _as_bits(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a)
    return a.view(np.int64) if a.dtype.itemsize == 8 else a.view(np.uint8)


def _one(task):
    w, cat, estimator, compare_dir = task
    import oracle
    oracle.lib()
    t0 = time.perf_counter()
    out = oracle.simulate(w, cat=cat, estimator=estimator)
    dt = time.perf_counter() - t0
    res = {"cat": cat, "seconds": dt, "n_src": int(out["A"].size), "n_iter": int(out["n_iter"]),
           "converged": int(out["converged"]), "n_resolved": int(out["n_resolved"]),
           "n_near_threshold": int(out["n_near_threshold"]), "rejected": int(out["rejected"]),
           "n_new_per_iter": [int(v) for v in out["n_new_per_iter"]], "stage_s": out["stage_s"]}
    if compare_dir:
        diff = {}
        for name in ROW_NAMES:
            path = os.path.join(compare_dir, f"{name}_{cat}.npy")
            got = np.load(path, mmap_mode="r")
            ref = _as_bits(out[name])
            gotb = _as_bits(np.asarray(got))
            if gotb.shape != ref.shape:
                diff[name] = {"n_diff": -1, "first": -1, "shape": [list(gotb.shape), list(ref.shape)]}
                continue
            ne = np.flatnonzero(gotb != ref)                  # element by element
            diff[name] = {"n_diff": int(ne.size), "first": int(ne[0]) if ne.size else -1, "n": int(ref.size)}
        res["diff"] = diff
    return res


def simulate_many(w, cats: Sequence[int], n_proc: Optional[int] = None, estimator: int = 0,
                  compare_dir: Optional[str] = None) -> Dict[str, object]:
    """oracle.simulate(w, cat=c) for every c in cats over a pool of n_proc processes (default: the host cores the
    process may use, at most 32 — a 1e7-source catalog holds ~0.6 GB while it runs).  Largest catalogs first.
    -> {"results": {cat: {...}}, "wall_seconds": ..., "n_proc": ...}"""
    import oracle
    oracle.build()
    cats = list(cats)
    if n_proc is None:
        n_proc = min(host_cores(), 32)
    n_proc = max(1, min(n_proc, len(cats)))
    order = sorted(cats, key=lambda c: (-int(w.pops[c].n_src), c))
    tasks = [(w, c, estimator, compare_dir) for c in order]
    t0 = time.perf_counter()
    if n_proc == 1:
        done: List[dict] = [_one(t) for t in tasks]
    else:
        ctx = mp.get_context("spawn")             # the parent may hold a CUDA context: never fork it
        with ctx.Pool(n_proc) as pool:
            done = pool.map(_one, tasks, chunksize=1)
    wall = time.perf_counter() - t0
    return {"results": {r["cat"]: r for r in done}, "wall_seconds": wall, "n_proc": n_proc}
