"""The N > 1 path on CPU: world_size-2 gloo processes deal the catalogs of a small batch between them
(paper_2602_18560_b200.shard), each runs its share (here through the oracle: no GPU in this container), and
the gathered outcomes and the max-over-ranks time are those of the single-process run.  No collective
touches the data path."""
import os
import socket

import numpy as np
import pytest

import gbfg_workloads as wl
from paper_2602_18560_b200 import shard


def test_partition_covers_every_catalog_once_and_balances():
    pops = wl.config4_population_table(64, 4)
    n = [p.n_src for p in pops]
    for world in (1, 2, 3, 8):
        parts = shard.partition_catalogs(n, world)
        assert sorted(c for p in parts for c in p) == list(range(64))
        loads = [sum(n[c] for c in p) for p in parts]
        assert max(loads) - min(loads) <= max(n)            # LPT bound
        assert parts == shard.partition_catalogs(n, world)  # deterministic
    assert shard.partition_catalogs([5, 5, 5], 2) == [[0, 2], [1]]
    assert shard.local_offsets([3, 4, 5], [0, 2]) == [0, 3, 8]
    with pytest.raises(ValueError):
        shard.partition_catalogs(n, 0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _batch():
    w = wl.scaled(wl.config(4), n_cat=5, name="cfg4_small")
    pops = [wl.replace(p, n_src=1500 + 700 * i) for i, p in enumerate(w.pops)]
    return wl.replace(wl.replace(w, pops=pops), f_max=3e-3, window=301)


def _run_share(w, cat_ids):
    import oracle
    oracle.build()
    oracle.lib()
    out = {}
    for c in cat_ids:
        r = oracle.simulate(w, cat=c)
        out[c] = {"n_iter": int(r["n_iter"]), "n_resolved": int(r["n_resolved"]),
                  "psd_sum": float(np.sum(r["psd"])), "n_src": int(r["A"].size)}
    return out


def _worker(rank, world, port, ret):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _batch()
        n = [p.n_src for p in w.pops]
        mine = shard.partition_catalogs(n, world)[rank]
        local = _run_share(w, mine)
        merged = shard.gather_outcomes(local)
        t = shard.max_over_ranks(10.0 + rank)               # the job's step time is the slowest rank's
        units = sum(v["n_src"] for v in merged.values())
        ret[rank] = (mine, merged, t, units)
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_matches_single_process():
    import torch.multiprocessing as mp
    world = 2
    port = _free_port()
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
        got = dict(ret)
    w = _batch()
    single = _run_share(w, range(w.n_cat))
    assert sorted(got[0][0] + got[1][0]) == list(range(w.n_cat))
    assert got[0][0] and got[1][0]                           # both ranks worked
    for rank in range(world):
        mine, merged, t, units = got[rank]
        assert merged == single                              # every rank sees every catalog's outcome, bit-equal sums
        assert t == 11.0
        assert units == w.n_src_total


def test_duplicate_catalog_is_a_partition_bug():
    # single process: gather is the identity
    assert shard.gather_outcomes({3: {"n_iter": 2}}) == {3: {"n_iter": 2}}
    assert shard.max_over_ranks(2.5) == 2.5
