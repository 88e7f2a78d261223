"""Parity of the CUDA path (through the C ABI) with the oracle, stage by stage and for the whole loop.

Bars (BASELINE.json:north_star): catalogs, spectra, medians, PSDs bit-exact; resolved sets identical
(sources within 1e-9 of the threshold counted); fp64 SNR relative error <= 1e-12.
All inputs are seeded and synthetic (gbfg_workloads).
"""
import numpy as np
import pytest

import gbfg_workloads as wl

pytestmark = pytest.mark.gpu

RHO2_RTOL = 1e-12          # north_star: "fp64 SNR values: relative error <= 1e-12"


@pytest.fixture(scope="module")
def torch():
    import torch as t
    return t


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def bits(a):
    return np.ascontiguousarray(a).view(np.int64)


def gpu_grid(gb, w):
    return gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)


def workspace(torch, gb, g, n, n_cat=1):
    return torch.empty(gb.workspace_bytes(g, n, n_cat), dtype=torch.uint8, device="cuda")


# ------------------------------------------------------------------------------------- stage (i)
@pytest.mark.parametrize("case", ["cfg0", "cfg1", "odd_offset_batch", "slopes"])
def test_sample_catalog_bit_exact(gb, orc, torch, case):
    if case == "cfg0":
        w = wl.config(0)
    elif case == "cfg1":
        w = wl.config(1)
    elif case == "odd_offset_batch":      # odd catalog sizes: unaligned pair path, several catalogs
        w = wl.scaled(wl.config(4), n_cat=5)
        w = wl.replace(w, pops=[wl.replace(p, n_src=1001 + 2 * i + (i % 2)) for i, p in enumerate(w.pops)])
    else:                                 # slope == 1 (log-uniform branch) and slopes near it
        w = wl.config(2)
        w = wl.replace(w, pops=[wl.replace(w.pops[0], slope=s, n_src=5000) for s in (1.0, 1.0 + 1e-13, 1.2, 2.0)])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    assert g.n_bins == og.n_bins
    off = w.offsets()
    n = int(off[-1])
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    gb.sample_catalog(g, w.pops, off, w.seed, A, f, fd)
    A, f, fd = A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()
    for c, p in enumerate(w.pops):
        oA, of, ofd = orc.sample_catalog(og, p, c, w.seed)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(bits(A[s]), bits(oA))
        assert np.array_equal(bits(f[s]), bits(of))
        assert np.array_equal(bits(fd[s]), bits(ofd))


def test_sample_catalog_pieces(gb, orc, torch):
    """first_cat_id lets a batch be drawn in pieces: catalog 3 alone == catalog 3 of the batch."""
    w = wl.scaled(wl.config(4), n_cat=4, n_src=777)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = (torch.empty(777, dtype=torch.float64, device="cuda") for _ in range(3))
    gb.sample_catalog(g, [w.pops[3]], [0, 777], w.seed, A, f, fd, first_cat_id=3)
    oA, of, ofd = orc.sample_catalog(og, w.pops[3], 3, w.seed)
    assert np.array_equal(bits(A.cpu().numpy()), bits(oA))
    assert np.array_equal(bits(fd.cpu().numpy()), bits(ofd))


@pytest.mark.parametrize("cfg", [0, 2])
def test_instrument_noise_bit_exact(gb, orc, torch, cfg):
    w = wl.config(cfg)
    g = gpu_grid(gb, w)
    s = torch.empty(g.n_bins, dtype=torch.float64, device="cuda")
    gb.instrument_noise(g, s)
    ref = orc.instrument_noise(orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2))
    assert np.array_equal(bits(s.cpu().numpy()), bits(ref))


# ------------------------------------------------------------------------------------ stage (ii)
def _deposit_both(gb, orc, torch, w, A, f, fd, sel=None, sign=1, start=None):
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n = A.size
    spec0 = np.zeros(og.n_bins, dtype=np.int64) if start is None else start.copy()
    ref = spec0.copy()
    rej_ref = orc.deposit(og, A, f, fd, ref, sel=sel, sign=sign)
    d_spec = dev(torch, spec0)
    err = torch.zeros(1, dtype=torch.int64, device="cuda")
    ws = workspace(torch, gb, g, n)
    kw = {}
    if sel is not None:
        kw = dict(dev_sel_idx=dev(torch, np.append(np.asarray(sel, dtype=np.int64), 0)),   # capacity >= 1
                  dev_sel_count=dev(torch, np.array([len(sel)], dtype=np.int64)))
    gb.deposit(g, dev(torch, A), dev(torch, f), dev(torch, fd), [0, n], d_spec, ws, sign=sign, dev_err_count=err, **kw)
    return d_spec.cpu().numpy(), ref, int(err.item()), rej_ref


@pytest.mark.parametrize("kind", ["narrow", "wide", "bad", "edges", "dupes"])
@pytest.mark.parametrize("cfg", [0, 2])
def test_deposit_handmade_bit_exact(gb, orc, torch, kind, cfg):
    w = wl.config(cfg)
    A, f, fd = wl.handmade_catalog(kind, w, n=3000, seed=7 + cfg)
    got, ref, err, rej = _deposit_both(gb, orc, torch, w, A, f, fd)
    assert np.array_equal(got, ref)
    assert err == rej
    if kind == "bad":
        assert rej > 0


@pytest.mark.parametrize("cfg,n", [(0, None), (1, None), (2, 200_000)])
def test_deposit_catalog_and_subtract(gb, orc, torch, cfg, n):
    w = wl.config(cfg)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pop = w.pops[0] if n is None else wl.replace(w.pops[0], n_src=n)
    A, f, fd = orc.sample_catalog(og, pop, 0, w.seed)
    got, ref, err, rej = _deposit_both(gb, orc, torch, w, A, f, fd)
    assert np.array_equal(got, ref) and err == rej == 0
    # subtract a subset (stage v form: index list + device count), incl. duplicates of wide sources
    rng = np.random.default_rng(5)
    sel = rng.choice(A.size, size=A.size // 7, replace=False).astype(np.int64)
    got2, ref2, _, _ = _deposit_both(gb, orc, torch, w, A, f, fd, sel=sel, sign=-1, start=ref)
    assert np.array_equal(got2, ref2)
    # empty selection leaves the spectrum untouched
    got3, ref3, _, _ = _deposit_both(gb, orc, torch, w, A, f, fd, sel=np.zeros(0, dtype=np.int64), sign=-1, start=ref)
    assert np.array_equal(got3, ref)
    # +1 then -1 of everything is exactly zero
    got4, _, _, _ = _deposit_both(gb, orc, torch, w, A, f, fd, sign=-1, start=ref)
    assert not got4.any()


def test_deposit_empty_catalog(gb, torch):
    w = wl.config(0)
    g = gpu_grid(gb, w)
    spec = torch.zeros(g.n_bins, dtype=torch.int64, device="cuda")
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    gb.deposit(g, e, e, e, [0, 0], spec, workspace(torch, gb, g, 0))
    assert not spec.any().item()


# ----------------------------------------------------------------------------------- stage (iii)
@pytest.mark.parametrize("kind", ["lognormal", "dupes", "zeros", "full64", "ramp", "const"])
@pytest.mark.parametrize("n,window", [(20011, 1001), (30000, 2001), (9000, 4097), (7000, 3), (6193, 2001),
                                      (6192, 2001), (1001, 2001), (501, 1001), (12500, 101), (8190, 1), (40000, 33)])
def test_running_median_bit_exact(gb, orc, torch, kind, n, window):
    x = wl.random_spectrum(n, seed=n + window, kind=kind)
    ref = orc.running_median(x, window)
    out = torch.empty(n, dtype=torch.int64, device="cuda")
    gb.running_median(dev(torch, x), n, 1, window, out)
    assert np.array_equal(out.cpu().numpy(), ref)


@pytest.mark.parametrize("n_big_minus_h", [-3, 0, 1, 40])
@pytest.mark.parametrize("window", [101, 2001])
def test_running_median_few_loud_bins(gb, orc, torch, window, n_big_minus_h):
    """Tiles whose keys need a fourth radix pass only for a few loud bins: about h of them per tile (the count up to which
    a sort that lumps them into its top digit would still be exact), with loud values on both sides of 2^24 and at the
    edge 0x00ff0000 of that digit; then a loud plateau as wide as the window."""
    n, h = 20000, window // 2
    rng = np.random.default_rng(window + n_big_minus_h)
    x = rng.integers(1000, 1 << 20, n).astype(np.int64)
    for start in (0, 9000):                                  # first tile, and a stretch that straddles two tiles
        n_big = h + n_big_minus_h
        at = start + rng.choice(3000, n_big, replace=False)
        loud = rng.choice(np.array([0x00ff0000, 0x00ff0001, 0x00ffffff, 1 << 24, (1 << 24) + 5, 0xfffffffe, 0xffffffff,
                                    0x00feffff], dtype=np.int64), n_big)
        x[at] = loud
    ref = orc.running_median(x, window)
    out = torch.empty(n, dtype=torch.int64, device="cuda")
    gb.running_median(dev(torch, x), n, 1, window, out)
    assert np.array_equal(out.cpu().numpy(), ref)
    # the same with a plateau of loud bins as wide as the window: every median inside it is loud
    x[4000:4000 + 3 * window] = (1 << 26) + rng.integers(0, 1000, 3 * window)
    ref = orc.running_median(x, window)
    gb.running_median(dev(torch, x), n, 1, window, out)
    assert np.array_equal(out.cpu().numpy(), ref)


def test_running_median_batch_rows(gb, orc, torch):
    n, window = 15000, 1001
    rows = [wl.random_spectrum(n, seed=100 + r, kind=k) for r, k in enumerate(["lognormal", "zeros", "full64"])]
    x = np.stack(rows)
    out = torch.empty((3, n), dtype=torch.int64, device="cuda")
    gb.running_median(dev(torch, x), n, 3, window, out)
    got = out.cpu().numpy()
    for r in range(3):
        assert np.array_equal(got[r], orc.running_median(rows[r], window))


def test_psd_bit_exact(gb, orc, torch):
    w = wl.config(0)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s_instr = orc.instrument_noise(og)
    med = wl.random_spectrum(og.n_bins, seed=3, kind="zeros")
    for norm in (1.0, wl.MEDIAN_NORM_PAPER):
        ref = orc.psd_from_median(med, s_instr, norm, w.scale_log2)
        out = torch.empty(og.n_bins, dtype=torch.float64, device="cuda")
        gb.psd(dev(torch, med), dev(torch, s_instr), og.n_bins, 1, norm, w.scale_log2, out)
        assert np.array_equal(bits(out.cpu().numpy()), bits(ref))


# ------------------------------------------------------------------------------------ stage (iv)
def _snr_case(gb, orc, torch, w, A, f, fd, rho_th, resolved0=None, psd=None):
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n = A.size
    if psd is None:
        s_instr = orc.instrument_noise(og)
        spec = np.zeros(og.n_bins, dtype=np.int64)
        orc.deposit(og, A, f, fd, spec)
        psd = orc.psd_from_median(orc.running_median(spec, w.window), s_instr, w.median_norm, w.scale_log2)
    res_ref = np.zeros(n, dtype=np.uint8) if resolved0 is None else resolved0.copy()
    res_gpu = dev(torch, res_ref)
    sel_ref, r2_ref, near_ref = orc.snr_select(og, A, f, fd, psd, rho_th, res_ref)
    r2 = torch.full((n,), -1.0, dtype=torch.float64, device="cuda")
    sel = torch.empty(max(n, 1), dtype=torch.int64, device="cuda")
    cnt = torch.empty(2, dtype=torch.int64, device="cuda")
    near = torch.zeros(1, dtype=torch.int64, device="cuda")
    gb.snr_select(g, dev(torch, A), dev(torch, f), dev(torch, fd), [0, n], dev(torch, psd), rho_th, res_gpu, sel, cnt,
                  workspace(torch, gb, g, n), dev_rho2_out=r2, dev_near_count=near)
    cnt = cnt.cpu().numpy()
    got_sel = np.sort(sel.cpu().numpy()[: cnt[0]])
    r2 = r2.cpu().numpy()
    tested = (np.zeros(n, dtype=np.uint8) if resolved0 is None else resolved0) == 0
    # untested entries untouched, rejected sources NaN on both sides
    assert np.all(r2[~tested] == -1.0)
    assert np.array_equal(np.isnan(r2[tested]), np.isnan(r2_ref[tested]))
    okm = tested & ~np.isnan(r2_ref)
    rel = np.abs(r2[okm] - r2_ref[okm]) / np.maximum(np.abs(r2_ref[okm]), 1e-300)
    assert rel.size == 0 or rel.max() <= RHO2_RTOL, rel.max()
    assert cnt[0] == cnt[1] == sel_ref.size
    assert np.array_equal(got_sel, sel_ref)                    # identical resolved set
    assert np.array_equal(res_gpu.cpu().numpy(), res_ref)
    assert int(near.item()) == near_ref
    return rel.max() if rel.size else 0.0, near_ref


@pytest.mark.parametrize("cfg,n", [(0, None), (1, None), (2, 300_000)])
def test_snr_select_catalog(gb, orc, torch, cfg, n):
    w = wl.config(cfg)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pop = w.pops[0] if n is None else wl.replace(w.pops[0], n_src=n)
    A, f, fd = orc.sample_catalog(og, pop, 0, w.seed)
    rng = np.random.default_rng(9)
    resolved0 = (rng.random(A.size) < 0.1).astype(np.uint8)
    _snr_case(gb, orc, torch, w, A, f, fd, w.rho_th)
    _snr_case(gb, orc, torch, w, A, f, fd, w.rho_th, resolved0=resolved0)
    _snr_case(gb, orc, torch, w, A, f, fd, float("inf"))
    _snr_case(gb, orc, torch, w, A, f, fd, 1e-30)


@pytest.mark.parametrize("kind", ["narrow", "wide", "bad", "edges", "dupes"])
def test_snr_select_handmade(gb, orc, torch, kind):
    w = wl.config(2)
    A, f, fd = wl.handmade_catalog(kind, w, n=2000, seed=21)
    _snr_case(gb, orc, torch, w, A, f, fd, w.rho_th)


def test_snr_threshold_decisions_on_the_definition(gb, orc, torch):
    """Wide sources whose rho^2 sits within rounding of the threshold: the decision is the oracle's."""
    w = wl.config(2)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = wl.handmade_catalog("wide", w, n=400, seed=33)
    s_instr = orc.instrument_noise(og)
    spec = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec)
    psd = orc.psd_from_median(orc.running_median(spec, w.window), s_instr, w.median_norm, w.scale_log2)
    # rescale every amplitude so that its own rho^2 lands within a few ulp of 49
    r2 = np.array([orc.rho2(og, A[i], f[i], fd[i], psd) for i in range(A.size)])
    ok = ~np.isnan(r2) & (r2 > 0)
    A2 = A.copy()
    A2[ok] = A[ok] * np.sqrt(49.0 / r2[ok]) * (1.0 + np.random.default_rng(1).integers(-3, 4, ok.sum()) * 1.1e-16)
    _, near = _snr_case(gb, orc, torch, w, A2, f, fd, 7.0, psd=psd)      # same PSD: rho^2 scales exactly as A^2
    assert near >= ok.sum() // 2


# ------------------------------------------------------------------------------- the whole loop
def _loop_case(gb, orc, torch, w, max_iter=None, rho_th=None, check_host=False, flags=0):
    max_iter = w.max_iter if max_iter is None else max_iter
    rho_th = w.rho_th if rho_th is None else rho_th
    w = wl.replace(w, max_iter=max_iter, rho_th=rho_th)
    ref = orc.simulate(w)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    s_instr = dev(torch, ref["s_instr"])
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    err = torch.zeros(1, dtype=torch.int64, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, rho_th, max_iter, flags)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, s_instr, params, A, f, fd, total, spec, med, psd, resolved,
                      workspace(torch, gb, g, n), dev_err_count=err)[0]
    assert np.array_equal(bits(A.cpu().numpy()), bits(ref["A"]))
    assert np.array_equal(total.cpu().numpy(), ref["total"])              # deposited spectrum: bit-exact
    assert np.array_equal(spec.cpu().numpy(), ref["residual"])            # residual: bit-exact
    assert np.array_equal(med.cpu().numpy(), ref["median"])               # median: bit-exact
    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))      # final PSD: bit-exact
    assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])        # resolved set: identical
    assert (res.n_iter, res.converged, res.n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    assert res.n_near_threshold == ref["n_near_threshold"]
    k = min(ref["n_iter"], gb.MAX_ITER_TRACE)
    assert list(res.n_new_per_iter[:k]) == list(ref["n_new_per_iter"][:k])
    assert int(err.item()) == ref["rejected"]
    if check_host:
        hp = np.empty(nb, dtype=np.float64)
        hr = np.empty(n, dtype=np.uint8)
        res2 = gb.simulate_host(g, w.pops, w.offsets(), w.seed, ref["s_instr"], params, hp, hr)[0]
        assert np.array_equal(bits(hp), bits(ref["psd"])) and np.array_equal(hr, ref["resolved"])
        assert res2.n_iter == ref["n_iter"]
    return ref


def test_loop_config0(gb, orc, torch):
    _loop_case(gb, orc, torch, wl.config(0), check_host=True)


def test_loop_config1(gb, orc, torch):
    _loop_case(gb, orc, torch, wl.config(1))


def test_loop_dense_short(gb, orc, torch):
    ref = _loop_case(gb, orc, torch, wl.dense_case("short"))
    assert ref["n_iter"] >= 4


def test_loop_dense_long(gb, orc, torch):
    ref = _loop_case(gb, orc, torch, wl.dense_case("long"))
    assert ref["n_iter"] >= 10


def test_loop_degenerate_thresholds_and_cap(gb, orc, torch):
    w = wl.config(0)
    ref = _loop_case(gb, orc, torch, w, rho_th=float("inf"))
    assert ref["n_iter"] == 1 and ref["n_resolved"] == 0
    ref = _loop_case(gb, orc, torch, w, rho_th=1e-30)
    assert not ref["residual"].any()
    ref = _loop_case(gb, orc, torch, wl.dense_case("short"), max_iter=1)       # cap branch
    assert ref["converged"] == 0
    ref = _loop_case(gb, orc, torch, wl.dense_case("short"), max_iter=3)
    assert ref["converged"] == 0 and ref["n_iter"] == 3


@pytest.mark.parametrize("flags", [1, 2, 3])
def test_loop_without_the_result_preserving_optimisations(gb, orc, torch, flags):
    """GBFG_FLAG_NO_PRESELECT (1) and GBFG_FLAG_NO_INCREMENTAL (2): pre-selection (R5) and dirty blocks
    (R7) never change a result, so the loop without them matches the oracle exactly as the default loop does."""
    _loop_case(gb, orc, torch, wl.dense_case("short"), flags=flags)
    _loop_case(gb, orc, torch, wl.config(1), flags=flags)


@pytest.mark.slow
def test_loop_config2_full(gb, orc, torch):
    ref = _loop_case(gb, orc, torch, wl.config(2))
    assert ref["n_iter"] > 10


@pytest.mark.slow
def test_loop_config3_full(gb, orc, torch):
    """The headline workload, in the launch configuration bench.py times."""
    _loop_case(gb, orc, torch, wl.config(3))


def test_loop_batch_matches_per_catalog_oracle(gb, orc, torch):
    """configs[4] in miniature: ragged catalogs with different Lambda iterate independently."""
    w = wl.scaled(wl.config(4), n_cat=4)
    w = wl.replace(w, pops=[wl.replace(p, n_src=n) for p, n in zip(w.pops, (60_000, 25_001, 90_000, 40_003))])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    s_instr_h = orc.instrument_noise(og)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, s_instr_h), params, A, f, fd, total, spec, med, psd,
                      resolved, workspace(torch, gb, g, n, nc))
    off = w.offsets()
    iters = set()
    for c in range(nc):
        ref = orc.simulate(w, cat=c)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(total[c].cpu().numpy(), ref["total"])
        assert np.array_equal(spec[c].cpu().numpy(), ref["residual"])
        assert np.array_equal(med[c].cpu().numpy(), ref["median"])
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"])
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
        assert res[c].n_near_threshold == ref["n_near_threshold"]
        iters.add(ref["n_iter"])
    assert len(iters) > 1          # the catalogs really stop at different iterations


@pytest.mark.slow
def test_loop_config4_full(gb, orc, torch):
    """configs[4] at full size (64 catalogs, 2.97e8 sources) in one batched launch sequence, EVERY catalog against the
    oracle element by element: total, residual, median, PSD, resolved flags, iteration count, outcome, per-iteration
    trace.  The 64 oracle runs are independent single-threaded runs of oracle.simulate, spread over the host cores by
    oracle/pool.py; each worker compares its catalog's rows with the GPU's (written to a scratch directory).
    GBFG_CFG4_CATS=n limits the oracle to the n smallest catalogs plus the largest (a box with few cores).  Every catalog
    is also checked through properties that hold at any size: power conservation in fixed point (total - residual = the
    deposit of exactly the resolved sources), residual and median >= 0, PSD >= S_instr, the iteration trace adds up."""
    import os
    import shutil
    import tempfile
    from oracle import pool
    w = wl.config(4)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    s_instr_h = orc.instrument_noise(og)
    s_instr = dev(torch, s_instr_h)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    ws = workspace(torch, gb, g, n, nc)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, s_instr, params, A, f, fd, total, spec, med, psd, resolved, ws)
    off = w.offsets()
    # properties, every catalog
    assert int(spec.min().item()) >= 0 and int(med.min().item()) >= 0
    assert bool((psd >= s_instr.unsqueeze(0)).all().item())
    sel = torch.nonzero(resolved, as_tuple=False).flatten().to(torch.int64)
    cnt = torch.tensor([sel.numel()], dtype=torch.int64, device="cuda")
    redep = torch.zeros((nc, nb), dtype=torch.int64, device="cuda")
    gb.deposit(g, A, f, fd, off, redep, ws, sign=+1, dev_sel_idx=sel, dev_sel_count=cnt)
    assert torch.equal(total - spec, redep)                       # power conservation, exactly
    del redep
    for c in range(nc):
        r = res[c]
        k = min(r.n_iter, gb.MAX_ITER_TRACE)
        assert 1 <= r.n_iter <= w.max_iter
        assert sum(r.n_new_per_iter[:k]) == r.n_resolved
        assert (r.n_new_per_iter[r.n_iter - 1] == 0) == bool(r.converged)
        assert int(resolved[int(off[c]):int(off[c + 1])].sum().item()) == r.n_resolved
    # the oracle, element by element, on every catalog
    order = sorted(range(nc), key=lambda c: w.pops[c].n_src)
    limit = int(os.environ.get("GBFG_CFG4_CATS", "0"))
    cats = order if limit <= 0 or limit >= nc else sorted(set(order[:limit] + [order[-1]]))
    tmp = tempfile.mkdtemp(prefix="gbfg_cfg4_")
    try:
        rows = {"total": total, "residual": spec, "median": med, "psd": psd}
        for c in cats:
            for name, t in rows.items():
                np.save(os.path.join(tmp, f"{name}_{c}.npy"), t[c].cpu().numpy())
            np.save(os.path.join(tmp, f"resolved_{c}.npy"), resolved[int(off[c]):int(off[c + 1])].cpu().numpy())
        out = pool.simulate_many(w, cats, compare_dir=tmp)
    finally:
        shutil.rmtree(tmp, ignore_errors=True)
    bad = []
    for c in cats:
        o, r = out["results"][c], res[c]
        if any(o["diff"][name]["n_diff"] != 0 for name in pool.ROW_NAMES):
            bad.append((c, {k: v for k, v in o["diff"].items() if v["n_diff"] != 0}))
        if (r.n_iter, r.converged, r.n_resolved, r.n_near_threshold) != (o["n_iter"], o["converged"], o["n_resolved"], o["n_near_threshold"]):
            bad.append((c, "outcome", (r.n_iter, r.converged, r.n_resolved), (o["n_iter"], o["converged"], o["n_resolved"])))
        k = min(o["n_iter"], gb.MAX_ITER_TRACE)
        if list(r.n_new_per_iter[:k]) != o["n_new_per_iter"][:k]:
            bad.append((c, "trace"))
    n_ok = len(cats) - len({b[0] for b in bad})
    print(f"config 4: {n_ok}/{len(cats)} catalogs bit-exact against the oracle "
          f"({out['n_proc']} oracle processes, {out['wall_seconds']:.0f} s)")
    assert not bad, f"{n_ok}/{len(cats)} catalogs match the oracle; differing: {bad[:4]}"
    assert len(cats) == nc or limit > 0


# ------------------------------------------------- running-mean estimator, eq. (D1) (R8)
@pytest.mark.parametrize("kind", ["lognormal", "dupes", "zeros", "ramp", "const"])
@pytest.mark.parametrize("n,window", [(20011, 1001), (30000, 2001), (9000, 4097), (7000, 3), (6193, 2001),
                                      (1001, 2001), (40000, 1)])
def test_running_mean_bit_exact(gb, orc, torch, kind, n, window):
    x = wl.random_spectrum(n, seed=3 * n + window, kind=kind)
    ref = orc.running_sum(x, window)
    s_instr = 10.0 ** np.random.default_rng(n).uniform(-41, -33, n)
    out = torch.empty(n, dtype=torch.int64, device="cuda")
    psd = torch.empty(n, dtype=torch.float64, device="cuda")
    gb.running_mean(dev(torch, x), n, 1, window, out, dev(torch, s_instr), -140, psd)
    assert np.array_equal(out.cpu().numpy(), ref)
    assert np.array_equal(bits(psd.cpu().numpy()), bits(orc.psd_from_sum(ref, s_instr, window, -140)))
    out2 = torch.empty(n, dtype=torch.int64, device="cuda")
    gb.running_mean(dev(torch, x), n, 1, window, out2)            # sums only
    assert np.array_equal(out2.cpu().numpy(), ref)


def test_running_mean_batch_rows_and_large_grid(gb, orc, torch):
    n, window = 3_774_349, 2001                                   # the 4-yr grid, three rows
    rows = np.stack([wl.random_spectrum(n, seed=70 + r, kind="lognormal") for r in range(3)])
    out = torch.empty((3, n), dtype=torch.int64, device="cuda")
    gb.running_mean(dev(torch, rows), n, 3, window, out)
    got = out.cpu().numpy()
    for r in range(3):
        assert np.array_equal(got[r], orc.running_sum(rows[r], window))


def _loop_case_mean(gb, orc, torch, w, flags=0):
    ref = orc.simulate(w, estimator=1)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, stat = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, gb.FLAG_ESTIMATOR_MEAN | flags)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, ref["s_instr"]), params, A, f, fd, total, spec, stat,
                      psd, resolved, workspace(torch, gb, g, n))[0]
    assert np.array_equal(total.cpu().numpy(), ref["total"])
    assert np.array_equal(spec.cpu().numpy(), ref["residual"])
    assert np.array_equal(stat.cpu().numpy(), ref["median"])              # window sums: bit-exact
    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
    assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])
    assert (res.n_iter, res.converged, res.n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    assert res.n_near_threshold == ref["n_near_threshold"]
    return ref


def test_loop_mean_estimator(gb, orc, torch):
    _loop_case_mean(gb, orc, torch, wl.config(0))
    ref = _loop_case_mean(gb, orc, torch, wl.dense_case("short"))
    assert ref["n_iter"] >= 3
    _loop_case_mean(gb, orc, torch, wl.dense_case("short"), flags=gb.FLAG_NO_PRESELECT)


@pytest.mark.slow
def test_loop_mean_estimator_config2_full(gb, orc, torch):
    _loop_case_mean(gb, orc, torch, wl.config(2))


# ------------------------------------------- coarse-graining, eqs. (13)-(14), (B1) (R10)
COARSE_RTOL = 1e-14        # compensated sums + a 256-leaf tree against the oracle's exactly rounded sum (R10)


@pytest.mark.parametrize("cfg,n_coarse,band", [(0, 100, (1e-4, 1e-2)), (2, 100, (1e-4, 1e-2)), (2, 37, None), (2, 1, None)])
def test_coarse_grain_matches_oracle(gb, orc, torch, cfg, n_coarse, band):
    w = wl.config(cfg)
    g = gpu_grid(gb, w)
    nb = g.n_bins
    rng = np.random.default_rng(cfg + n_coarse)
    psd = np.stack([10.0 ** rng.uniform(-41, -34, nb), 10.0 ** (-38 + 0.5 * np.sin(np.arange(nb) / 3e4))])
    e = wl.log_bin_edges(w, n_coarse, *(band or (None, None)))
    S = torch.empty((2, n_coarse), dtype=torch.float64, device="cuda")
    hc = torch.empty((2, n_coarse), dtype=torch.float64, device="cuda")
    fk = torch.empty(n_coarse, dtype=torch.float64, device="cuda")
    gb.coarse_grain(dev(torch, psd), nb, 2, dev(torch, e), n_coarse, w.f_min, w.t_obs, S, fk, hc)
    for r in range(2):
        S_ref, f_ref, hc_ref = orc.coarse_grain(psd[r], e, w.f_min, w.t_obs)
        assert np.allclose(S[r].cpu().numpy(), S_ref, rtol=COARSE_RTOL, atol=0, equal_nan=True)
        assert np.allclose(hc[r].cpu().numpy(), hc_ref, rtol=COARSE_RTOL, atol=0, equal_nan=True)
        assert np.allclose(fk.cpu().numpy(), f_ref, rtol=1e-15, atol=0, equal_nan=True)


def test_coarse_grain_empty_bins_and_clipping(gb, orc, torch):
    w = wl.config(0)
    g = gpu_grid(gb, w)
    nb = g.n_bins
    psd = np.full(nb, 2.0 ** -131)
    e = np.array([0, 7, 7, 100, nb, nb + 50], dtype=np.int64)           # an empty bin, one past the end
    S = torch.empty((1, 5), dtype=torch.float64, device="cuda")
    gb.coarse_grain(dev(torch, psd), nb, 1, dev(torch, e), 5, w.f_min, w.t_obs, S)
    got = S.cpu().numpy()[0]
    assert got[0] == 2.0 ** -131 and np.isnan(got[1]) and got[2] == 2.0 ** -131 and got[3] == 2.0 ** -131 and np.isnan(got[4])


# ----------------------------------------------- SciRDv1 A/E/T noise, eqs. (C1)-(C5), (B2)-(B5) (R11)
@pytest.mark.parametrize("cfg,tdi2", [(0, True), (0, False), (2, True)])
def test_instrument_noise_aet_bit_exact(gb, orc, torch, cfg, tdi2):
    w = wl.config(cfg)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    ref = orc.instrument_noise_aet(og, tdi2=tdi2)
    outs = [torch.empty(g.n_bins, dtype=torch.float64, device="cuda") for _ in range(4)]
    gb.instrument_noise_aet(g, *outs, tdi2=tdi2)
    for o, r in zip(outs, ref):
        assert np.array_equal(bits(o.cpu().numpy()), bits(r))
    only = torch.empty(g.n_bins, dtype=torch.float64, device="cuda")
    gb.instrument_noise_aet(g, dev_Sh_AA=only, tdi2=tdi2)
    assert np.array_equal(bits(only.cpu().numpy()), bits(ref[2]))


def test_loop_with_the_aet_strain_noise(gb, orc, torch):
    """The loop takes any s_instr: here S^AA / R_AA of eqs. (C3), (B2)-(B4) in place of the Robson curve."""
    w = wl.dense_case("short")
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    sh_aa = orc.instrument_noise_aet(og)[2]
    A, f, fd = orc.sample_catalog(og, w.pops[0], 0, w.seed)
    spec = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec)
    ref_spec = spec.copy()
    ref = orc.subtract_until_converged(og, A, f, fd, sh_aa, w.window, w.median_norm, w.rho_th, w.max_iter, ref_spec)
    n, nb = A.size, g.n_bins
    d_spec = dev(torch, spec)
    med = torch.empty(nb, dtype=torch.int64, device="cuda")
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.zeros(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    res = gb.subtract_until_converged(g, dev(torch, A), dev(torch, f), dev(torch, fd), [0, n], dev(torch, sh_aa), params,
                                      d_spec, med, psd, resolved, workspace(torch, gb, g, n))[0]
    assert np.array_equal(d_spec.cpu().numpy(), ref_spec)
    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
    assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])
    assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"])


# ------------------------------------------------------------------------------ edge cases of the loop
def _loop_on_given_spectrum(gb, orc, torch, w, A, f, fd, spec0, flags=0):
    """gbfg_subtract_until_converged on a caller-supplied spectrum against the oracle's loop on the same one."""
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s_instr = orc.instrument_noise(og)
    ref_spec = spec0.copy()
    ref = orc.subtract_until_converged(og, A, f, fd, s_instr, w.window, w.median_norm, w.rho_th, w.max_iter, ref_spec)
    n, nb = A.size, g.n_bins
    d_spec = dev(torch, spec0)
    med = torch.empty(nb, dtype=torch.int64, device="cuda")
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.zeros(max(n, 1), dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, flags)
    res = gb.subtract_until_converged(g, dev(torch, A), dev(torch, f), dev(torch, fd), [0, n], dev(torch, s_instr), params,
                                      d_spec, med, psd, resolved, workspace(torch, gb, g, n))[0]
    assert np.array_equal(d_spec.cpu().numpy(), ref_spec)
    assert np.array_equal(med.cpu().numpy(), ref["median"])
    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
    assert np.array_equal(resolved.cpu().numpy()[:n], ref["resolved"])
    assert (res.n_iter, res.converged, res.n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    ref["residual"] = ref_spec
    return ref, res


def test_loop_empty_catalog(gb, orc, torch):
    w = wl.config(0)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    e = np.empty(0)
    spec0 = wl.random_spectrum(og.n_bins, seed=3, kind="lognormal")
    ref, res = _loop_on_given_spectrum(gb, orc, torch, w, e, e, e, spec0)
    assert (res.n_iter, res.converged, res.n_resolved) == (1, 1, 0)


def test_loop_on_a_spectrum_that_does_not_contain_the_catalog(gb, orc, torch):
    """Only every other source was deposited: subtracting the rest drives bins and medians negative, S_n >= S_instr
    no longer holds and the pre-selection must be abandoned on the way (R5, loop.cu).  Same answer as the
    oracle, which never pre-selects."""
    w = wl.replace(wl.dense_case("short"), max_iter=6)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = orc.sample_catalog(og, wl.replace(w.pops[0], n_src=60_000), 0, w.seed)
    spec0 = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec0, sel=np.arange(0, A.size, 2, dtype=np.int64))
    ref, res = _loop_on_given_spectrum(gb, orc, torch, w, A, f, fd, spec0)
    assert ref["residual"].min() < 0 and ref["n_resolved"] > 0
    _loop_on_given_spectrum(gb, orc, torch, w, A, f, fd, spec0, flags=gb.FLAG_NO_PRESELECT)


def test_loop_batch_with_an_empty_and_a_rejected_catalog(gb, orc, torch):
    """A batch whose second catalog is empty and whose third holds sources the generator cannot place (f_max draws are
    clamped into the band, so 'rejected' is exercised through a zero-amplitude scatter instead): ragged, degenerate rows."""
    w = wl.scaled(wl.config(4), n_cat=3)
    w = wl.replace(w, pops=[wl.replace(w.pops[0], n_src=30_000), wl.replace(w.pops[1], n_src=0), wl.replace(w.pops[2], n_src=7)])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, orc.instrument_noise(og)), params, A, f, fd, total, spec,
                      med, psd, resolved, workspace(torch, gb, g, n, nc))
    off = w.offsets()
    for c in range(nc):
        ref = orc.simulate(w, cat=c)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(spec[c].cpu().numpy(), ref["residual"])
        assert np.array_equal(med[c].cpu().numpy(), ref["median"])
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"])
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    assert (res[1].n_iter, res[1].n_resolved) == (1, 0)


# ------------------------------------------------ the paper's population sampler (R12)
@pytest.mark.parametrize("case", ["fig1", "priors", "flat_in_log", "batch"])
def test_sample_catalog_paper_bit_exact(gb, orc, torch, case):
    w = wl.config(1)                                          # 0.1-10 mHz: the band of Table I
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    if case == "fig1":
        pops = [wl.PaperPopulation(n_src=150_001)]
    elif case == "priors":
        pops = [wl.paper_prior_draw(s, n_src=40_000) for s in (1, 2, 3)]
    elif case == "flat_in_log":
        pops = [wl.replace(wl.PaperPopulation(n_src=30_000), alpha_pl=-1.0, rho=0.0, sigma=0.0)]
    else:
        pops = [wl.PaperPopulation(n_src=777), wl.replace(wl.PaperPopulation(n_src=0), rho=0.5),
                wl.replace(wl.PaperPopulation(n_src=12_345), alpha_gamma=1.0, beta_gamma=3.0, rho=0.3)]
    off = np.concatenate([[0], np.cumsum([p.n_src for p in pops])]).astype(np.int64)
    n = int(off[-1])
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    gb.sample_catalog_paper(g, pops, off, 5, A, f, fd, first_cat_id=4)
    for c, p in enumerate(pops):
        rA, rf, rfd = orc.sample_catalog_paper(og, p, 4 + c, 5)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(bits(A[s].cpu().numpy()), bits(rA))
        assert np.array_equal(bits(f[s].cpu().numpy()), bits(rf))
        assert np.array_equal(bits(fd[s].cpu().numpy()), bits(rfd))


def test_paper_catalog_through_the_loop(gb, orc, torch):
    """A catalog drawn from the paper's model (Fig. 1 parameters) goes through deposit and loop like any other."""
    w = wl.replace(wl.config(1), max_iter=8)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pop = wl.PaperPopulation(n_src=200_000)
    n = pop.n_src
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    gb.sample_catalog_paper(g, [pop], [0, n], 9, A, f, fd)
    hA, hf, hfd = A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()
    spec0 = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, hA, hf, hfd, spec0)
    d_spec = torch.zeros(g.n_bins, dtype=torch.int64, device="cuda")
    gb.deposit(g, A, f, fd, [0, n], d_spec, workspace(torch, gb, g, n))
    assert np.array_equal(d_spec.cpu().numpy(), spec0)
    _loop_on_given_spectrum(gb, orc, torch, w, hA, hf, hfd, spec0)


def test_release_cached_and_reuse(gb, orc, torch):
    """gbfg_release_cached frees the host-call arena and the loop's side stream; the next calls rebuild them."""
    w = wl.config(0)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s_instr = orc.instrument_noise(og)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    hp1, hp2 = (np.empty(g.n_bins, dtype=np.float64) for _ in range(2))
    gb.simulate_host(g, w.pops, w.offsets(), w.seed, s_instr, params, hp1)
    gb.release_cached()
    gb.release_cached()                                    # idempotent
    gb.simulate_host(g, w.pops, w.offsets(), w.seed, s_instr, params, hp2)
    assert np.array_equal(bits(hp1), bits(hp2))
    _loop_case(gb, orc, torch, w)


# ------------------------------------------------- second stop rule: convergence in S_n (R13)
@pytest.mark.parametrize("tol", [1e300, 3e-2, 1e-3, 1e-6, 1e-300])
@pytest.mark.parametrize("estimator", [0, 1])
def test_loop_psd_stop_rule(gb, orc, torch, tol, estimator):
    w = wl.dense_case("short")
    ref = orc.simulate(w, estimator=estimator, psd_rtol=tol)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, stat = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    flags = gb.FLAG_ESTIMATOR_MEAN if estimator else 0
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, flags, psd_rtol=tol)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, ref["s_instr"]), params, A, f, fd, total, spec, stat,
                      psd, resolved, workspace(torch, gb, g, n))[0]
    assert (res.n_iter, res.converged, res.n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    assert np.array_equal(spec.cpu().numpy(), ref["residual"])
    assert np.array_equal(stat.cpu().numpy(), ref["median"])
    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
    assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])
    k = min(ref["n_iter"], gb.MAX_ITER_TRACE)
    assert list(res.n_new_per_iter[:k]) == list(ref["n_new_per_iter"][:k])
    if tol == 1e300:
        assert (res.n_iter, res.converged) == (2, 2)


def test_loop_psd_stop_rule_batch(gb, orc, torch):
    """Catalogs of a batch stop on their own: some by the PSD rule, at different iterations."""
    w = wl.scaled(wl.config(4), n_cat=3)
    w = wl.replace(w, pops=[wl.replace(p, n_src=n) for p, n in zip(w.pops, (80_000, 30_001, 120_000))])
    tol = 2e-3
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, psd_rtol=tol)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, orc.instrument_noise(og)), params, A, f, fd, total, spec,
                      med, psd, resolved, workspace(torch, gb, g, n, nc))
    off = w.offsets()
    outcomes = set()
    for c in range(nc):
        ref = orc.simulate(w, cat=c, psd_rtol=tol)
        s = slice(int(off[c]), int(off[c + 1]))
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
        assert np.array_equal(spec[c].cpu().numpy(), ref["residual"])
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"])
        outcomes.add((ref["n_iter"], ref["converged"]))
    assert len(outcomes) > 1


def test_running_median_random_sweep(gb, orc, torch):
    """Seeded sweep over sizes, windows and value structures (plateaus, values straddling 2^32, negatives, ties),
    sizes just above the minimum n = h + 1 and around the tile boundaries."""
    rng = np.random.default_rng(2024)
    kinds = ["lognormal", "dupes", "zeros", "full64", "plateaus", "straddle32", "negative"]
    cases = []
    for _ in range(36):
        window = int(rng.choice([1, 3, 31, 33, 255, 1001, 2001, 3001, 4097]))
        h = window // 2
        n = int(rng.choice([h + 1, h + 2, 2 * h + 1, 6192, 6193, 8192, 8193, 12384, int(rng.integers(h + 1, 40000))]))
        n = max(n, h + 1)
        cases.append((n, window, str(rng.choice(kinds)), int(rng.integers(1 << 30))))
    for n, window, kind, seed in cases:
        x = wl.random_spectrum(n, seed=seed, kind=kind)
        out = torch.empty(n, dtype=torch.int64, device="cuda")
        gb.running_median(dev(torch, x), n, 1, window, out)
        assert np.array_equal(out.cpu().numpy(), orc.running_median(x, window)), (n, window, kind, seed)
        s = torch.empty(n, dtype=torch.int64, device="cuda")
        gb.running_mean(dev(torch, x), n, 1, window, s)
        assert np.array_equal(s.cpu().numpy(), orc.running_sum(x, window)), (n, window, kind, seed)


def test_loop_batch_mean_estimator(gb, orc, torch):
    """Ragged batch with the estimator of eq. (D1): rows skip the tiles without a dirty block independently."""
    w = wl.scaled(wl.config(4), n_cat=3)
    w = wl.replace(w, pops=[wl.replace(p, n_src=n) for p, n in zip(w.pops, (50_000, 20_003, 70_000))])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    s_instr_h = orc.instrument_noise(og)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, stat = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, gb.FLAG_ESTIMATOR_MEAN)
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, s_instr_h), params, A, f, fd, total, spec, stat, psd,
                      resolved, workspace(torch, gb, g, n, nc))
    off = w.offsets()
    for c in range(nc):
        ref = orc.simulate(w, cat=c, estimator=1)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(spec[c].cpu().numpy(), ref["residual"])
        assert np.array_equal(stat[c].cpu().numpy(), ref["median"])
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"])
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
        # what the estimator recomputed: everything in the first pass, never more than everything later
        assert nb <= res[c].n_median_outputs <= (ref["n_iter"] + 1) * nb


def test_simulate_back_to_back_on_a_stream(gb, orc, torch):
    """Two calls queued on one non-default stream right behind the kernel that writes S_instr, sharing the workspace:
    the library's side stream must order itself behind the caller's stream, and a call leaves nothing in flight."""
    w = wl.config(0)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    refs = [orc.simulate(wl.replace(w, seed=s)) for s in (w.seed, w.seed + 1)]
    st = torch.cuda.Stream()
    ws = workspace(torch, gb, g, n)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    outs = []
    with torch.cuda.stream(st):
        s_instr = torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda")
        gb.instrument_noise(g, s_instr, stream=st)                          # not synchronised before the calls below
        for k, s in enumerate((w.seed, w.seed + 1)):
            A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
            total, spec, med = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
            psd = torch.empty(nb, dtype=torch.float64, device="cuda")
            resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
            res = gb.simulate(g, w.pops, w.offsets(), s, s_instr, params, A, f, fd, total, spec, med, psd, resolved, ws,
                              stream=st)[0]
            outs.append((res, spec, med, psd, resolved))
    st.synchronize()
    for ref, (res, spec, med, psd, resolved) in zip(refs, outs):
        assert np.array_equal(spec.cpu().numpy(), ref["residual"])
        assert np.array_equal(med.cpu().numpy(), ref["median"])
        assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])
        assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"])


def test_loop_repeated_runs_are_bit_identical(gb, orc, torch):
    """The kernels of one iteration start while their predecessor drains (programmatic dependent launches) and the
    plan runs on a side stream: 30 back-to-back runs of two alternating catalogs on a multi-tile grid must give the
    oracle's bits every time (a missing wait shows up as a run that differs)."""
    w = wl.config(1)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    seeds = (w.seed, w.seed + 7)
    refs = [orc.simulate(wl.replace(w, seed=s)) for s in seeds]
    s_instr = dev(torch, refs[0]["s_instr"])
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    ws = workspace(torch, gb, g, n)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    for rep in range(30):
        ref = refs[rep & 1]
        res = gb.simulate(g, w.pops, w.offsets(), seeds[rep & 1], s_instr, params, A, f, fd, total, spec, med, psd,
                          resolved, ws)[0]
        assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"]), rep
        assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"])), rep
        assert np.array_equal(med.cpu().numpy(), ref["median"]), rep
        assert np.array_equal(resolved.cpu().numpy(), ref["resolved"]), rep


def test_simulate_host_never_reads_a_stale_s_instr(gb, orc, torch):
    """gbfg_simulate_host uploads S_instr on the library's side stream while the catalog is sampled; the first
    estimator pass must wait for it.  The cached device arena still holds the previous call's S_instr (here 4x
    larger), so a pass that ran early would give another PSD.  A small catalog on the 4-yr grid: sampling and deposit
    take microseconds, the 30 MB upload half a millisecond (without the wait 7.7e5 bins of the PSD come out wrong)."""
    w = wl.config(2)
    w = wl.scaled(w, n_src=20_000, name="cfg2_20k")
    ref = orc.simulate(w)
    g = gpu_grid(gb, w)
    nb, n = g.n_bins, w.n_src_total
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    h_noise = torch.from_numpy(ref["s_instr"]).pin_memory()
    h_wrong = (h_noise * 4.0).pin_memory()
    h_psd = torch.empty(nb, dtype=torch.float64).pin_memory()
    h_res = torch.empty(n, dtype=torch.uint8).pin_memory()
    for rep in range(4):
        gb.simulate_host(g, w.pops, w.offsets(), w.seed, h_wrong.numpy(), params, h_psd.numpy(), h_res.numpy())
        res = gb.simulate_host(g, w.pops, w.offsets(), w.seed, h_noise.numpy(), params, h_psd.numpy(), h_res.numpy())[0]
        assert np.array_equal(bits(h_psd.numpy()), bits(ref["psd"])), rep
        assert np.array_equal(h_res.numpy(), ref["resolved"]), rep
        assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"])


def test_simulate_from_two_host_threads(gb, orc, torch):
    """The loop's host-side state is per host thread (side stream, events, the mapped scratch the plan kernel writes the
    iteration's counters into, the sequence number the host polls): two threads running different catalogs at the same
    time, each on its own stream and buffers, must both get the oracle's bits, run after run."""
    import threading
    w = wl.config(0)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    seeds = (w.seed, w.seed + 3)
    refs = [orc.simulate(wl.replace(w, seed=s)) for s in seeds]
    s_instr = dev(torch, refs[0]["s_instr"])
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    torch.cuda.synchronize()
    errors = []

    def run(k):
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
                total, spec, med = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
                psd = torch.empty(nb, dtype=torch.float64, device="cuda")
                resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
                ws = workspace(torch, gb, g, n)
                for rep in range(8):
                    res = gb.simulate(g, w.pops, w.offsets(), seeds[k], s_instr, params, A, f, fd, total, spec, med, psd,
                                      resolved, ws, stream=st)[0]
                    st.synchronize()
                    ref = refs[k]
                    assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"]), (k, rep)
                    assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"])), (k, rep)
                    assert np.array_equal(spec.cpu().numpy(), ref["residual"]), (k, rep)
                    assert np.array_equal(resolved.cpu().numpy(), ref["resolved"]), (k, rep)
        except BaseException as e:          # noqa: BLE001 — reported by the main thread
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=run, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


@pytest.mark.parametrize("pattern", ["alternating", "random", "word_edges", "pairs"])
def test_loop_dirty_block_patterns(gb, orc, torch, pattern):
    """plan_kernel keeps a row's dirty blocks as bits (32 per word) and finds the runs from the words' edges.  A window
    of 3 bins and one loud narrow source in the middle of chosen 256-bin blocks make the second pass's dirty set exactly
    those blocks: every other block (the largest possible number of runs), a random half, blocks around the word
    boundaries with the first and the (partial, 1221 = 38 * 32 + 5) last block, and pairs that straddle words.  The
    background is a spectrum the catalog is not part of, so a block the plan missed keeps a stale median."""
    w = wl.replace(wl.config(0), window=3, max_iter=5)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    nb = og.n_bins
    n_blk = (nb + 255) // 256
    assert n_blk % 32 != 0
    rng = np.random.default_rng(11)
    if pattern == "alternating":
        blocks = np.arange(0, n_blk, 2)
    elif pattern == "random":
        blocks = np.flatnonzero(rng.random(n_blk) < 0.5)
    elif pattern == "word_edges":
        edges = np.arange(32, n_blk, 32)
        blocks = np.unique(np.concatenate([[0, n_blk - 1], edges - 1, edges[::2], edges[1::3] + 1]))
    else:
        starts = np.arange(31, n_blk - 1, 7)
        blocks = np.unique(np.concatenate([starts, starts + 1]))
    last_len = nb - (n_blk - 1) * 256
    off = np.where(blocks == n_blk - 1, min(128, last_len - 2), 128)          # away from the block's ends: h = 1
    k = blocks * 256 + off
    f = w.f_min + (k + 0.5) / w.t_obs
    A = np.full(k.size, 1e-20) * (1.0 + 0.5 * rng.random(k.size))
    fd = np.zeros(k.size)
    spec0 = wl.random_spectrum(nb, seed=5, kind="lognormal")
    assert orc.deposit(og, A, f, fd, spec0) == 0
    ref, res = _loop_on_given_spectrum(gb, orc, torch, w, A, f, fd, spec0)
    assert ref["n_resolved"] >= 0.95 * k.size and ref["n_iter"] == 2     # (a few at 0.1 mHz stay under the threshold)
    hit = blocks[ref["resolved"] == 1]
    assert res.n_median_outputs == nb + sum(min(256, nb - b * 256) for b in hit)      # second pass: exactly those blocks
    _loop_on_given_spectrum(gb, orc, torch, w, A, f, fd, spec0, flags=gb.FLAG_NO_INCREMENTAL)


def test_loop_random_sweep(gb, orc, torch):
    """Seeded sweep of the whole path (sample -> deposit -> loop) over observation times, bands, windows, catalog sizes
    (down to a single source), amplitudes, slopes, thresholds, iteration caps, both estimators and the flags that switch
    the result-preserving optimisations off; every case bit-exact against the oracle.  GBFG_SWEEP_SECONDS extends the
    sweep beyond the default number of cases (8 minutes of it: 6766 cases, none differing)."""
    import os
    import time
    rng = np.random.default_rng(777)
    budget = float(os.environ.get("GBFG_SWEEP_SECONDS", "0"))
    t0, i = time.time(), 0
    while i < 40 or time.time() - t0 < budget:
        i += 1
        seed = int(rng.integers(1 << 31))
        years = float(rng.choice([0.5, 1.0, 2.0]))
        f_max = float(rng.choice([1.5e-3, 2e-3, 3e-3, 5e-3, 1e-2]))
        window = int(rng.choice([101, 501, 1001, 2001, 3001]))
        n = int(rng.choice([1, 37, 5_000, 50_000, 200_000, 333_333]))
        pop = wl.Population(n_src=n, logA_offset=float(rng.choice([-22.8, -22.5, -22.3, -22.0])),
                            slope=float(rng.uniform(1.0, 2.0)))
        w = wl.Workload(name=f"sweep{i}", t_obs=years * wl.YEAR_S, f_min=1e-4, f_max=f_max, window=window,
                        rho_th=float(rng.choice([5.0, 7.0, 12.0])), max_iter=int(rng.choice([5, 30, 60])),
                        seed=seed, pops=[pop])
        flags = int(rng.choice([0, 0, 0, 1, 2, 3]))
        try:
            if bool(rng.integers(2)) and window <= 2001:
                _loop_case_mean(gb, orc, torch, w, flags=flags)
            else:
                _loop_case(gb, orc, torch, w, flags=flags, check_host=bool(rng.integers(2)))
        except AssertionError as e:
            raise AssertionError(f"case {i}: {w} flags={flags}") from e


def _batch_case(gb, orc, torch, w, estimator=0, flags=0):
    """One batched launch sequence over w's catalogs against the oracle run catalog by catalog."""
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    A, f, fd = (torch.empty(max(n, 1), dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, stat = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(max(n, 1), dtype=torch.uint8, device="cuda")
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter,
                                 flags | (gb.FLAG_ESTIMATOR_MEAN if estimator else 0))
    res = gb.simulate(g, w.pops, w.offsets(), w.seed, dev(torch, orc.instrument_noise(og)), params, A, f, fd, total,
                      spec, stat, psd, resolved, workspace(torch, gb, g, n, nc))
    off = w.offsets()
    for c in range(nc):
        ref = orc.simulate(w, cat=c, estimator=estimator)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(total[c].cpu().numpy(), ref["total"]), c
        assert np.array_equal(spec[c].cpu().numpy(), ref["residual"]), c
        assert np.array_equal(stat[c].cpu().numpy(), ref["median"]), c
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"])), c
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"]), c
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"]), c
        assert res[c].n_near_threshold == ref["n_near_threshold"], c


def test_loop_batch_random_sweep(gb, orc, torch):
    """Seeded sweep of ragged batches in the manner of configs[4]: 2-6 catalogs per launch sequence, each with its own
    Lambda from the prior box and its own size (empty catalogs and single sources included), both estimators, the flags.
    GBFG_SWEEP_SECONDS extends it as in test_loop_random_sweep."""
    import os
    import time
    rng = np.random.default_rng(4242)
    budget = float(os.environ.get("GBFG_SWEEP_SECONDS", "0"))
    t0, i = time.time(), 0
    while i < 12 or time.time() - t0 < budget:
        i += 1
        nc = int(rng.integers(2, 7))
        pops = [wl.Population(slope=float(rng.uniform(1.0, 2.0)), logA_offset=float(rng.uniform(-23.0, -22.0)),
                              logA_sigma=float(rng.uniform(0.2, 0.6)), logMc_mean=float(rng.uniform(-0.8, -0.2)),
                              n_src=int(rng.choice([0, 1, 4_099, 30_000, 120_001])))
                for _ in range(nc)]
        w = wl.Workload(name=f"batch_sweep{i}", t_obs=float(rng.choice([0.5, 1.0])) * wl.YEAR_S, f_min=1e-4,
                        f_max=float(rng.choice([2e-3, 3e-3, 1e-2])), window=int(rng.choice([501, 1001, 2001])),
                        rho_th=float(rng.choice([5.0, 7.0])), max_iter=int(rng.choice([4, 30])),
                        seed=int(rng.integers(1 << 31)), pops=pops)
        estimator, flags = int(rng.integers(2)), int(rng.choice([0, 0, 1, 2, 3]))
        try:
            _batch_case(gb, orc, torch, w, estimator=estimator, flags=flags)
        except AssertionError as e:
            raise AssertionError(f"case {i}: {w} estimator={estimator} flags={flags}") from e


def test_sample_catalog_paper_prior_sweep(gb, orc, torch):
    """48 draws of Lambda from the priors of Table I in one batched call, each catalog bit-exact:
    the inverse Gamma CDF, Phi and its inverse and the copula (App. A) over the whole prior box.
    GBFG_SWEEP_SECONDS repeats it with further draws."""
    import os
    import time
    w = wl.config(1)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    budget = float(os.environ.get("GBFG_SWEEP_SECONDS", "0"))
    t0, rnd = time.time(), 0
    while rnd < 1 or time.time() - t0 < budget:
        pops = [wl.paper_prior_draw(1000 + 48 * rnd + s, n_src=10_007 + 64 * (s % 5)) for s in range(48)]
        off = np.concatenate([[0], np.cumsum([p.n_src for p in pops])]).astype(np.int64)
        n = int(off[-1])
        A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        gb.sample_catalog_paper(g, pops, off, 77 + rnd, A, f, fd, first_cat_id=0)
        hA, hf, hfd = A.cpu().numpy(), f.cpu().numpy(), fd.cpu().numpy()
        for c, p in enumerate(pops):
            rA, rf, rfd = orc.sample_catalog_paper(og, p, c, 77 + rnd)
            s = slice(int(off[c]), int(off[c + 1]))
            assert np.array_equal(bits(hA[s]), bits(rA)), (rnd, c, p)
            assert np.array_equal(bits(hf[s]), bits(rf)), (rnd, c, p)
            assert np.array_equal(bits(hfd[s]), bits(rfd)), (rnd, c, p)
        rnd += 1


# ------------------------------------------------- near-threshold sources that appear late (any_near)
def _replay_psds(orc, og, A, f, fd, w, n_iter_max):
    """The oracle's loop, stage by stage (test_oracle_snr_loop.py pins this composition to the C loop): the PSD of every
    iteration, the per-iteration near-threshold counts and the final flags."""
    s_instr = orc.instrument_noise(og)
    spec = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec)
    resolved = np.zeros(A.size, dtype=np.uint8)
    psds, nears, touched = [], [], np.zeros(og.n_bins, dtype=bool)
    for _ in range(n_iter_max):
        psd = orc.psd_from_median(orc.running_median(spec, w.window), s_instr, w.median_norm, w.scale_log2)
        psds.append(psd)
        sel, _, near = orc.snr_select(og, A, f, fd, psd, w.rho_th, resolved)
        nears.append(near)
        if sel.size == 0:
            break
        before = spec.copy()
        orc.deposit(og, A, f, fd, spec, sel=sel, sign=-1)
        touched |= before != spec
    return psds, nears, touched, spec


@pytest.mark.parametrize("flags", [0, 1])
def test_loop_sources_that_become_near_threshold_in_a_late_iteration(gb, orc, torch, flags):
    """Sources within 1e-9 of the threshold that FIRST come that close in iteration >= 2, on a record list of more than one
    wave of CTAs (flags = 1: every source is a candidate, 4.5e5 records = 1758 CTAs of 256 against 1184 resident).  A
    record flagged near-threshold is tested and counted in every later iteration (R7); the range of records a
    pass tests must be the same for every CTA of its launch.  The planted sources are one bin wide and sit in bins no
    subtraction touches whose value stays above the local median, so they change no median and their rho^2 follows the
    PSD of the unplanted run, which is where their amplitude is tuned."""
    w = wl.replace(wl.dense_case("short"), pops=[wl.replace(wl.dense_case("short").pops[0], n_src=450_000)], max_iter=12)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    A, f, fd = orc.sample_catalog(og, w.pops[0], 0, w.seed)
    psds, nears, touched, _ = _replay_psds(orc, og, A, f, fd, w, w.max_iter)
    assert len(psds) >= 5 and sum(nears) == 0
    spec_tot = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec_tot)
    med0 = orc.running_median(spec_tot, w.window)
    h = w.window // 2
    rng = np.random.default_rng(5)
    ok = np.flatnonzero(~touched & (spec_tot > 4 * med0) & (med0 > 0))
    ok = ok[(ok > 2 * h) & (ok < og.n_bins - 2 * h)]
    bins, pA = [], []
    for b in rng.permutation(ok):
        k = int(rng.integers(2, len(psds) - 1))
        # the PSD at b must really move between iterations k-1 and k, so that the source is not near before k
        if abs(psds[k - 1][b] / psds[k][b] - 1.0) < 1e-6:
            continue
        target = 49.0 * (1.0 - 5e-10) if len(bins) % 2 else 49.0 * (1.0 + 5e-10)
        bins.append(int(b))
        pA.append(np.sqrt(target * psds[k][b] / (2.0 * w.t_obs)))
        if len(bins) == 24:
            break
    assert len(bins) == 24
    bins = np.array(bins)
    A2 = np.concatenate([A, np.array(pA)])
    f2 = np.concatenate([f, w.f_min + (bins + 0.5) / w.t_obs])
    fd2 = np.concatenate([fd, np.zeros(bins.size)])
    psds2, nears2, _, _ = _replay_psds(orc, og, A2, f2, fd2, w, w.max_iter)
    assert nears2[0] == 0 and nears2[1] == 0 and sum(nears2[2:]) >= 12, nears2     # the construction worked
    spec0 = np.zeros(og.n_bins, dtype=np.int64)
    orc.deposit(og, A2, f2, fd2, spec0)
    for _ in range(3):                                   # a race would show as a run that differs
        ref, res = _loop_on_given_spectrum(gb, orc, torch, w, A2, f2, fd2, spec0, flags=flags)
        assert res.n_near_threshold == ref["n_near_threshold"] == sum(nears2[:ref["n_iter"]])


# ------------------------------------------------- shares of a batch on their own
def test_shares_of_a_batch_match_the_batched_run(gb, orc, torch):
    """configs[4] in miniature dealt to two ranks with shard.partition_catalogs (non-contiguous ids): each share, run
    through gbfg_simulate on its own with the catalogs' ids, gives row by row the bits of the single batched call, and
    those of the oracle (cat = c)."""
    from paper_2602_18560_b200 import shard
    w = wl.scaled(wl.config(4), n_cat=5)
    sizes = (60_000, 25_001, 90_000, 40_003, 33_000)
    w = wl.replace(w, pops=[wl.replace(p, n_src=n) for p, n in zip(w.pops, sizes)])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    s_instr = dev(torch, orc.instrument_noise(og))
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    nb = g.n_bins

    def run(pops, ids):
        off = np.concatenate([[0], np.cumsum([p.n_src for p in pops])]).astype(np.int64)
        n, nc = int(off[-1]), len(pops)
        A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
        total, spec, med = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
        psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
        resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
        res = gb.simulate(g, pops, off, w.seed, s_instr, params, A, f, fd, total, spec, med, psd, resolved,
                          workspace(torch, gb, g, n, nc), cat_ids=ids)
        return off, A, total, spec, med, psd, resolved, res

    whole = run(w.pops, None)
    parts = shard.partition_catalogs(sizes, 2)
    assert sorted(parts[0] + parts[1]) == list(range(5)) and any(b - a > 1 for p in parts for a, b in zip(p, p[1:]))
    for ids in parts:
        part = run([w.pops[c] for c in ids], ids)
        assert list(part[0]) == shard.local_offsets(sizes, ids)
        for r, c in enumerate(ids):
            sw = slice(int(whole[0][c]), int(whole[0][c + 1]))
            sp = slice(int(part[0][r]), int(part[0][r + 1]))
            assert torch.equal(part[1][sp], whole[1][sw])                         # the catalog itself
            for k in (2, 3, 4, 5):
                assert torch.equal(part[k][r].view(torch.int64), whole[k][c].view(torch.int64)), (c, k)
            assert torch.equal(part[6][sp], whole[6][sw])
            a, b = part[7][r], whole[7][c]
            assert (a.n_iter, a.converged, a.n_resolved, a.n_near_threshold) == (b.n_iter, b.converged, b.n_resolved, b.n_near_threshold)
    for c in (1, 4):                                                              # and the oracle, on two of them
        ref = orc.simulate(w, cat=c)
        assert np.array_equal(whole[3][c].cpu().numpy(), ref["residual"])
        assert np.array_equal(bits(whole[5][c].cpu().numpy()), bits(ref["psd"]))


@pytest.mark.parametrize("case", ["dense_long", "batch"])
def test_simulate_host_with_pinned_buffers(gb, orc, torch, case):
    """With a pinned PSD buffer gbfg_simulate_host sends the PSD on its way before the loop has ended and stores the
    blocks that still change afterwards straight into the host buffer (loop.cu, EarlyOut): every bin must arrive with its
    final value.  A long-tailed single catalog (about 28 iterations, most of them touching a few blocks) and a ragged
    batch whose catalogs stop at different iterations; the buffer is poisoned before every call."""
    if case == "dense_long":
        w = wl.dense_case("long")
    else:
        w = wl.scaled(wl.config(4), n_cat=3)
        w = wl.replace(w, t_obs=wl.YEAR_S, f_max=2e-3, window=1001,
                       pops=[wl.replace(p, n_src=n, logA_offset=-22.3, slope=1.5) for p, n in zip(w.pops, (300_000, 60_001, 200_000))])
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    nb, n, nc = g.n_bins, w.n_src_total, w.n_cat
    refs = [orc.simulate(w, cat=c) for c in range(nc)]
    assert max(r["n_iter"] for r in refs) >= 8
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
    h_noise = torch.from_numpy(refs[0]["s_instr"]).pin_memory()
    h_psd = torch.empty((nc, nb), dtype=torch.float64).pin_memory()
    h_res = torch.empty(n, dtype=torch.uint8).pin_memory()
    off = w.offsets()
    for rep in range(3):
        h_psd.fill_(float("nan"))
        h_res.fill_(7)
        res = gb.simulate_host(g, w.pops, off, w.seed, h_noise.numpy(), params, h_psd.numpy(), h_res.numpy())
        for c, ref in enumerate(refs):
            assert np.array_equal(bits(h_psd[c].numpy()), bits(ref["psd"])), (rep, c)
            assert np.array_equal(h_res.numpy()[int(off[c]):int(off[c + 1])], ref["resolved"]), (rep, c)
            assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
    # no curve handed in: the library's own (gbfg_instrument_noise), made on the device
    h_psd.fill_(float("nan"))
    gb.simulate_host(g, w.pops, off, w.seed, None, params, h_psd.numpy(), h_res.numpy())
    for c, ref in enumerate(refs):
        assert np.array_equal(bits(h_psd[c].numpy()), bits(ref["psd"])), c


# ------------------------------------------------- SNR summed over the TDI channels, eq. (11) (R14)
def test_channel_summed_snr_loop(gb, orc, torch):
    """gbfg_channel_sum_noise bit for bit, and the loop on S_sum as its s_instr: every SNR is then the sum over A, E, T of
    eq. (11).  With three channels instead of the strain-equivalent A channel alone more sources are resolved."""
    w = wl.dense_case("short")
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    _, _, sh_aa, sh_tt = orc.instrument_noise_aet(og)
    ref_sum = orc.channel_sum_noise(sh_aa, sh_tt)
    nb = g.n_bins
    d = [torch.empty(nb, dtype=torch.float64, device="cuda") for _ in range(3)]
    gb.instrument_noise_aet(g, dev_Sh_AA=d[0], dev_Sh_TT=d[1])
    gb.channel_sum_noise(d[0], d[1], nb, d[2])
    assert np.array_equal(bits(d[2].cpu().numpy()), bits(ref_sum))
    A, f, fd = orc.sample_catalog(og, w.pops[0], 0, w.seed)
    spec = np.zeros(nb, dtype=np.int64)
    orc.deposit(og, A, f, fd, spec)
    n = A.size
    outs = {}
    for name, curve in (("sum", ref_sum), ("aa", sh_aa)):
        ref_spec = spec.copy()
        ref = orc.subtract_until_converged(og, A, f, fd, curve, w.window, w.median_norm, w.rho_th, w.max_iter, ref_spec)
        d_spec = dev(torch, spec)
        med = torch.empty(nb, dtype=torch.int64, device="cuda")
        psd = torch.empty(nb, dtype=torch.float64, device="cuda")
        resolved = torch.zeros(n, dtype=torch.uint8, device="cuda")
        params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)
        res = gb.subtract_until_converged(g, dev(torch, A), dev(torch, f), dev(torch, fd), [0, n], dev(torch, curve), params,
                                          d_spec, med, psd, resolved, workspace(torch, gb, g, n))[0]
        assert np.array_equal(d_spec.cpu().numpy(), ref_spec)
        assert np.array_equal(bits(psd.cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved.cpu().numpy(), ref["resolved"])
        assert (res.n_iter, res.n_resolved) == (ref["n_iter"], ref["n_resolved"])
        outs[name] = ref["n_resolved"]
    assert outs["sum"] > outs["aa"]


# ------------------------------------------------- the path as the paper runs it
@pytest.mark.parametrize("estimator,tol", [(1, 2e-3), (0, 0.0)])
def test_simulate_paper_population_to_coarse_grained_psd(gb, orc, torch, estimator, tol):
    """gbfg_simulate_paper: Lambda of Table I -> catalog -> deposit -> loop -> coarse-grained S_n, f and h_c (eqs. 13-14, B1),
    two catalogs in one call, with the paper's production settings (running mean of eq. D1 + the S_n stop rule) and with
    the running median; against the oracle's stages run catalog by catalog."""
    w = wl.replace(wl.config(1), max_iter=10)
    g = gpu_grid(gb, w)
    og = orc.make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pops = [wl.PaperPopulation(n_src=150_000), wl.replace(wl.paper_prior_draw(5, n_src=90_001), mu=-21.6)]
    off = np.concatenate([[0], np.cumsum([p.n_src for p in pops])]).astype(np.int64)
    n, nb, nc = int(off[-1]), g.n_bins, len(pops)
    s_instr_h = orc.instrument_noise(og)
    edges = wl.log_bin_edges(w, 100, 1e-4, 1e-2)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, stat = (torch.empty((nc, nb), dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty((nc, nb), dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    S = torch.empty((nc, 100), dtype=torch.float64, device="cuda")
    hc = torch.empty((nc, 100), dtype=torch.float64, device="cuda")
    fk = torch.empty(100, dtype=torch.float64, device="cuda")
    flags = gb.FLAG_ESTIMATOR_MEAN if estimator else 0
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, flags, psd_rtol=tol)
    res = gb.simulate_paper(g, pops, off, 9, dev(torch, s_instr_h), params, A, f, fd, total, spec, stat, psd, resolved,
                            workspace(torch, gb, g, n, nc), dev_edges=dev(torch, edges), n_coarse=100, dev_S_coarse=S,
                            dev_f_coarse=fk, dev_hc=hc, cat_ids=[0, 1])
    for c, p in enumerate(pops):
        rA, rf, rfd = orc.sample_catalog_paper(og, p, c, 9)
        s = slice(int(off[c]), int(off[c + 1]))
        assert np.array_equal(bits(A[s].cpu().numpy()), bits(rA))
        ref_spec = np.zeros(nb, dtype=np.int64)
        orc.deposit(og, rA, rf, rfd, ref_spec)
        assert np.array_equal(total[c].cpu().numpy(), ref_spec)
        ref = orc.subtract_until_converged(og, rA, rf, rfd, s_instr_h, w.window, w.median_norm, w.rho_th, w.max_iter, ref_spec,
                                           estimator=estimator, psd_rtol=tol)
        assert np.array_equal(spec[c].cpu().numpy(), ref_spec)
        assert np.array_equal(stat[c].cpu().numpy(), ref["median"])
        assert np.array_equal(bits(psd[c].cpu().numpy()), bits(ref["psd"]))
        assert np.array_equal(resolved[s].cpu().numpy(), ref["resolved"])
        assert (res[c].n_iter, res[c].converged, res[c].n_resolved) == (ref["n_iter"], ref["converged"], ref["n_resolved"])
        S_ref, f_ref, hc_ref = orc.coarse_grain(ref["psd"], edges, w.f_min, w.t_obs)
        assert np.allclose(S[c].cpu().numpy(), S_ref, rtol=COARSE_RTOL, atol=0, equal_nan=True)
        assert np.allclose(hc[c].cpu().numpy(), hc_ref, rtol=COARSE_RTOL, atol=0, equal_nan=True)
        assert np.allclose(fk.cpu().numpy(), f_ref, rtol=1e-15, atol=0, equal_nan=True)


# ------------------------------------------------------------------------- measurement helpers
def test_profile_read_and_timeline_agree(gb, torch):
    """gbfg_profile_read (time per kernel class) and gbfg_profile_timeline (launch by launch) describe the same record:
    the same launches per class, the same summed time, starts and ends in order; and a call made with the helper off
    leaves no record."""
    w = wl.config(0)
    g = gpu_grid(gb, w)
    n, nb = w.n_src_total, g.n_bins
    s_instr = torch.empty(nb, dtype=torch.float64, device="cuda")
    gb.instrument_noise(g, s_instr)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3))
    total, spec, med = (torch.empty(nb, dtype=torch.int64, device="cuda") for _ in range(3))
    psd = torch.empty(nb, dtype=torch.float64, device="cuda")
    resolved = torch.empty(n, dtype=torch.uint8, device="cuda")
    ws = workspace(torch, gb, g, n)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter)

    def run():
        gb.simulate(g, w.pops, w.offsets(), w.seed, s_instr, params, A, f, fd, total, spec, med, psd, resolved, ws)
        torch.cuda.synchronize()

    run()
    gb.profile_enable(True)
    before = gb.kernel_launch_count()
    run()
    launched = gb.kernel_launch_count() - before
    tl = gb.profile_timeline()
    per_class = gb.profile_read()                        # clears the record
    gb.profile_enable(False)
    assert len(tl) > 0 and tl[0][1] == 0.0
    assert all(b >= a >= 0.0 for _, a, b in tl)
    assert sum(v[0] for v in per_class.values()) == len(tl) <= launched      # (a timer may bracket several launches)
    for k, (cnt, total_ms, max_ms) in per_class.items():
        mine = [b - a for kk, a, b in tl if kk == k]
        assert len(mine) == cnt
        if cnt:
            assert abs(sum(mine) - total_ms) <= 1e-3 * max(total_ms, 1e-3) + 1e-3 and abs(max(mine) - max_ms) <= 1e-3
    run()                                                # helper off: nothing recorded
    gb.profile_enable(True)
    assert gb.profile_timeline() == []
    gb.profile_enable(False)

