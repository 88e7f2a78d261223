"""The C ABI without a GPU: the library loads, exports every function include/gbfg.h declares, and the
argument checks that run before any CUDA call answer with the documented status (include/gbfg.h)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gbfg.h")


@pytest.fixture(scope="module")
def gbcpu():
    import paper_2602_18560_b200 as gb
    from paper_2602_18560_b200 import build
    build.build()          # nvcc cross-compiles without a GPU
    gb.load()
    return gb


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gbfg_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_five_calls_of_the_north_star():
    names = declared_functions()
    for f in ["gbfg_sample_catalog", "gbfg_deposit", "gbfg_running_median", "gbfg_snr_select",
              "gbfg_subtract_until_converged"]:
        assert f in names


def test_library_exports_every_declared_function(gbcpu):
    lib = C.CDLL(gbcpu.LIB_PATH)
    names = declared_functions()
    assert len(names) >= 18
    for f in names:
        assert hasattr(lib, f), f"{f} is declared in gbfg.h but not exported"
    assert sorted(gbcpu.EXPORTS) == names          # the binding knows exactly the declared set


def test_struct_sizes_match_the_header(gbcpu):
    # gbfg_grid: 2 x 4 + 3 x 8 + 8; gbfg_pop: 2 x 4 + 5 x 8 + 8; gbfg_iter_params: 4+4+8+8+4+4+8
    assert C.sizeof(gbcpu.Grid) == 40 and C.sizeof(gbcpu.Pop) == 56 and C.sizeof(gbcpu.IterParams) == 40
    # gbfg_iter_result: 2 x 4 + 5 x 8 + 64 x 8
    assert C.sizeof(gbcpu.IterResult) == 8 + 5 * 8 + 8 * gbcpu.MAX_ITER_TRACE


def test_version_and_strerror(gbcpu):
    L = gbcpu.load()
    assert L.gbfg_version() >= 100
    assert L.gbfg_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5, -6):
        assert len(L.gbfg_strerror(code)) > 3
    assert b"static" in L.gbfg_strerror(-6)
    assert L.gbfg_strerror(-77) == b"unknown status"


def test_grid_init_n_bins_rule(gbcpu):
    """n_bins = ceil((f_max - f_min) T) (R2): the two grids of BASELINE.json."""
    g = gbcpu.grid_init(1e-4, 1e-2, 3.15581e7, -140)
    assert g.n_bins == 312426
    g = gbcpu.grid_init(1e-4, 3e-2, 4 * 3.15581e7, -140)
    assert g.n_bins == 3774349
    for bad in [(0.0, 1e-2, 1e7), (1e-2, 1e-3, 1e7), (1e-4, 1e-2, 0.0), (1e-4, 1e-2, float("nan")), (1e-4, 1e9, 1e9)]:
        with pytest.raises(gbcpu.GbfgError) as e:
            gbcpu.grid_init(bad[0], bad[1], bad[2], -140)
        assert e.value.status == -1
    with pytest.raises(gbcpu.GbfgError):
        gbcpu.grid_init(1e-4, 1e-2, 3e7, 5)


def test_invalid_arguments_are_rejected_before_any_cuda_call(gbcpu):
    L = gbcpu.load()
    g = gbcpu.grid_init(1e-4, 1e-2, 3.15581e7, -140)
    off = (C.c_int64 * 2)(0, 10)
    # running median: even window, window wider than the build supports, n_bins < h + 1, aliasing
    assert L.gbfg_running_median(8, 1000, 1, 10, 16, 32, 1 << 20, None) == -1
    assert L.gbfg_running_median(8, 100000, 1, 4099, 16, 32, 1 << 20, None) == -5
    assert L.gbfg_running_median(8, 100, 1, 1001, 16, 32, 1 << 20, None) == -1
    assert L.gbfg_running_median(8, 1000, 1, 11, 8, 32, 1 << 20, None) == -1
    assert L.gbfg_running_median(None, 1000, 1, 11, 16, 32, 1 << 20, None) == -1
    # the caller's workspace: missing, misaligned, too small
    assert L.gbfg_running_median(8, 1000, 1, 11, 16, None, 0, None) == -2
    assert L.gbfg_running_median(8, 1000, 1, 11, 16, 36, 1 << 20, None) == -2
    assert L.gbfg_running_median(8, 1000, 1, 11, 16, 32, 64, None) == -2
    need = L.gbfg_running_median_workspace_bytes(3774349, 1, 2001)
    assert 256 < need < (1 << 20) and L.gbfg_running_median_workspace_bytes(3774349, 1, 2000) == 0
    # deposit: sign, null spectrum, list without count, missing workspace
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 2, 8, None, 8, 1 << 30, None) == -1
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 1, None, None, 8, 1 << 30, None) == -1
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, 8, None, 1, 8, None, 8, 1 << 30, None) == -1
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 1, 8, None, None, 0, None) == -2
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 1, 8, None, 8, 16, None) == -2
    # offsets must start at 0 and not decrease; n_cat within GBFG_MAX_CAT
    bad_off = (C.c_int64 * 2)(1, 10)
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, bad_off, 1, None, None, 1, 8, None, 8, 1 << 30, None) == -1
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 0, None, None, 1, 8, None, 8, 1 << 30, None) == -1
    # struct_size guards
    g2 = gbcpu.Grid.from_buffer_copy(g)
    g2.struct_size = 12
    assert L.gbfg_instrument_noise(C.byref(g2), 8, None) == -1
    assert L.gbfg_workspace_bytes(C.byref(g2), 10, 1) == 0
    p = gbcpu.make_iter_params(1001, 729.0 / 512.0, 7.0, 30)
    p2 = gbcpu.IterParams.from_buffer_copy(p)
    p2.window = 1000
    res = (gbcpu.IterResult * 1)()
    assert L.gbfg_subtract_until_converged(C.byref(g), 8, 8, 8, off, 1, 8, C.byref(p2), 8, 8, 8, 8, res, 8, 1 << 40, None) == -1
    p2.window = 1001
    p2.max_iter = 0
    assert L.gbfg_subtract_until_converged(C.byref(g), 8, 8, 8, off, 1, 8, C.byref(p2), 8, 8, 8, 8, res, 8, 1 << 40, None) == -1
    # a workspace must be 32-byte aligned (the candidate records and the scan move 256-bit vectors): checked before any CUDA call
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 1, 8, None, 48, 1 << 40, None) == -2
    assert L.gbfg_deposit(C.byref(g), 8, 8, 8, off, 1, None, None, 1, 8, None, 64, 1 << 40, None) != -2


def test_profile_timeline_rejects_bad_arguments(gbcpu):
    L = gbcpu.load()
    n = C.c_int32(0)
    assert L.gbfg_profile_timeline(None, 4, C.byref(n), C.byref(n)) == -1
    buf = (gbcpu.LaunchTime * 4)()
    assert L.gbfg_profile_timeline(buf, -1, C.byref(n), C.byref(n)) == -1
    assert L.gbfg_profile_timeline(buf, 4, None, C.byref(n)) == -1


def test_paper_sampler_rejects_parameters_outside_the_stated_domain(gbcpu):
    """DESIGN.md R12: the special functions of the paper's sampler are stated and pinned for 0.25 <= alpha_Gamma <= 16."""
    L = gbcpu.load()
    g = gbcpu.grid_init(1e-4, 1e-2, 3.15581e7, -140)
    off = (C.c_int64 * 2)(0, 10)

    class P:
        alpha_pl, alpha_gamma, beta_gamma, mu_gamma, mu, sigma, rho, n_src = -2.9, 1.96, 1.8, -21.0, -22.0, 0.18, 0.5, 10

    def call(**kw):
        p = P()
        for k, v in kw.items():
            setattr(p, k, v)
        arr = (gbcpu.PopPaper * 1)(gbcpu.make_pop_paper(p))
        return L.gbfg_sample_catalog_paper(C.byref(g), arr, off, 1, 0, 1, 16, 16, 16, None)

    assert call(alpha_gamma=0.2) == -5 and call(alpha_gamma=16.5) == -5
    assert call(alpha_gamma=-1.0) == -1 and call(beta_gamma=0.0) == -1 and call(rho=1.0) == -1 and call(sigma=-0.1) == -1
    assert call(alpha_gamma=1.0) in (0, -3, -4)            # accepted: reaches the device check (no GPU here: -3 / -4)


def test_workspace_bytes_grows_with_the_problem(gbcpu):
    g = gbcpu.grid_init(1e-4, 3e-2, 4 * 3.15581e7, -140)
    a = gbcpu.workspace_bytes(g, 10**6, 1)
    b = gbcpu.workspace_bytes(g, 10**7, 1)
    c = gbcpu.workspace_bytes(g, 10**7, 4)
    assert 0 < a < b < c
    # per source: the 28 bytes of a candidate record as first compacted, its 32-byte ordered record, the index list
    assert (b - a) / 9e6 == pytest.approx(68.0, rel=0.05)


def test_no_cpu_fallback(gbcpu):
    """Without a CUDA device a compute call fails loudly (GBFG_ERR_CUDA / GBFG_ERR_ARCH), it never computes."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = gbcpu.load()
    g = gbcpu.grid_init(1e-4, 1e-2, 3.15581e7, -140)
    out = np.zeros(16)
    assert L.gbfg_instrument_noise(C.byref(g), out.ctypes.data, None) in (-3, -4)
    assert np.all(out == 0.0)
