"""gbfg_running_median_static: the running median for callers that cannot allocate (include/gbfg.h).

Its scratch (the list of tiles the 32-bit-key kernel hands to the 64-bit-key one) is a static array in the library's
device image instead of a caller's workspace.  The results must be those of gbfg_running_median to the bit (integer work:
the tolerance of every running-median test here is zero), on calls in a row that share the array and leave different
contents in it.  Collected last (the file name), so that a failure here hides no other test under `pytest -x`.
"""
import numpy as np
import pytest

import gbfg_workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    return t


def both_paths(gb, torch, x, n, n_cat, window):
    xd = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ref = torch.empty(x.shape, dtype=torch.int64, device="cuda")
    out = torch.full(x.shape, -7, dtype=torch.int64, device="cuda")
    gb.running_median(xd, n, n_cat, window, ref)                  # the existing path: workspace from the caller
    gb.running_median_static(xd, n, n_cat, window, out)           # the static array
    torch.cuda.synchronize()
    return out.cpu().numpy(), ref.cpu().numpy()


def test_static_scratch_matches_the_workspace_path_on_calls_in_a_row(gb, torch):
    # full64 / straddle32: every tile goes through the list in the static array; lognormal: none does, and the list of the
    # call before is still there; then a longer list than any before, and a batch of rows
    cases = [("full64", 30000, 1, 2001), ("lognormal", 30000, 1, 2001), ("straddle32", 52000, 1, 1001),
             ("full64", 9000, 1, 4097), ("zeros", 20011, 1, 33), ("full64", 15000, 3, 1001), ("full64", 30000, 1, 2001)]
    for i, (kind, n, n_cat, window) in enumerate(cases):
        rows = [wl.random_spectrum(n, seed=7000 + 10 * i + r, kind=kind) for r in range(n_cat)]
        x = np.stack(rows) if n_cat > 1 else rows[0]
        got, ref = both_paths(gb, torch, x, n, n_cat, window)
        assert np.array_equal(got, ref), (i, kind, n, n_cat, window)


def test_static_scratch_same_input_twice(gb, torch):
    n, window = 41000, 2001
    x = wl.random_spectrum(n, seed=99, kind="full64")
    x[::7] = wl.random_spectrum(n, seed=98, kind="lognormal")[::7]
    first, ref = both_paths(gb, torch, x, n, 1, window)
    second, _ = both_paths(gb, torch, x, n, 1, window)
    assert np.array_equal(first, ref) and np.array_equal(second, ref)


def test_static_scratch_against_the_oracle(gb, orc, torch):
    n, window = 20000, 1001
    x = wl.random_spectrum(n, seed=5, kind="straddle32")
    out = torch.empty(n, dtype=torch.int64, device="cuda")
    gb.running_median_static(torch.from_numpy(x).cuda(), n, 1, window, out)
    assert np.array_equal(out.cpu().numpy(), orc.running_median(x, window))


def test_static_scratch_limit_is_an_error_and_launches_nothing(gb, torch):
    # 64 rows of 1024 tiles each: 65536 > GBFG_STATIC_MAX_TILES = 65520.  The call returns before it touches the arrays,
    # so small ones stand in for them
    window = 1
    n = 8704 * 1024
    small = torch.zeros(16, dtype=torch.int64, device="cuda")
    out = torch.full((16,), -7, dtype=torch.int64, device="cuda")
    before = gb.kernel_launch_count()
    with pytest.raises(gb.GbfgError) as e:
        gb.running_median_static(small, n, 64, window, out)
    assert e.value.status == -6 and "static" in str(e.value)
    assert gb.kernel_launch_count() == before
    torch.cuda.synchronize()
    assert (out == -7).all().item()
    assert gb.STATIC_MAX_TILES == 65520
    # the largest batch under the limit by the same rule is accepted as far as the argument checks go: invalid arguments
    # keep their own codes
    with pytest.raises(gb.GbfgError) as e:
        gb.running_median_static(small, n, 64, 2, out)
    assert e.value.status == -1
