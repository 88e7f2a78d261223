"""ctypes binding of libgbfg (include/gbfg.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; torch supplies device memory and
the stream.  There is no CPU fallback: `load()` raises if the library is missing, and every call
raises `GbfgError` on a non-zero status.  Function names and argument order follow gbfg.h.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgbfg.so")

MAX_CAT = 256
MAX_WINDOW = 4097
MAX_ITER_TRACE = 64
FLAG_NO_PRESELECT = 1
FLAG_NO_INCREMENTAL = 2
FLAG_ESTIMATOR_MEAN = 4

EXPORTS = [
    "gbfg_version", "gbfg_strerror", "gbfg_last_cuda_error", "gbfg_grid_init", "gbfg_instrument_noise",
    "gbfg_sample_catalog", "gbfg_deposit", "gbfg_running_median", "gbfg_psd", "gbfg_snr_select",
    "gbfg_subtract_until_converged", "gbfg_simulate", "gbfg_simulate_host", "gbfg_workspace_bytes",
    "gbfg_kernel_launch_count", "gbfg_profile_enable", "gbfg_profile_read", "gbfg_release_cached",
    "gbfg_running_mean", "gbfg_coarse_grain", "gbfg_instrument_noise_aet",
    "gbfg_sample_catalog_paper", "gbfg_running_median_workspace_bytes", "gbfg_channel_sum_noise", "gbfg_simulate_paper",
    "gbfg_running_median_static", "gbfg_profile_timeline",
]

KERNEL_CLASSES = ["sample", "noise", "deposit", "scan", "median", "psd", "inv_blocks", "snr", "aux"]


class GbfgError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(what)


class Grid(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("scale_log2", C.c_int32), ("f_min", C.c_double),
                ("f_max", C.c_double), ("t_obs", C.c_double), ("n_bins", C.c_int64)]


class Pop(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("reserved", C.c_uint32), ("slope", C.c_double),
                ("logA_offset", C.c_double), ("logA_sigma", C.c_double), ("logMc_mean", C.c_double),
                ("logMc_sigma", C.c_double), ("n_src", C.c_int64)]


class PopPaper(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("reserved", C.c_uint32), ("alpha_pl", C.c_double),
                ("alpha_gamma", C.c_double), ("beta_gamma", C.c_double), ("mu_gamma", C.c_double),
                ("mu", C.c_double), ("sigma", C.c_double), ("rho", C.c_double), ("n_src", C.c_int64)]


class IterParams(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("window", C.c_int32), ("median_norm", C.c_double),
                ("rho_th", C.c_double), ("max_iter", C.c_int32), ("flags", C.c_uint32), ("psd_rtol", C.c_double)]


class IterResult(C.Structure):
    _fields_ = [("n_iter", C.c_int32), ("converged", C.c_int32), ("n_resolved", C.c_int64),
                ("n_near_threshold", C.c_int64), ("n_candidates", C.c_int64),
                ("n_median_outputs", C.c_int64), ("n_snr_tests", C.c_int64),
                ("n_new_per_iter", C.c_int64 * MAX_ITER_TRACE)]


class KernelTime(C.Structure):
    _fields_ = [("launches", C.c_int64), ("total_ms", C.c_double), ("max_ms", C.c_double)]


_lib = None


def load():
    """Loads libgbfg.so (built in-tree by paper_2602_18560_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GbfgError(-100, f"{LIB_PATH} is missing: run `python -m paper_2602_18560_b200.build` "
                              "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u32, u64, dbl, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_double, C.c_size_t
    gp, pp, ip, rp = C.POINTER(Grid), C.POINTER(Pop), C.POINTER(IterParams), C.POINTER(IterResult)
    op = C.POINTER(C.c_int64)
    L.gbfg_version.restype = C.c_int
    L.gbfg_strerror.restype = C.c_char_p
    L.gbfg_strerror.argtypes = [C.c_int]
    L.gbfg_last_cuda_error.restype = C.c_char_p
    L.gbfg_kernel_launch_count.restype = i64
    L.gbfg_grid_init.argtypes = [dbl, dbl, dbl, i32, gp]
    L.gbfg_instrument_noise.argtypes = [gp, vp, vp]
    L.gbfg_instrument_noise_aet.argtypes = [gp, dbl, dbl, dbl, i32, vp, vp, vp, vp, vp]
    L.gbfg_channel_sum_noise.argtypes = [vp, vp, i64, vp, vp]
    L.gbfg_sample_catalog.argtypes = [gp, pp, op, i32, u32, u64, vp, vp, vp, vp]
    L.gbfg_sample_catalog_paper.argtypes = [gp, C.POINTER(PopPaper), op, i32, u32, u64, vp, vp, vp, vp]
    L.gbfg_deposit.argtypes = [gp, vp, vp, vp, op, i32, vp, vp, i32, vp, vp, vp, sz, vp]
    L.gbfg_running_median.argtypes = [vp, i64, i32, i32, vp, vp, sz, vp]
    L.gbfg_running_median_static.argtypes = [vp, i64, i32, i32, vp, vp]
    L.gbfg_running_median_workspace_bytes.restype = sz
    L.gbfg_running_median_workspace_bytes.argtypes = [i64, i32, i32]
    L.gbfg_psd.argtypes = [vp, vp, i64, i32, dbl, i32, vp, vp]
    L.gbfg_running_mean.argtypes = [vp, i64, i32, i32, vp, vp, i32, vp, vp]
    L.gbfg_coarse_grain.argtypes = [vp, i64, i32, vp, i32, dbl, dbl, vp, vp, vp, vp]
    L.gbfg_snr_select.argtypes = [gp, vp, vp, vp, op, i32, vp, dbl, vp, vp, vp, vp, vp, vp, sz, vp]
    L.gbfg_subtract_until_converged.argtypes = [gp, vp, vp, vp, op, i32, vp, ip, vp, vp, vp, vp, rp, vp, sz, vp]
    L.gbfg_simulate.argtypes = [gp, pp, op, i32, u64, C.POINTER(u32), vp, ip, vp, vp, vp, vp, vp, vp, vp, vp, vp, rp, vp, sz, vp]
    L.gbfg_simulate_paper.argtypes = [gp, C.POINTER(PopPaper), op, i32, u64, C.POINTER(u32), vp, ip, vp, vp, vp, vp, vp, vp, vp, vp, vp,
                                      rp, vp, i32, vp, vp, vp, vp, sz, vp]
    L.gbfg_simulate_host.argtypes = [gp, pp, op, i32, u64, C.POINTER(u32), vp, ip, vp, vp, rp]
    L.gbfg_profile_enable.argtypes = [C.c_int]
    L.gbfg_profile_read.argtypes = [C.POINTER(KernelTime), i32]
    L.gbfg_workspace_bytes.restype = sz
    L.gbfg_workspace_bytes.argtypes = [gp, i64, i32]
    _lib = L
    return L


def _check(status: int):
    if status != 0:
        L = load()
        msg = L.gbfg_strerror(status).decode()
        if status == -3:
            msg += ": " + L.gbfg_last_cuda_error().decode()
        raise GbfgError(status, msg)


def _ptr(t) -> Optional[int]:
    """Device (or host) address of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


def _offsets(offsets: Sequence[int]):
    return (C.c_int64 * len(offsets))(*[int(o) for o in offsets])


def _pops(pops):
    arr = (Pop * len(pops))()
    for i, p in enumerate(pops):
        arr[i] = p if isinstance(p, Pop) else make_pop(p)
    return arr


def make_pop(p) -> Pop:
    """From any object with the fields of gbfg_pop (e.g. gbfg_workloads.Population)."""
    return Pop(C.sizeof(Pop), 0, p.slope, p.logA_offset, p.logA_sigma, p.logMc_mean, p.logMc_sigma, p.n_src)


def make_iter_params(window: int, median_norm: float, rho_th: float, max_iter: int, flags: int = 0,
                     psd_rtol: float = 0.0) -> IterParams:
    return IterParams(C.sizeof(IterParams), window, median_norm, rho_th, max_iter, flags, psd_rtol)


def version() -> int:
    return load().gbfg_version()


def release_cached():
    """Frees the device arena gbfg_simulate_host keeps between calls."""
    _check(load().gbfg_release_cached())


def kernel_launch_count() -> int:
    return load().gbfg_kernel_launch_count()


class LaunchTime(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("start_ms", C.c_float), ("end_ms", C.c_float)]


def profile_timeline(cap: int = 4096) -> list:
    """[(kernel class, start_ms, end_ms)] of the launches timed since the last profile_read / profile_enable, in issue
    order, times since the first launch's start."""
    arr = (LaunchTime * cap)()
    n_w, n_t = C.c_int32(0), C.c_int32(0)
    L = load()
    L.gbfg_profile_timeline.argtypes = [C.POINTER(LaunchTime), C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    _check(L.gbfg_profile_timeline(arr, cap, C.byref(n_w), C.byref(n_t)))
    return [(KERNEL_CLASSES[arr[i].kernel], float(arr[i].start_ms), float(arr[i].end_ms)) for i in range(n_w.value)]


def profile_enable(on: bool):
    _check(load().gbfg_profile_enable(1 if on else 0))


def profile_read() -> dict:
    """{kernel class: (launches, total_ms, max_ms)} of the launches timed since the last read."""
    arr = (KernelTime * len(KERNEL_CLASSES))()
    _check(load().gbfg_profile_read(arr, len(KERNEL_CLASSES)))
    return {k: (int(arr[i].launches), float(arr[i].total_ms), float(arr[i].max_ms)) for i, k in enumerate(KERNEL_CLASSES)}


def grid_init(f_min: float, f_max: float, t_obs: float, scale_log2: int = -140) -> Grid:
    g = Grid()
    _check(load().gbfg_grid_init(f_min, f_max, t_obs, scale_log2, C.byref(g)))
    return g


def workspace_bytes(grid: Grid, n_src_total: int, n_cat: int = 1) -> int:
    return load().gbfg_workspace_bytes(C.byref(grid), n_src_total, n_cat)


def instrument_noise(grid: Grid, dev_s_instr, stream=None):
    _check(load().gbfg_instrument_noise(C.byref(grid), _ptr(dev_s_instr), _stream(stream)))


def make_pop_paper(p) -> PopPaper:
    """From any object with the fields of gbfg_pop_paper (e.g. gbfg_workloads.PaperPopulation)."""
    return PopPaper(C.sizeof(PopPaper), 0, p.alpha_pl, p.alpha_gamma, p.beta_gamma, p.mu_gamma, p.mu, p.sigma, p.rho, p.n_src)


def sample_catalog_paper(grid: Grid, pops, offsets, seed: int, dev_A, dev_f, dev_fdot, first_cat_id: int = 0, stream=None):
    arr = (PopPaper * len(pops))()
    for i, p in enumerate(pops):
        arr[i] = p if isinstance(p, PopPaper) else make_pop_paper(p)
    _check(load().gbfg_sample_catalog_paper(C.byref(grid), arr, _offsets(offsets), len(pops), first_cat_id, seed,
                                            _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _stream(stream)))


def instrument_noise_aet(grid: Grid, dev_S_AA=None, dev_S_TT=None, dev_Sh_AA=None, dev_Sh_TT=None, P_pm: float = 15.0,
                         A_fm: float = 3.0, L_m: float = 2.5e9, tdi2: bool = True, stream=None):
    _check(load().gbfg_instrument_noise_aet(C.byref(grid), P_pm, A_fm, L_m, 1 if tdi2 else 0, _ptr(dev_S_AA), _ptr(dev_S_TT),
                                            _ptr(dev_Sh_AA), _ptr(dev_Sh_TT), _stream(stream)))


def channel_sum_noise(dev_Sh_AA, dev_Sh_TT, n_bins: int, dev_Sh_sum, stream=None):
    _check(load().gbfg_channel_sum_noise(_ptr(dev_Sh_AA), _ptr(dev_Sh_TT), n_bins, _ptr(dev_Sh_sum), _stream(stream)))


def sample_catalog(grid: Grid, pops, offsets, seed: int, dev_A, dev_f, dev_fdot, first_cat_id: int = 0, stream=None):
    _check(load().gbfg_sample_catalog(C.byref(grid), _pops(pops), _offsets(offsets), len(pops), first_cat_id, seed,
                                      _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _stream(stream)))


def deposit(grid: Grid, dev_A, dev_f, dev_fdot, offsets, dev_spectrum, workspace, sign: int = 1,
            dev_sel_idx=None, dev_sel_count=None, dev_err_count=None, stream=None):
    _check(load().gbfg_deposit(C.byref(grid), _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _offsets(offsets),
                               len(offsets) - 1, _ptr(dev_sel_idx), _ptr(dev_sel_count), sign, _ptr(dev_spectrum),
                               _ptr(dev_err_count), _ptr(workspace), workspace.numel() * workspace.element_size(),
                               _stream(stream)))


def running_median_workspace_bytes(n_bins: int, n_cat: int, window: int) -> int:
    return load().gbfg_running_median_workspace_bytes(n_bins, n_cat, window)


def running_median(dev_spectrum, n_bins: int, n_cat: int, window: int, dev_median_out, workspace=None, stream=None):
    """workspace: a device tensor of >= running_median_workspace_bytes(...) bytes; None: one is taken from torch."""
    if workspace is None:
        import torch
        workspace = torch.empty(max(running_median_workspace_bytes(n_bins, n_cat, window), 256), dtype=torch.uint8,
                                device=dev_spectrum.device)
    _check(load().gbfg_running_median(_ptr(dev_spectrum), n_bins, n_cat, window, _ptr(dev_median_out), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream(stream)))


STATIC_SCRATCH_BYTES = 1 << 20                       # GBFG_STATIC_SCRATCH_BYTES
STATIC_MAX_TILES = (STATIC_SCRATCH_BYTES - 256) // 16  # GBFG_STATIC_MAX_TILES


def running_median_static(dev_spectrum, n_bins: int, n_cat: int, window: int, dev_median_out, stream=None):
    """gbfg_running_median_static: no workspace, no allocation (the scratch is a static array in the library's device
    image); GbfgError(-6) beyond STATIC_MAX_TILES tiles.  Calls that overlap on the GPU race on the shared array."""
    _check(load().gbfg_running_median_static(_ptr(dev_spectrum), n_bins, n_cat, window, _ptr(dev_median_out),
                                             _stream(stream)))


def running_mean(dev_spectrum, n_bins: int, n_cat: int, window: int, dev_sum_out, dev_s_instr=None,
                 scale_log2: int = -140, dev_psd=None, stream=None):
    _check(load().gbfg_running_mean(_ptr(dev_spectrum), n_bins, n_cat, window, _ptr(dev_sum_out), _ptr(dev_s_instr),
                                    scale_log2, _ptr(dev_psd), _stream(stream)))


def coarse_grain(dev_psd, n_bins: int, n_cat: int, dev_edges, n_coarse: int, f_min: float, t_obs: float, dev_S,
                 dev_f=None, dev_hc=None, stream=None):
    _check(load().gbfg_coarse_grain(_ptr(dev_psd), n_bins, n_cat, _ptr(dev_edges), n_coarse, f_min, t_obs, _ptr(dev_S),
                                    _ptr(dev_f), _ptr(dev_hc), _stream(stream)))


def psd(dev_median, dev_s_instr, n_bins: int, n_cat: int, median_norm: float, scale_log2: int, dev_psd, stream=None):
    _check(load().gbfg_psd(_ptr(dev_median), _ptr(dev_s_instr), n_bins, n_cat, median_norm, scale_log2,
                           _ptr(dev_psd), _stream(stream)))


def snr_select(grid: Grid, dev_A, dev_f, dev_fdot, offsets, dev_psd, rho_th: float, dev_resolved, dev_sel_idx,
               dev_sel_count, workspace, dev_rho2_out=None, dev_near_count=None, stream=None):
    _check(load().gbfg_snr_select(C.byref(grid), _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _offsets(offsets),
                                  len(offsets) - 1, _ptr(dev_psd), rho_th, _ptr(dev_resolved), _ptr(dev_rho2_out),
                                  _ptr(dev_sel_idx), _ptr(dev_sel_count), _ptr(dev_near_count), _ptr(workspace),
                                  workspace.numel() * workspace.element_size(), _stream(stream)))


def subtract_until_converged(grid: Grid, dev_A, dev_f, dev_fdot, offsets, dev_s_instr, params: IterParams,
                             dev_spectrum, dev_median, dev_psd, dev_resolved, workspace, stream=None):
    n_cat = len(offsets) - 1
    res = (IterResult * n_cat)()
    _check(load().gbfg_subtract_until_converged(
        C.byref(grid), _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _offsets(offsets), n_cat, _ptr(dev_s_instr),
        C.byref(params), _ptr(dev_spectrum), _ptr(dev_median), _ptr(dev_psd), _ptr(dev_resolved), res,
        _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))
    return list(res)


def _cat_ids(cat_ids, n_cat: int):
    if cat_ids is None:
        return None
    if len(cat_ids) != n_cat:
        raise ValueError("cat_ids must name every catalog of the call")
    return (C.c_uint32 * n_cat)(*[int(c) for c in cat_ids])


def simulate(grid: Grid, pops, offsets, seed: int, dev_s_instr, params: IterParams, dev_A, dev_f, dev_fdot,
             dev_total, dev_spectrum, dev_median, dev_psd, dev_resolved, workspace, dev_err_count=None, stream=None,
             cat_ids=None):
    n_cat = len(offsets) - 1
    res = (IterResult * n_cat)()
    _check(load().gbfg_simulate(
        C.byref(grid), _pops(pops), _offsets(offsets), n_cat, seed, _cat_ids(cat_ids, n_cat), _ptr(dev_s_instr), C.byref(params),
        _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _ptr(dev_total), _ptr(dev_spectrum), _ptr(dev_median),
        _ptr(dev_psd), _ptr(dev_resolved), _ptr(dev_err_count), res, _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream)))
    return list(res)


def simulate_paper(grid: Grid, pops, offsets, seed: int, dev_s_instr, params: IterParams, dev_A, dev_f, dev_fdot,
                   dev_total, dev_spectrum, dev_median, dev_psd, dev_resolved, workspace, dev_edges=None, n_coarse: int = 0,
                   dev_S_coarse=None, dev_f_coarse=None, dev_hc=None, dev_err_count=None, stream=None, cat_ids=None):
    n_cat = len(offsets) - 1
    res = (IterResult * n_cat)()
    arr = (PopPaper * len(pops))()
    for i, p in enumerate(pops):
        arr[i] = p if isinstance(p, PopPaper) else make_pop_paper(p)
    _check(load().gbfg_simulate_paper(
        C.byref(grid), arr, _offsets(offsets), n_cat, seed, _cat_ids(cat_ids, n_cat), _ptr(dev_s_instr), C.byref(params),
        _ptr(dev_A), _ptr(dev_f), _ptr(dev_fdot), _ptr(dev_total), _ptr(dev_spectrum), _ptr(dev_median), _ptr(dev_psd),
        _ptr(dev_resolved), _ptr(dev_err_count), res, _ptr(dev_edges), n_coarse, _ptr(dev_S_coarse), _ptr(dev_f_coarse),
        _ptr(dev_hc), _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))
    return list(res)


def simulate_host(grid: Grid, pops, offsets, seed: int, host_s_instr, params: IterParams, host_psd,
                  host_resolved=None, cat_ids=None):
    n_cat = len(offsets) - 1
    res = (IterResult * n_cat)()
    _check(load().gbfg_simulate_host(C.byref(grid), _pops(pops), _offsets(offsets), n_cat, seed, _cat_ids(cat_ids, n_cat),
                                     _ptr(host_s_instr),
                                     C.byref(params), _ptr(host_psd), _ptr(host_resolved), res))
    return list(res)
