"""ctypes view of the oracle (oracle/gbfg_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2602_18560_b200 and the product imports
nothing from here.  Arrays are numpy, host memory; every function is a thin marshalling layer
over the C function of the same name (see the C file for the passages each one follows).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gbfg_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

GCC_FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-std=c11", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (IEEE arithmetic, no contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *GCC_FLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


class Grid(C.Structure):
    _fields_ = [("f_min", C.c_double), ("f_max", C.c_double), ("t_obs", C.c_double),
                ("n_bins", C.c_int64), ("scale_log2", C.c_int32)]


class Pop(C.Structure):
    _fields_ = [("slope", C.c_double), ("logA_offset", C.c_double), ("logA_sigma", C.c_double),
                ("logMc_mean", C.c_double), ("logMc_sigma", C.c_double), ("n_src", C.c_int64)]


class PopPaper(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("reserved", C.c_uint32), ("alpha_pl", C.c_double),
                ("alpha_gamma", C.c_double), ("beta_gamma", C.c_double), ("mu_gamma", C.c_double),
                ("mu", C.c_double), ("sigma", C.c_double), ("rho", C.c_double), ("n_src", C.c_int64)]


class IterResult(C.Structure):
    _fields_ = [("n_iter", C.c_int32), ("converged", C.c_int32), ("n_resolved", C.c_int64),
                ("n_near_threshold", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        dp, ip, up = C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_uint8)
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_u01.restype = C.c_double
        L.orc_u01.argtypes = [C.c_uint32, C.c_uint32]
        for name in ("orc_log", "orc_exp10", "orc_robson_sn"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double]
        for name in ("orc_sincos2pi", "orc_sincos"):
            getattr(L, name).argtypes = [C.c_double, dp, dp]
        L.orc_n_bins.restype = C.c_int64
        L.orc_n_bins.argtypes = [C.c_double] * 3
        L.orc_sample_catalog.argtypes = [C.POINTER(Grid), C.POINTER(Pop), C.c_uint32, C.c_uint64,
                                         C.c_int64, C.c_int64, dp, dp, dp]
        L.orc_instrument_noise.argtypes = [C.POINTER(Grid), dp]
        L.orc_source_bins.argtypes = [C.POINTER(Grid), C.c_double, C.c_double, C.c_double,
                                      ip, ip, ip, dp, ip]
        L.orc_deposit.restype = C.c_int64
        L.orc_deposit.argtypes = [C.POINTER(Grid), dp, dp, dp, C.c_int64, ip, C.c_int64, C.c_int32, ip]
        L.orc_running_median_sort.argtypes = [ip, C.c_int64, C.c_int32, C.c_int64, C.c_int64, ip]
        L.orc_running_median.argtypes = [ip, C.c_int64, C.c_int32, ip]
        L.orc_psd.argtypes = [ip, dp, C.c_int64, C.c_double, C.c_int32, dp]
        L.orc_rho2.restype = C.c_double
        L.orc_rho2.argtypes = [C.POINTER(Grid), C.c_double, C.c_double, C.c_double, dp]
        L.orc_rho2_ld_as_double.restype = C.c_double
        L.orc_rho2_ld_as_double.argtypes = L.orc_rho2.argtypes
        L.orc_snr_select.restype = C.c_int64
        L.orc_snr_select.argtypes = [C.POINTER(Grid), dp, dp, dp, C.c_int64, dp, C.c_double, up, dp, ip, ip]
        L.orc_subtract_until_converged.argtypes = [
            C.POINTER(Grid), dp, dp, dp, C.c_int64, dp, C.c_int32, C.c_double, C.c_double, C.c_int32,
            ip, ip, dp, up, C.POINTER(IterResult), ip]
        L.orc_subtract_until_converged_est.argtypes = [
            C.POINTER(Grid), dp, dp, dp, C.c_int64, dp, C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_int32,
            ip, ip, dp, up, C.POINTER(IterResult), ip]
        L.orc_erfc_pos.restype = C.c_double
        L.orc_erfc_pos.argtypes = [C.c_double]
        L.orc_norm_tail.restype = C.c_double
        L.orc_norm_tail.argtypes = [C.c_double]
        L.orc_gamma_pq.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp, dp]
        L.orc_gamma_quantile.restype = C.c_double
        L.orc_gamma_quantile.argtypes = [C.c_double] * 4
        L.orc_sample_catalog_paper.argtypes = [C.POINTER(Grid), C.POINTER(PopPaper), C.c_uint32, C.c_uint64,
                                               C.c_int64, C.c_int64, dp, dp, dp]
        L.orc_aet_noise.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, dp]
        L.orc_instrument_noise_aet.argtypes = [C.POINTER(Grid), C.c_double, C.c_double, C.c_double, C.c_int, dp, dp, dp, dp]
        L.orc_subtract_until_converged_tol.argtypes = [
            C.POINTER(Grid), dp, dp, dp, C.c_int64, dp, C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_int32, C.c_double,
            ip, ip, dp, up, C.POINTER(IterResult), ip]
        L.orc_channel_sum_noise.argtypes = [dp, dp, C.c_int64, dp]
        L.orc_stage_seconds.argtypes = [C.POINTER(C.c_double), C.c_int]
        L.orc_running_sum_def.argtypes = [ip, C.c_int64, C.c_int32, C.c_int64, C.c_int64, ip]
        L.orc_running_sum.argtypes = [ip, C.c_int64, C.c_int32, ip]
        L.orc_psd_mean.argtypes = [ip, dp, C.c_int64, C.c_int32, C.c_int32, dp]
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _u(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def u01(w_lo: int, w_hi: int) -> float:
    return lib().orc_u01(w_lo, w_hi)


def log(x: float) -> float:
    return lib().orc_log(x)


def exp10(y: float) -> float:
    return lib().orc_exp10(y)


def sincos2pi(u: float):
    s, c = C.c_double(), C.c_double()
    lib().orc_sincos2pi(u, C.byref(s), C.byref(c))
    return s.value, c.value


def sincos(x: float):
    s, c = C.c_double(), C.c_double()
    lib().orc_sincos(x, C.byref(s), C.byref(c))
    return s.value, c.value


def robson_sn(f: float) -> float:
    return lib().orc_robson_sn(f)


def make_grid(f_min: float, f_max: float, t_obs: float, scale_log2: int = -140) -> Grid:
    n = lib().orc_n_bins(f_min, f_max, t_obs)
    return Grid(f_min, f_max, t_obs, n, scale_log2)


def make_pop(p) -> Pop:
    return Pop(p.slope, p.logA_offset, p.logA_sigma, p.logMc_mean, p.logMc_sigma, p.n_src)


def sample_catalog(grid: Grid, pop, cat_id: int, seed: int, i_begin: int = 0, i_end: int | None = None):
    pp = pop if isinstance(pop, Pop) else make_pop(pop)
    if i_end is None:
        i_end = pp.n_src
    n = i_end - i_begin
    A, f, fd = (np.empty(n, dtype=np.float64) for _ in range(3))
    lib().orc_sample_catalog(C.byref(grid), C.byref(pp), cat_id, seed, i_begin, i_end, _d(A), _d(f), _d(fd))
    return A, f, fd


def instrument_noise(grid: Grid) -> np.ndarray:
    s = np.empty(grid.n_bins, dtype=np.float64)
    lib().orc_instrument_noise(C.byref(grid), _d(s))
    return s


def source_bins(grid: Grid, A: float, f: float, fdot: float):
    """-> (status, k0, w, w_eff, p, q); status 0 ok, 1 domain, 2 range."""
    k0, w, we, q = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
    p = C.c_double()
    st = lib().orc_source_bins(C.byref(grid), A, f, fdot, C.byref(k0), C.byref(w), C.byref(we),
                               C.byref(p), C.byref(q))
    return st, k0.value, w.value, we.value, p.value, q.value


def deposit(grid: Grid, A, f, fdot, spectrum: np.ndarray, sel=None, sign: int = 1) -> int:
    A, f, fdot = _f64(A), _f64(f), _f64(fdot)
    assert spectrum.dtype == np.int64 and spectrum.flags.c_contiguous and spectrum.size == grid.n_bins
    if sel is None:
        return lib().orc_deposit(C.byref(grid), _d(A), _d(f), _d(fdot), A.size, None, 0, sign, _i(spectrum))
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    return lib().orc_deposit(C.byref(grid), _d(A), _d(f), _d(fdot), A.size, _i(sel), sel.size, sign, _i(spectrum))


def running_median_sort(x: np.ndarray, window: int, k_begin: int = 0, k_end: int | None = None) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.int64)
    if k_end is None:
        k_end = x.size
    out = np.empty(k_end - k_begin, dtype=np.int64)
    rc = lib().orc_running_median_sort(_i(x), x.size, window, k_begin, k_end, _i(out))
    if rc:
        raise ValueError("invalid window / size")
    return out


def running_median(x: np.ndarray, window: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.int64)
    out = np.empty_like(x)
    rc = lib().orc_running_median(_i(x), x.size, window, _i(out))
    if rc:
        raise ValueError("invalid window / size")
    return out


def erfc_pos(t: float) -> float:
    return lib().orc_erfc_pos(t)


def norm_tail(z: float) -> float:
    """Phi(z) for z <= 0, 1 - Phi(z) for z > 0."""
    return lib().orc_norm_tail(z)


def gamma_pq(a: float, x: float):
    """(P(a,x), Q(a,x)) regularized incomplete gamma functions."""
    import math
    P, Q, pref = C.c_double(), C.c_double(), C.c_double()
    lib().orc_gamma_pq(a, x, math.lgamma(a), C.byref(P), C.byref(Q), C.byref(pref))
    return P.value, Q.value


def gamma_quantile(a: float, z: float) -> float:
    """x with P(a, x) = Phi(z)."""
    import math
    return lib().orc_gamma_quantile(a, math.lgamma(a), math.lgamma(a + 1.0), z)


def make_pop_paper(p) -> PopPaper:
    return PopPaper(C.sizeof(PopPaper), 0, p.alpha_pl, p.alpha_gamma, p.beta_gamma, p.mu_gamma, p.mu, p.sigma, p.rho, p.n_src)


def sample_catalog_paper(grid: Grid, pop, cat_id: int, seed: int, i_begin: int = 0, i_end: int | None = None):
    """The paper's population sampler (Table I, eqs. 7-9, Gaussian copula): -> (A, f, fdot)."""
    pp = pop if isinstance(pop, PopPaper) else make_pop_paper(pop)
    if i_end is None:
        i_end = pp.n_src
    n = i_end - i_begin
    A, f, fd = (np.empty(n, dtype=np.float64) for _ in range(3))
    lib().orc_sample_catalog_paper(C.byref(grid), C.byref(pp), cat_id, seed, i_begin, i_end, _d(A), _d(f), _d(fd))
    return A, f, fd


def aet_noise(f: float, P: float = 15.0, A: float = 3.0, L: float = 2.5e9, tdi2: bool = True):
    """(S_AA, S_TT, S_AA / R_AA, S_TT / R_TT) at frequency f: eqs. (C1)-(C5), (B2)-(B5)."""
    out = (C.c_double * 4)()
    lib().orc_aet_noise(f, P, A, L, 1 if tdi2 else 0, out)
    return tuple(out)


def instrument_noise_aet(grid: Grid, P: float = 15.0, A: float = 3.0, L: float = 2.5e9, tdi2: bool = True):
    outs = [np.empty(grid.n_bins, dtype=np.float64) for _ in range(4)]
    lib().orc_instrument_noise_aet(C.byref(grid), P, A, L, 1 if tdi2 else 0, *[_d(o) for o in outs])
    return tuple(outs)


def channel_sum_noise(sh_aa, sh_tt) -> np.ndarray:
    """S_sum = 1 / (2 / S_h^AA + 1 / S_h^TT): the noise curve of the SNR summed over A, E, T (eq. 11; R14)."""
    sh_aa, sh_tt = _f64(sh_aa), _f64(sh_tt)
    out = np.empty_like(sh_aa)
    lib().orc_channel_sum_noise(_d(sh_aa), _d(sh_tt), sh_aa.size, _d(out))
    return out


def running_sum_def(x: np.ndarray, window: int, k_begin: int = 0, k_end: int | None = None) -> np.ndarray:
    """Window sums of the running-mean estimator (eq. D1), the definition: one loop per output."""
    x = np.ascontiguousarray(x, dtype=np.int64)
    if k_end is None:
        k_end = x.size
    out = np.empty(k_end - k_begin, dtype=np.int64)
    if lib().orc_running_sum_def(_i(x), x.size, window, k_begin, k_end, _i(out)):
        raise ValueError("invalid window / size")
    return out


def running_sum(x: np.ndarray, window: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.int64)
    out = np.empty_like(x)
    if lib().orc_running_sum(_i(x), x.size, window, _i(out)):
        raise ValueError("invalid window / size")
    return out


def psd_from_sum(wsum: np.ndarray, s_instr: np.ndarray, window: int, scale_log2: int) -> np.ndarray:
    wsum = np.ascontiguousarray(wsum, dtype=np.int64)
    s_instr = _f64(s_instr)
    out = np.empty(wsum.size, dtype=np.float64)
    lib().orc_psd_mean(_i(wsum), _d(s_instr), wsum.size, window, scale_log2, _d(out))
    return out


def psd_from_median(med: np.ndarray, s_instr: np.ndarray, median_norm: float, scale_log2: int) -> np.ndarray:
    med = np.ascontiguousarray(med, dtype=np.int64)
    s_instr = _f64(s_instr)
    out = np.empty(med.size, dtype=np.float64)
    lib().orc_psd(_i(med), _d(s_instr), med.size, median_norm, scale_log2, _d(out))
    return out


def rho2(grid: Grid, A: float, f: float, fdot: float, psd: np.ndarray, long_double: bool = False) -> float:
    psd = _f64(psd)
    fn = lib().orc_rho2_ld_as_double if long_double else lib().orc_rho2
    return fn(C.byref(grid), A, f, fdot, _d(psd))


def snr_select(grid: Grid, A, f, fdot, psd, rho_th: float, resolved: np.ndarray):
    """-> (sel_idx ascending, rho2 for every tested source (NaN where untested), n_near). Updates resolved."""
    A, f, fdot, psd = _f64(A), _f64(f), _f64(fdot), _f64(psd)
    assert resolved.dtype == np.uint8 and resolved.flags.c_contiguous
    n = A.size
    r2 = np.full(n, np.nan)
    sel = np.empty(max(n, 1), dtype=np.int64)
    near = C.c_int64()
    m = lib().orc_snr_select(C.byref(grid), _d(A), _d(f), _d(fdot), n, _d(psd), rho_th, _u(resolved),
                             _d(r2), _i(sel), C.byref(near))
    return sel[:m].copy(), r2, near.value


def subtract_until_converged(grid: Grid, A, f, fdot, s_instr, window: int, median_norm: float,
                             rho_th: float, max_iter: int, spectrum: np.ndarray,
                             resolved: np.ndarray | None = None, estimator: int = 0, psd_rtol: float = 0.0):
    """Runs the loop in place on `spectrum` (total -> residual).
    -> dict(median, psd, resolved, n_iter, converged, n_resolved, n_near_threshold, n_new_per_iter)"""
    A, f, fdot, s_instr = _f64(A), _f64(f), _f64(fdot), _f64(s_instr)
    assert spectrum.dtype == np.int64 and spectrum.flags.c_contiguous
    n = A.size
    if resolved is None:
        resolved = np.zeros(n, dtype=np.uint8)
    med = np.empty(grid.n_bins, dtype=np.int64)
    psd = np.empty(grid.n_bins, dtype=np.float64)
    res = IterResult()
    trace = np.zeros(max(max_iter, 1), dtype=np.int64)
    rc = lib().orc_subtract_until_converged_tol(C.byref(grid), _d(A), _d(f), _d(fdot), n, _d(s_instr), window,
                                                median_norm, rho_th, max_iter, estimator, psd_rtol, _i(spectrum),
                                                _i(med), _d(psd), _u(resolved), C.byref(res), _i(trace))
    if rc:
        raise ValueError("invalid window / size")
    return dict(median=med, psd=psd, resolved=resolved, n_iter=res.n_iter, converged=res.converged,
                n_resolved=res.n_resolved, n_near_threshold=res.n_near_threshold,
                n_new_per_iter=trace[:max_iter])


def stage_seconds(reset: bool = True):
    """Seconds the calling thread's loop calls spent in (estimator passes, SNR passes, subtractions) since the last reset."""
    out = (C.c_double * 3)()
    lib().orc_stage_seconds(out, 1 if reset else 0)
    return tuple(out)


def simulate(w, cat: int = 0, n_src: int | None = None, estimator: int = 0, psd_rtol: float = 0.0, cat_id: int | None = None):
    """Whole path for catalog `cat` of a gbfg_workloads.Workload: sample -> deposit -> loop.  `stage_s` of the result:
    wall-clock seconds per stage (measurement only).  cat_id: Philox catalog id (default: cat)."""
    import time
    grid = make_grid(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    pop = make_pop(w.pops[cat])
    if n_src is not None:
        pop.n_src = n_src
    t0 = time.perf_counter()
    A, f, fd = sample_catalog(grid, pop, cat if cat_id is None else cat_id, w.seed)
    t1 = time.perf_counter()
    s_instr = instrument_noise(grid)
    t2 = time.perf_counter()
    spec = np.zeros(grid.n_bins, dtype=np.int64)
    rejected = deposit(grid, A, f, fd, spec)
    t3 = time.perf_counter()
    total = spec.copy()
    stage_seconds(reset=True)
    out = subtract_until_converged(grid, A, f, fd, s_instr, w.window, w.median_norm, w.rho_th, w.max_iter, spec,
                                   estimator=estimator, psd_rtol=psd_rtol)
    est_s, snr_s, sub_s = stage_seconds(reset=True)
    out.update(A=A, f=f, fdot=fd, s_instr=s_instr, total=total, residual=spec, rejected=rejected, grid=grid,
               stage_s={"sample": t1 - t0, "noise": t2 - t1, "deposit": t3 - t2, "estimator_passes": est_s,
                        "snr_passes": snr_s, "subtract": sub_s})
    return out


# ---------------------------------------------------------------------------------------------
# Coarse-graining of the PSD, eqs. (13)-(14) PAPER.md:186-199, and the characteristic strain, eq. (B1)
# PAPER.md:465 (R10).  Plain Python / numpy: math.fsum is the exactly rounded sum.
# ---------------------------------------------------------------------------------------------
def coarse_grain(psd: np.ndarray, edges, f_min: float, t_obs: float):
    """edges: n_coarse+1 non-decreasing fine-bin indices; coarse bin k holds the fine bins
    edges[k] <= i < edges[k+1], whose frequencies are the bin centres f_i = f_min + (i + 1/2)/T.
    -> (S[k] = (1/N_k) sum S_n(f_i)  (eq. 13),  f[k] = (1/N_k) sum f_i  (eq. 14),  hc[k] = sqrt(f[k] S[k])  (eq. B1));
    an empty coarse bin gives NaN in all three."""
    import math
    psd = _f64(psd)
    n_coarse = len(edges) - 1
    S = np.full(n_coarse, np.nan)
    fk = np.full(n_coarse, np.nan)
    hc = np.full(n_coarse, np.nan)
    for k in range(n_coarse):
        i0, i1 = int(edges[k]), int(edges[k + 1])
        nk = i1 - i0
        if nk <= 0:
            continue
        S[k] = math.fsum(psd[i0:i1].tolist()) / nk
        fk[k] = math.fsum(f_min + (i + 0.5) / t_obs for i in range(i0, i1)) / nk
        hc[k] = math.sqrt(fk[k] * S[k])
    return S, fk, hc
