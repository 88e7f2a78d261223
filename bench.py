#!/usr/bin/env python
"""bench.py — catalog -> converged foreground on B200 (BASELINE.json:metric, configs[3]).

One "step" = one pass of the whole hot path (sample -> deposit -> [median+PSD ->
SNR+select -> subtract] until converged or capped) over one 1e7-source, 4-yr synthetic catalog,
through the C ABI (gbfg_simulate).  Prints ONE JSON line (see the task contract):
  value      sources/s with every buffer resident in HBM (the catalog is drawn on the device by stage i)
  e2e        the same through gbfg_simulate_host: host buffers, H2D/D2H inside the timed region
  roofline   the dominant kernel's algorithmic bytes / CUDA-event time against MEASURED_PEAKS.json
  kernels    the same for every kernel class (events recorded on the launching stream, live)
  cpu_baseline  the oracle, as it stands, on one host core, on the SAME workload in full (config 3: about half a
                minute), with the seconds it spends per stage; `--cpu-config4` adds the 64 catalogs of configs[4]
                over all host cores (one oracle process per catalog)

`--impl reference` times the oracle alone (rank 0 only) on the same full workload and prints its own line; it
honours --steps up to a time budget (REFERENCE_BUDGET_S), with a floor of one step, and says how many it ran.
N > 1 (torchrun): every rank runs its own independent catalog (seed + rank); no data-path
collective; value = all ranks' sources / max-over-ranks time; scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import gbfg_workloads as wl

METRIC = "catalog_to_foreground_throughput"
UNIT = "sources/s"
REFERENCE_BUDGET_S = 150.0          # the reference arm stops taking further steps once this much oracle time is spent


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock, power and throttle reasons while the GPU is under the benchmark's load: an NVML polling thread
    (one sample every 2 ms, so that a 30 ms timed region is seen a dozen times); `nvidia-smi -lms` when the
    NVML binding is missing."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
    PERIOD_S = 0.002

    def __init__(self, index: int, uuid=None):
        self.index = index
        self.uuid = uuid
        self.proc = None
        self.thread = None
        self.stop_flag = False
        self.sm, self.pw, self.reasons, self.mx = [], [], set(), None

    def _nvml_loop(self, nv, h):
        masks = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self.stop_flag:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                self.pw.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for name, m in masks.items():
                    if r & m:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.PERIOD_S)

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            h = None
            if self.uuid:
                try:
                    h = nv.nvmlDeviceGetHandleByUUID(self.uuid if str(self.uuid).startswith("GPU-") else "GPU-" + str(self.uuid))
                except Exception:
                    h = None
            if h is None:
                h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._nvml_loop, args=(nv, h), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def mark(self):
        """Forget what was sampled so far (called where the timed region starts)."""
        if self.thread is not None:
            self.sm, self.pw = [], []

    def stop(self) -> dict:
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            if not self.sm:
                return {"sm_mhz": None, "sm_max_mhz": self.mx, "reasons": ["no samples"]}
            return {"sm_mhz": float(np.median(self.sm)), "sm_min_mhz": float(min(self.sm)), "sm_max_mhz": self.mx,
                    "power_w_max": float(max(self.pw)), "samples": len(self.sm), "source": "nvml, 2 ms period",
                    "reasons": sorted(self.reasons)}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "source": "nvidia-smi -lms 20", "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------- reference arm
def oracle_full_run(w: wl.Workload):
    """The oracle, as it stands, on workload w's catalog 0 in full, whole path, one thread."""
    import oracle
    oracle.build()
    oracle.lib()
    t0 = time.perf_counter()
    out = oracle.simulate(w, cat=0)
    dt = time.perf_counter() - t0
    return dt, out


def oracle_sample_text(w: wl.Workload, out) -> str:
    return (f"{w.name} in full: all {w.n_src_total} sources of the seeded catalog on the full grid (window {w.window}, "
            f"cap {w.max_iter}), whole path sample->deposit->loop, {int(out['n_iter'])} iterations, "
            f"{int(out['n_resolved'])} resolved, 1 thread")


def run_reference(args, w: wl.Workload):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    # the oracle has no warm-up state: warm-up steps are not run (half a minute each)
    times, out = [], None
    spent = 0.0
    for _ in range(max(1, args.steps)):
        dt, out = oracle_full_run(w)
        times.append(dt)
        spent += dt
        if spent + dt > REFERENCE_BUDGET_S:
            break
    t = float(np.mean(times))
    n = w.n_src_total
    val = n / t
    sample = oracle_sample_text(w, out) + f"; {len(times)} of the {args.steps} requested steps run (time budget {REFERENCE_BUDGET_S:.0f} s)"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "steps_run": len(times), "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64+i64", "data": "synthetic",
        "config": {"workload": w.name, "n_src": n, "n_cat": w.n_cat, "window": w.window, "rho_th": w.rho_th,
                   "max_iter": w.max_iter, "t_obs_s": w.t_obs, "band_hz": [w.f_min, w.f_max], "seed": w.seed,
                   "n_iter": int(out["n_iter"]), "converged": int(out["converged"]), "n_resolved": int(out["n_resolved"])},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "seconds": t, "stage_seconds": out["stage_s"]},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def oracle_config4_leg():
    """configs[4] through the oracle: 64 independent single-threaded runs over the host cores."""
    from oracle import pool
    w4 = wl.config(4)
    out = pool.simulate_many(w4, range(w4.n_cat))
    core_s = sum(r["seconds"] for r in out["results"].values())
    return {"workload": w4.name, "n_src": w4.n_src_total, "n_cat": w4.n_cat, "cores": out["n_proc"],
            "host_cores": pool.host_cores(), "wall_seconds": out["wall_seconds"], "core_seconds": core_s,
            "value": w4.n_src_total / out["wall_seconds"], "unit": UNIT, "kind": "oracle",
            "sample": "all 64 catalogs in full, one oracle process per catalog"}


# ------------------------------------------------------------------------------------ GPU arm
def algorithmic_bytes(w: wl.Workload, n_bins: int, res, prof) -> dict:
    """Algorithmic bytes of ONE step per kernel class: what the method itself
    must move for the work that was actually done, not what the implementation happens to move.  The library
    counts the running-median outputs it computed and the SNR tests it evaluated (gbfg_iter_result), so
    skipped (clean) work is not counted as moved bytes."""
    n = w.n_src_total
    n_iter = res.n_iter
    trace = [int(res.n_new_per_iter[i]) for i in range(min(n_iter, 64))]
    n_sub = sum(trace)
    n_scan = prof["scan"][0]
    return {
        "sample": 24 * n,                                   # 24 B written per source
        "deposit": 24 * n,                                  # catalog read once (the loop subtracts inside the SNR test)
        "scan": 16 * n_bins * n_scan,                       # spectrum read + written per range-update pass (upper bound: untouched tiles are skipped)
        "median": 32 * int(res.n_median_outputs),           # per output: spectrum in, median out, s_instr in, PSD out
        "inv_blocks": 8 * int(res.n_median_outputs) + 8 * n_bins,   # PSD read where it changed (+ s_instr once)
        "snr": 25 * n + 25 * int(res.n_snr_tests),          # candidate build reads the catalog once; 24 B + flag per test
        "aux": 4 * ((n_bins + 255) // 256) * prof["aux"][0],   # plan: one stamp per 256-bin block
        "_counts": {"n_iter": n_iter, "n_sub": n_sub, "median_outputs": int(res.n_median_outputs),
                    "snr_tests": int(res.n_snr_tests)},
    }


def median_kernel_counters():
    """dram bytes and warp instructions of the running-median kernel per output it recomputes, as the committed
    `ncu --set full` summary states them (profiles/r02_ncu_full.md, lines `median_...: value`); nothing is hard-coded here,
    so a stale figure can only come from a stale summary, whose commit is reported next to it."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_full.md")
    out = {"source": "profiles/r02_ncu_full.md"}
    try:
        with open(path) as fh:
            for line in fh:
                for key in ("median_dram_bytes_per_output", "median_warp_instr_per_output", "median_capture_commit"):
                    if line.startswith(key + ":"):
                        v = line.split(":", 1)[1].strip()
                        out[key] = v if key.endswith("commit") else float(v)
    except OSError:
        pass
    return out


def run_gpu(args, w: wl.Workload):
    import torch
    import paper_2602_18560_b200 as gb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libgbfg has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gb.load()
    dev = torch.device("cuda", local)
    w = wl.replace(w, seed=w.seed + 1000 * rank)           # independent catalogs, one per rank
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb, nc = w.n_src_total, g.n_bins, w.n_cat
    off = w.offsets()

    s_instr = torch.empty(nb, dtype=torch.float64, device=dev)
    gb.instrument_noise(g, s_instr)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device=dev) for _ in range(3))
    spec, med = (torch.empty((nc, nb), dtype=torch.int64, device=dev) for _ in range(2))
    psd = torch.empty((nc, nb), dtype=torch.float64, device=dev)
    resolved = torch.empty(n, dtype=torch.uint8, device=dev)
    ws = torch.empty(gb.workspace_bytes(g, n, nc), dtype=torch.uint8, device=dev)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, args.flags)

    def step():
        return gb.simulate(g, w.pops, off, w.seed, s_instr, params, A, f, fd, None, spec, med, psd, resolved, ws)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    uuid = getattr(torch.cuda.get_device_properties(dev), "uuid", None)
    clocks = ClockSampler(local, uuid)  # runs from the warm-up on; the samples kept are those of the two timed regions
    clocks.start()
    for _ in range(max(args.warmup, 0)):
        step()
    barrier()

    # ---- device-resident timing (value): K steps between two CUDA events, clocks sampled meanwhile
    launches0 = gb.kernel_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clocks.mark()
    e0.record()
    for _ in range(args.steps):
        res = step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = gb.kernel_launch_count() - launches0
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * n / (ms_step * 1e-3)

    # ---- the same K steps again with every kernel launch bracketed by a pair of CUDA events on its own stream
    # (gbfg_profile_*): the per-kernel times of the roofline.  The event pairs cost about 10 % of the step, which is
    # why the headline region above runs without them.
    gb.profile_enable(True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_step_prof = e0.elapsed_time(e1) / args.steps
    prof = gb.profile_read()
    gb.profile_enable(False)
    clk = clocks.stop()

    # ---- end to end through the host-buffer entry point (gbfg_simulate_host): what goes in every step is the step's
    # input, the population parameters Lambda and the seed (the instrument-noise curve is a function of the grid alone and
    # is made on the device: host_s_instr = NULL); what comes back every step is the PSD and the resolved flags, into
    # pinned host memory.  The same call with the 30 MB curve uploaded every step is timed next to it.
    h_s = s_instr.cpu().pin_memory()
    h_psd = torch.empty((nc, nb), dtype=torch.float64).pin_memory()
    h_res = torch.empty(n, dtype=torch.uint8).pin_memory()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))

    def timed_host(curve):
        gb.simulate_host(g, w.pops, off, w.seed, curve, params, h_psd.numpy(), h_res.numpy())
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            gb.simulate_host(g, w.pops, off, w.seed, curve, params, h_psd.numpy(), h_res.numpy())
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / e2e_steps
        if dist is not None:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        return dt

    e2e_upload_s = timed_host(h_s.numpy())
    e2e_s = timed_host(None)
    same_psd = bool(torch.equal(h_psd.view(torch.int64), psd.cpu().view(torch.int64)))
    same_res = bool(torch.equal(h_res, resolved.cpu()))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of every kernel class, and of the dominant one
    peak, peak_src = measured_peaks()
    r0 = res[0]
    ab = algorithmic_bytes(w, nb, r0, {k: (v[0] // args.steps, v[1], v[2]) for k, v in prof.items()})
    kernels = {}
    for k, (cnt, tot, mx) in prof.items():
        if cnt == 0:
            continue
        per_step_ms = tot / args.steps
        gbs = ab.get(k, 0) / (per_step_ms * 1e-3) / 1e9 if per_step_ms > 0 else 0.0
        kernels[k] = {"launches_per_step": cnt / args.steps, "ms_per_step": per_step_ms, "avg_launch_ms": tot / cnt,
                      "max_launch_ms": mx, "algorithmic_bytes_per_step": ab.get(k, 0), "achieved_gbs": gbs,
                      "frac_of_hbm": gbs / peak, "share_of_step": per_step_ms / ms_step_prof}
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_step"])
    kd = kernels[dom]
    bytes_per_launch = kd["algorithmic_bytes_per_step"] / kd["launches_per_step"]
    traffic = args.traffic
    mk = median_kernel_counters()
    if traffic is None and dom == "median" and "median_dram_bytes_per_output" in mk:
        # per launch like `achieved`: an average launch recomputes bytes_per_launch / 32 outputs
        traffic = mk["median_dram_bytes_per_output"] * bytes_per_launch / 32.0
    roofline = {"kernel": dom, "bound": "hbm", "achieved": bytes_per_launch / (kd["avg_launch_ms"] * 1e-3) / 1e9,
                "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": bytes_per_launch / (kd["avg_launch_ms"] * 1e-3) / 1e9 / peak,
                "algorithmic_bytes_per_launch": bytes_per_launch, "avg_launch_ms": kd["avg_launch_ms"],
                "traffic": traffic, "traffic_source": mk if dom == "median" else None}

    # What actually bounds the running median is instruction issue, not HBM: the same launches
    # against the issue rate of the part, 4 warp instructions per SM and clock (B200_PROFILING.md: 148 SMs x 4 schedulers)
    roofline_issue = None
    if dom == "median" and "median_warp_instr_per_output" in mk:
        ipo = mk["median_warp_instr_per_output"]
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        mhz = (clk or {}).get("sm_mhz") or (clk or {}).get("sm_max_mhz") or 1965.0
        peak_issue = sms * 4 * mhz * 1e6 / 1e9                      # G warp-instructions / s
        ach = ipo * (bytes_per_launch / 32.0) / (kd["avg_launch_ms"] * 1e-3) / 1e9
        roofline_issue = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": peak_issue,
                          "unit": "G warp-instr/s", "frac": ach / peak_issue,
                          "peak_source": f"{sms} SMs x 4 schedulers x {mhz:.0f} MHz (sm clock under load)",
                          "instr_per_output": ipo}

    # ---- the oracle on one host core, the same workload in full (a reported baseline, not the target)
    cpu = None
    if not args.no_cpu_baseline:
        dt, out = oracle_full_run(wl.replace(w, seed=w.seed))
        same = (int(out["n_iter"]), int(out["n_resolved"])) == (int(r0.n_iter), int(r0.n_resolved))
        cpu = {"value": n / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "stage_seconds": out["stage_s"], "host_cores": os.cpu_count(),
               "same_outcome_as_gpu": same, "sample": oracle_sample_text(w, out)}
        if args.cpu_config4:
            cpu["config4"] = oracle_config4_leg()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64+i64", "data": "synthetic",
        "config": {"workload": w.name, "n_src": n, "n_cat": nc, "n_bins": nb, "window": w.window, "rho_th": w.rho_th,
                   "max_iter": w.max_iter, "t_obs_s": w.t_obs, "band_hz": [w.f_min, w.f_max], "seed": w.seed,
                   "n_iter": r0.n_iter, "converged": r0.converged, "n_resolved": r0.n_resolved,
                   "n_near_threshold": r0.n_near_threshold, "flags": args.flags,
                   "l2": "inputs larger than L2: every step redraws and re-reads the 240 MB catalog (126 MB L2)",
                   "wall_time_s": ms_step * 1e-3},
        "ms_per_step_with_kernel_events": ms_step_prof,
        "e2e": {"value": world * n / e2e_s, "unit": UNIT, "ms_per_step": 1e3 * e2e_s, "steps": e2e_steps,
                "h2d_bytes_per_step": 56 * nc + 8 * (nc + 1) + 64, "d2h_bytes_per_step": 8 * nc * nb + n,
                "inputs": "population parameters, offsets, seed, loop parameters (host structs); noise curve made on the device",
                "outputs": "PSD [n_cat][n_bins] f64 + resolved flags [N] u8 into pinned host memory",
                "psd_equal_to_device_run": same_psd, "resolved_equal_to_device_run": same_res,
                "ms_per_step_with_the_noise_curve_uploaded": 1e3 * e2e_upload_s, "h2d_bytes_with_the_curve": 8 * nb},
        "gpu_launches": int(launches),
        "clocks": clk,
        "roofline": roofline,
        "roofline_issue": roofline_issue,
        "kernels": kernels,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_stage_bench(args, w: wl.Workload):
    """`--stage-bench`: the two PSD estimators alone, one full pass over the workload's grid per launch (stage calls
    gbfg_running_median / gbfg_running_mean on the deposited spectrum of the workload's catalog), CUDA events on the
    launching stream, 256 MB written between repetitions to flush the 126 MB L2.  Prints one JSON line."""
    import torch
    import paper_2602_18560_b200 as gb
    torch.cuda.set_device(0)
    gb.load()
    dev = torch.device("cuda", 0)
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb = w.n_src_total, g.n_bins
    A, f, fd = (torch.empty(n, dtype=torch.float64, device=dev) for _ in range(3))
    gb.sample_catalog(g, w.pops, w.offsets(), w.seed, A, f, fd)
    spec = torch.zeros(nb, dtype=torch.int64, device=dev)
    ws = torch.empty(gb.workspace_bytes(g, n, 1), dtype=torch.uint8, device=dev)
    gb.deposit(g, A, f, fd, w.offsets(), spec, ws)
    s_instr = torch.empty(nb, dtype=torch.float64, device=dev)
    gb.instrument_noise(g, s_instr)
    out = torch.empty(nb, dtype=torch.int64, device=dev)
    psd = torch.empty(nb, dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    peak, peak_src = measured_peaks()
    res = {}
    calls = {"running_median": (lambda: gb.running_median(spec, nb, 1, w.window, out, ws), 16),
             "running_mean": (lambda: gb.running_mean(spec, nb, 1, w.window, out, s_instr, w.scale_log2, psd), 32)}
    for name, (fn, bytes_per_bin) in calls.items():
        for _ in range(3):
            fn()
        ts = []
        for _ in range(max(args.steps, 5)):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        t = float(np.median(ts))
        gbs = bytes_per_bin * nb / (t * 1e-3) / 1e9
        res[name] = {"ms": t, "algorithmic_bytes": bytes_per_bin * nb, "achieved_gbs": gbs, "frac_of_hbm": gbs / peak}
    print(json.dumps({"stage_bench": res, "workload": w.name, "n_bins": nb, "window": w.window, "peak_gbs": peak,
                      "peak_source": peak_src, "l2": "flushed between repetitions (256 MB written)",
                      "note": "running_median: stage call without the PSD epilogue (16 B per bin), two launches"}), flush=True)
    return 0


def run_paper_path(args):
    """`--paper-path`: the path as the paper runs it (Fig. 3) through gbfg_simulate_paper: Lambda of Fig. 1
     with N_b = 1e7, T_obs = 4 yr, 0.1-10 mHz (Table I), running mean of eq. (D1) over 2001 bins, S_n stop rule
    at 1e-3, 100 coarse bins (eqs. 13-14).  Prints one JSON line (not the headline metric: another population model)."""
    import torch
    import paper_2602_18560_b200 as gb
    torch.cuda.set_device(0)
    gb.load()
    dev = torch.device("cuda", 0)
    w = wl.Workload(name="paper_fig1_1e7_4yr", t_obs=4 * wl.YEAR_S, f_min=1e-4, f_max=1e-2, window=2001, rho_th=7.0, max_iter=30, seed=7)
    pop = wl.PaperPopulation(n_src=10_000_000)
    g = gb.grid_init(w.f_min, w.f_max, w.t_obs, w.scale_log2)
    n, nb = pop.n_src, g.n_bins
    s_instr = torch.empty(nb, dtype=torch.float64, device=dev)
    gb.instrument_noise(g, s_instr)
    A, f, fd = (torch.empty(n, dtype=torch.float64, device=dev) for _ in range(3))
    spec, stat = (torch.empty(nb, dtype=torch.int64, device=dev) for _ in range(2))
    psd = torch.empty(nb, dtype=torch.float64, device=dev)
    resolved = torch.empty(n, dtype=torch.uint8, device=dev)
    ws = torch.empty(gb.workspace_bytes(g, n, 1), dtype=torch.uint8, device=dev)
    edges = torch.from_numpy(wl.log_bin_edges(w, 100)).to(dev)
    S, hc = (torch.empty(100, dtype=torch.float64, device=dev) for _ in range(2))
    fk = torch.empty(100, dtype=torch.float64, device=dev)
    params = gb.make_iter_params(w.window, w.median_norm, w.rho_th, w.max_iter, gb.FLAG_ESTIMATOR_MEAN, psd_rtol=1e-3)

    def step():
        return gb.simulate_paper(g, [pop], [0, n], w.seed, s_instr, params, A, f, fd, None, spec, stat, psd, resolved, ws,
                                 dev_edges=edges, n_coarse=100, dev_S_coarse=S, dev_f_coarse=fk, dev_hc=hc)
    for _ in range(max(args.warmup, 1)):
        res = step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        res = step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    r = res[0]
    print(json.dumps({"paper_path": {"ms_per_simulation": ms, "sources_per_s": n / (ms * 1e-3), "n_src": n, "n_bins": nb,
                                     "estimator": "running mean (eq. D1), 2001 bins", "psd_rtol": 1e-3, "n_iter": r.n_iter,
                                     "converged": r.converged, "n_resolved": r.n_resolved, "coarse_bins": 100,
                                     "population": "Fig. 1 parameters of the paper's model (Table I)", "steps": args.steps}}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gbfg", choices=["gbfg", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (default 3: the headline 1e7-source run)")
    ap.add_argument("--n-src", type=int, default=None, help="override the number of sources (parity/debug only)")
    ap.add_argument("--flags", type=int, default=0, help="gbfg_iter_params.flags")
    ap.add_argument("--max-iter", type=int, default=None, help="override the iteration cap (debug only: cost per iteration)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--stage-bench", action="store_true", help="time the two PSD estimators alone (one full pass each) and exit")
    ap.add_argument("--paper-path", action="store_true", help="time gbfg_simulate_paper (the paper's population, mean estimator, S_n stop rule, coarse-grained output) and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-config4", action="store_true",
                    help="also time the oracle on configs[4] (64 catalogs) over all host cores: minutes")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu --set full capture")
    args = ap.parse_args()
    w = wl.config(args.config)
    if args.n_src is not None:
        w = wl.scaled(w, n_src=args.n_src, name=f"{w.name}_n{args.n_src}")
    if args.max_iter is not None:
        w = wl.replace(w, max_iter=args.max_iter, name=f"{w.name}_cap{args.max_iter}")
    if args.impl == "reference":
        return run_reference(args, w)
    if args.stage_bench:
        return run_stage_bench(args, w)
    if args.paper_path:
        return run_paper_path(args)
    return run_gpu(args, w)


if __name__ == "__main__":
    sys.exit(main())
