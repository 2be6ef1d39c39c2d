#!/usr/bin/env python
"""bench.py - the whole hot path (geometry -> quiet spectrum -> active time series) on workload C3.

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --gpus N --steps K ...   # the fp64 CPU oracle, timed on the host cores

One "step" = soap_disk_geometry + soap_integrate_quiet + soap_active_timeseries for one star of the
full-visible-range workload (BASELINE.json configs[2]: N=300, 310 000 px, 20 mu bins x {quiet, spot, facula},
25 phases, fp32), inputs resident in HBM.  Prints ONE JSON line (rank 0).  See DESIGN.md section 7 for what
every field means and how the roofline numbers are derived.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "integrated spectra/s and cell*pixel interps/s (full visible, 300^2 grid), % roofline"
N_SM, FP32_LANES_PER_SM = 148, 128
FLOPS_PER_UNIT = 4  # one lerp-accumulate = 2 FP32 FMAs per (entry, pixel): acc += W u_r; acc += (W a) v_r
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture of this
# workload (profiles/r01_v5_sia_full.md); algorithmic: active 74.4 MB in + 31 MB out, quiet 24.8 MB in.
NCU_DRAM_TRAFFIC_BYTES = {"sia_f32_kernel<quiet>": 25.1e6, "sia_f32_kernel<active>": 109.5e6}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return dict(sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), hbm_gbs=float(d.get("hbm_gbs", 6650.0)), source="measured")
    return dict(sm_max_mhz=1965.0, hbm_gbs=6650.0, source="fallback")


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, torch_device_index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self._nv = pynvml
            try:
                uuid = torch.cuda.get_device_properties(torch_device_index).uuid
                self._h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = int(vis.split(",")[torch_device_index]) if vis and vis.split(",")[0].isdigit() else torch_device_index
                self._h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None

    def _loop(self):
        nv = self._nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.001)

    def start(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
        return dict(sm_mhz=float(np.median(self.samples)) if self.samples else None,
                    sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons), samples=len(self.samples))


def cpu_oracle_rate(wl, budget_s: float):
    """Times the oracle, as it stands, on a bounded pixel sample of the workload.  Returns
    (spectra/s extrapolated to the full pixel count, threads, sample description, seconds)."""
    import oracle
    oracle.build()
    threads = oracle.num_threads()
    probe = 2048
    t0 = time.perf_counter()
    oracle.run_workload(wl, 0, probe)
    t_probe = time.perf_counter() - t0
    px = int(min(wl.n_pix, max(probe, (budget_s / t_probe) * probe)))
    px = max(2048, (px // 2048) * 2048)
    lo = (wl.n_pix - px) // 2
    t0 = time.perf_counter()
    oracle.run_workload(wl, lo, lo + px)
    t = time.perf_counter() - t0
    n_spec = 1 + len(wl.phases)
    rate = n_spec / (t * wl.n_pix / px)
    return rate, threads, f"pixels [{lo}, {lo + px}) of {wl.n_pix} ({px / wl.n_pix:.1%}), all cells, all {len(wl.phases)} phases, extrapolated linearly in pixels", t


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads
    wl = workloads.make_config3()
    total_budget = 150.0
    per_step = max(1.0, total_budget / max(1, args.steps + args.warmup))
    rates, times = [], []
    sample = ""
    threads = 1
    for i in range(args.warmup + args.steps):
        rate, threads, sample, t = cpu_oracle_rate(wl, per_step * 0.8)
        if i >= args.warmup:
            rates.append(rate)
            times.append(t)
    n_spec = 1 + len(wl.phases)
    value = float(n_spec * len(rates) / sum(n_spec / r for r in rates))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "spectra/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * n_spec / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "C3 full visible range: N=300, 310000 px, 20 mu bins x {quiet,spot,facula}, 25 phases",
                   "note": "fp64 CPU oracle (oracle/soap_oracle.c, OpenMP) on a bounded pixel sample per step; ms_per_step is the extrapolated full-workload time"},
        "cpu_baseline": {"value": value, "unit": "spectra/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "spectra/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_graft(args):
    import torch
    import torch.distributed as dist

    import paper_2301_04259_b200 as soap
    import workloads
    from paper_2301_04259_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    soap.binding.load_library()
    peaks = load_peaks()

    # ---- workload: every rank synthesises its own star of the same shape (weak scaling, no collective) ----
    wl = workloads.make_config3()
    n_ph, P = len(wl.phases), wl.n_pix
    n_spec = 1 + n_ph
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    Q = torch.empty(P, dtype=torch.float32, device=dev)
    D = torch.empty((n_ph, P), dtype=torch.float32, device=dev)
    star = soap.soap_create(local_rank)
    if args.form is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, args.form)
    flush_buf = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step():
        soap.soap_disk_geometry(star, wl, want_info=False)
        soap.soap_integrate_quiet(star, q, Q)
        soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warmup = max(3, args.warmup)
    for _ in range(warmup):
        flush_buf.zero_()
        step()
    barrier()
    info = soap.soap_disk_geometry(star, wl)
    n_active = soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D, want_n_active=True)
    stats0 = soap.soap_get_stats(star)

    # ---- timed region: K steps, L2 flushed before each, CUDA events around each step --------------------
    sampler = ClockSampler(local_rank)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler.start()
    wall0 = time.perf_counter()
    for a, b in ev:
        flush_buf.zero_()
        a.record()
        step()
        b.record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    stats1 = soap.soap_get_stats(star)
    launches = stats1["launches"] - stats0["launches"]
    total_ms = sharding.max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / args.steps
    value = world * n_spec / (ms_per_step * 1e-3)

    # ---- per-kernel durations (CUDA events inside the library, same stream), L2 flushed ------------------
    soap.soap_set_option(star, soap.binding.SOAP_OPT_KERNEL_TIMING, 1)
    kq, ka = [], []
    for _ in range(max(5, min(args.steps, 30))):
        flush_buf.zero_()
        step()
        st = soap.soap_get_stats(star)
        kq.append(st["quiet_kernel_ms"])
        ka.append(st["active_kernel_ms"])
    soap.soap_set_option(star, soap.binding.SOAP_OPT_KERNEL_TIMING, 0)
    stats = soap.soap_get_stats(star)
    units_q = stats["quiet_entries"] * P
    units_a = stats["active_entries"] * P
    kern = {
        "sia_f32_kernel<quiet>": dict(ms=float(np.mean(kq)), units=units_q),
        "sia_f32_kernel<active>": dict(ms=float(np.mean(ka)), units=units_a),
    }
    dom = max(kern, key=lambda k: kern[k]["ms"])
    peak_tflops = N_SM * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    achieved = kern[dom]["units"] * FLOPS_PER_UNIT / (kern[dom]["ms"] * 1e-3) / 1e12
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops, "traffic": NCU_DRAM_TRAFFIC_BYTES.get(dom),
        "peak_source": f"148 SMs x 128 FP32 lanes x 2 FLOP x {peaks['sm_max_mhz']:.0f} MHz (sm_max_mhz, {peaks['source']} MEASURED_PEAKS.json)",
        "kernel_ms": kern[dom]["ms"], "units_per_launch": kern[dom]["units"], "flop_per_unit": FLOPS_PER_UNIT,
    }
    if clocks.get("sm_mhz"):
        roofline["frac_at_observed_clock"] = achieved / (peak_tflops * clocks["sm_mhz"] / peaks["sm_max_mhz"])
    other = [k for k in kern if k != dom][0]
    roofline["other_kernel"] = {"kernel": other, "kernel_ms": kern[other]["ms"],
                                "achieved": kern[other]["units"] * FLOPS_PER_UNIT / (kern[other]["ms"] * 1e-3) / 1e12}

    # ---- the run-collapsed form (SOAP_FORM_FIR): same sums, every run of entries with one integer
    # shift collapsed into one record by the producer warps.  Reported beside the north_star form, never as it.
    star_fir = soap.soap_create(local_rank)
    soap.soap_set_option(star_fir, soap.binding.SOAP_OPT_FORM, 3)
    Qf = torch.empty_like(Q)
    Df = torch.empty_like(D)

    def step_fir():
        soap.soap_disk_geometry(star_fir, wl, want_info=False)
        soap.soap_integrate_quiet(star_fir, q, Qf)
        soap.soap_active_timeseries(star_fir, q, s, f, wl.regions, wl.phases, Df)

    for _ in range(3):
        step_fir()
    fir_steps = max(5, min(args.steps, 30))
    fir_ms = 0.0
    soap.soap_set_option(star_fir, soap.binding.SOAP_OPT_KERNEL_TIMING, 1)
    fq, fa = [], []
    for _ in range(fir_steps):
        flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        step_fir()
        b.record()
        b.synchronize()
        fir_ms += a.elapsed_time(b)
        st = soap.soap_get_stats(star_fir)
        fq.append(st["quiet_kernel_ms"])
        fa.append(st["active_kernel_ms"])
    fir_ms = sharding.max_over_ranks(fir_ms, dev) / fir_steps
    fir = {"form": "fir (runs collapsed; SOAP_OPT_FORM=3)", "ms_per_step": fir_ms, "value": world * n_spec / (fir_ms * 1e-3),
           "unit": "spectra/s", "quiet_kernel_ms": float(np.mean(fq)), "active_kernel_ms": float(np.mean(fa)),
           "max_abs_diff_vs_binned_over_sum_w": float((Qf - Q).abs().max().item()) / info["sum_weights"],
           "note": "event timing inside the library adds ~10 us per step to this figure"}
    soap.soap_destroy(star_fir)

    # ---- resolution lowering of the 26 final spectra to R = 115 000 (HBM-bound: 1 read + 1 write)
    F = torch.empty((n_spec, P), dtype=torch.float32, device=dev)
    F[0] = Q
    F[1:] = Q.unsqueeze(0) + D
    Flow = torch.empty_like(F)
    lsf_ms = []
    for it in range(8):
        flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        soap.soap_lower_resolution(star, F, P, wl.lambda0, wl.dlambda, 115000.0, Flow)
        b.record()
        b.synchronize()
        if it >= 3:
            lsf_ms.append(a.elapsed_time(b))
    lsf_bytes = 2 * n_spec * P * 4
    lsf = {"kernel": "lower_resolution_kernel<float>", "R": 115000, "rows": n_spec, "ms": float(np.mean(lsf_ms)),
           "bound": "hbm", "achieved": lsf_bytes / (float(np.mean(lsf_ms)) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
           "algorithmic_bytes": lsf_bytes}
    lsf["frac"] = lsf["achieved"] / lsf["peak"]

    # ---- first-moment RV of every generated line in every lowered spectrum (the reduction after the path)
    centres = torch.from_numpy(wl.line_centres.astype(np.float64)).to(dev)
    halfw = torch.from_numpy((3.0 * np.maximum(wl.line_sigmas, 0.03)).astype(np.float64)).to(dev)
    norm = torch.full((n_spec,), float(info["sum_weights"]), dtype=torch.float64, device=dev)
    rv_ms = []
    for it in range(8):
        flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        rvs = soap.soap_line_rvs(star, Flow, P, wl.lambda0, wl.dlambda, centres, halfw, norm, 64)
        b.record()
        b.synchronize()
        if it >= 3:
            rv_ms.append(a.elapsed_time(b))
    rv_bytes = n_spec * P * 4 + n_spec * len(wl.line_centres) * 8
    line_rv = {"kernel": "line_rv_kernel<float>", "lines": int(len(wl.line_centres)), "rows": n_spec, "ms": float(np.mean(rv_ms)),
               "bound": "hbm", "achieved": rv_bytes / (float(np.mean(rv_ms)) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
               "algorithmic_bytes": rv_bytes, "finite": int(torch.isfinite(rvs).sum().item())}
    line_rv["frac"] = line_rv["achieved"] / line_rv["peak"]

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ------------
    pitch = q.pitch

    def pinned(rows):
        t = torch.zeros((rows.shape[0], pitch), dtype=torch.float32).pin_memory()
        t[:, :P] = torch.from_numpy(rows)
        return t

    hq = soap.Spectra(pinned(wl.quiet), P, wl.lambda0, wl.dlambda)
    hs = soap.Spectra(pinned(wl.spot), P, wl.lambda0, wl.dlambda, contrast=torch.from_numpy(wl.spot_contrast).pin_memory(), lb=wl.spot_lb)
    hf = soap.Spectra(pinned(wl.facula), P, wl.lambda0, wl.dlambda, contrast=None, lb=wl.facula_lb)
    hQ = torch.empty(P, dtype=torch.float32).pin_memory()
    hD = torch.empty((n_ph, P), dtype=torch.float32).pin_memory()
    star2 = soap.soap_create(local_rank)
    for _ in range(3):
        soap.soap_synthesize_host(star2, wl, hq, hs, hf, wl.regions, wl.phases, hQ, hD)
    e2e_steps = max(3, min(args.steps, 20))
    barrier()
    e2e_ms = 0.0
    for _ in range(e2e_steps):
        flush_buf.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        soap.soap_synthesize_host(star2, wl, hq, hs, hf, wl.regions, wl.phases, hQ, hD)
        b.record()
        b.synchronize()
        e2e_ms += a.elapsed_time(b)
    e2e_ms = sharding.max_over_ranks(e2e_ms, dev)
    e2e_value = world * n_spec / (e2e_ms / e2e_steps * 1e-3)
    h2d = 3 * wl.n_mu * pitch * 4 + P * 4
    d2h = n_spec * P * 4
    # the host path computes wavelength chunks (different CTA ranges => different fp64 summation order): equal to rounding
    assert float((hQ.to(dev) - Q).abs().max()) <= 1e-6 * info["sum_weights"]
    assert float((hD.to(dev) - D).abs().max()) <= 1e-5 * float(D.abs().max())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    n_vis = info["n_visible"]
    act_cells = int(n_active.sum())
    eff_interps = (n_vis + 2 * act_cells) * P  # what Alg. 1 / Alg. 5 would execute per star
    exec_units = units_q + units_a
    line = {
        "metric": METRIC, "value": value, "unit": "spectra/s", "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": "C3 full visible range (BASELINE.json configs[2]): N=300, vsini=2 km/s, i=90, 310000 px 3800-6900 A, "
                               "20 mu bins x {quiet,spot,facula}, 25000 lines, 3% facula + 1% spot, 25 phases, fp32",
                   "stars_per_gpu": 1, "spectra_per_step": n_spec, "form": {1: "binned", 2: "cells", 3: "fir", 4: "composite"}[stats["form"]],
                   "l2": "512 MB buffer written before every timed step (inputs+outputs 106 MB < 126 MB L2)",
                   "timing": "sum of per-step CUDA-event intervals, max over ranks", "sharding": "independent stars per rank, no collective"},
        "cell_pixel_interps_per_s": world * eff_interps / (ms_per_step * 1e-3),
        "executed_lerp_accumulates_per_s": world * exec_units / (ms_per_step * 1e-3),
        "definitional": {"n_visible": n_vis, "active_cells_all_phases": act_cells, "quiet_entries": stats["quiet_entries"],
                         "active_entries_all_phases": stats["active_entries"]},
        "roofline": roofline, "fir_form": fir, "lower_resolution": lsf, "line_rvs": line_rv, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "spectra/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "api": "soap_synthesize_host (pinned host buffers)"},
        "gpu_launches": launches, "wall_s_timed_region": wall,
    }
    if world == 1 and not args.no_cpu_baseline:
        rate, threads, sample, _ = cpu_oracle_rate(wl, 12.0)
        line["cpu_baseline"] = {"value": rate, "unit": "spectra/s", "cores": threads, "kind": "oracle", "sample": sample}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_configs(args):
    """--workload C2|C4|C5|all: device-resident timing of the other BASELINE.json configs (parity-test cases, not the
    headline): one JSON line per config with the step time and the two kernels' durations and ALU fractions."""
    import torch

    import paper_2301_04259_b200 as soap
    import workloads

    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    peaks = load_peaks()
    peak_tflops = N_SM * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    flush_buf = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)
    which = ["C2", "C3", "C4", "C5"] if args.workload == "all" else [args.workload]
    for name in which:
        if name == "C5":
            shared = workloads.make_config5_star(0)
            wls = [shared] + [workloads.make_config5_star(k, shared=shared) for k in range(1, 64)]
        else:
            wls = [{"C2": workloads.make_config2, "C3": workloads.make_config3, "C4": workloads.make_config4}[name]()]
        if args.vsini is not None:
            for w in wls:
                w.vsini_kms = args.vsini
        w0 = wls[0]
        P, n_ph = w0.n_pix, len(w0.phases)
        q = soap.to_device_spectra(w0.quiet, w0.lambda0, w0.dlambda, dev)
        sp = soap.to_device_spectra(w0.spot, w0.lambda0, w0.dlambda, dev, w0.spot_contrast, w0.spot_lb)
        fa = None if w0.facula is None else soap.to_device_spectra(w0.facula, w0.lambda0, w0.dlambda, dev, w0.facula_contrast, w0.facula_lb)
        stars = [soap.soap_create(dev.index) for _ in wls]
        if args.form is not None:
            for st_ in stars:
                soap.soap_set_option(st_, soap.binding.SOAP_OPT_FORM, args.form)
        Q = torch.empty((len(wls), P), dtype=torch.float32, device=dev)
        D = torch.empty((len(wls), n_ph, P), dtype=torch.float32, device=dev)

        def step():
            if len(wls) == 1:
                soap.soap_disk_geometry(stars[0], wls[0], want_info=False)
                soap.soap_integrate_quiet(stars[0], q, Q[0])
                soap.soap_active_timeseries(stars[0], q, sp, fa, wls[0].regions, wls[0].phases, D[0])
                return
            for st, wl in zip(stars, wls):  # config 5: the batch entry points (three lanes, one stream to the caller)
                soap.soap_disk_geometry(st, wl, want_info=False)
            soap.soap_batch_integrate_quiet(stars, [q] * len(wls), [Q[k] for k in range(len(wls))])
            soap.soap_batch_active_timeseries(stars, [q] * len(wls), [sp] * len(wls), [fa] * len(wls), [w.regions for w in wls],
                                              [w.phases for w in wls], [D[k] for k in range(len(wls))])

        for _ in range(3):
            step()
        torch.cuda.synchronize()
        steps = max(3, min(args.steps, 10))
        ms = 0.0
        for _ in range(steps):
            flush_buf.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            step()
            b.record()
            b.synchronize()
            ms += a.elapsed_time(b)
        ms /= steps
        # kernel durations of the first star
        soap.soap_set_option(stars[0], soap.binding.SOAP_OPT_KERNEL_TIMING, 1)
        soap.soap_disk_geometry(stars[0], wls[0], want_info=False)
        soap.soap_integrate_quiet(stars[0], q, Q[0])
        soap.soap_active_timeseries(stars[0], q, sp, fa, wls[0].regions, wls[0].phases, D[0])
        st = soap.soap_get_stats(stars[0])
        n_spec = len(wls) * (1 + n_ph)
        line = {"workload": workloads.CONFIG_NAMES[int(name[1])], "vsini_kms": float(w0.vsini_kms), "stars": len(wls), "ms_per_step": ms,
                "spectra_per_s": n_spec / (ms * 1e-3), "first_star": {
                    "quiet_entries": st["quiet_entries"], "active_entries": st["active_entries"],
                    "quiet_kernel_ms": st["quiet_kernel_ms"], "active_kernel_ms": st["active_kernel_ms"],
                    "quiet_alu_frac": st["quiet_entries"] * P * FLOPS_PER_UNIT / (st["quiet_kernel_ms"] * 1e-3) / 1e12 / peak_tflops,
                    "active_alu_frac": (st["active_entries"] * P * FLOPS_PER_UNIT / (st["active_kernel_ms"] * 1e-3) / 1e12 / peak_tflops)
                    if st["active_kernel_ms"] > 0 else None}}
        print(json.dumps(line))
        for s_ in stars:
            soap.soap_destroy(s_)
        del Q, D, q, sp, fa


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["graft", "reference"], default="graft")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--form", type=int, default=None, help="SOAP_OPT_FORM of the timed star (default: the library's AUTO)")
    ap.add_argument("--vsini", type=float, default=None, help="with --workload: override v sin i (km/s) of every star")
    ap.add_argument("--workload", choices=["C3", "C2", "C4", "C5", "all"], default="C3",
                    help="C3 (default) is the bench contract; the others print per-config timing lines only")
    args = ap.parse_args()
    if args.impl != "reference" and (args.workload != "C3" or args.vsini is not None):
        run_configs(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_graft(args)


if __name__ == "__main__":
    main()
