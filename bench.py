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
import csv
import hashlib
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
# Algorithmic FP32 lane-instructions, each credited as one FMA = 2 FLOP against the FMA peak:
#   binned entries: 2 FMAs per (entry, pixel):  acc1 += W u,  acc2 += (W a) d
#   composite columns: 1 FMA per (column, mu-bin, pixel) + 4 per (column, pixel): t = a c - q, d = x1 - x0, acc += t d, acc += x0
LANE_INSTR_PER_UNIT_BINNED = 2
LANE_INSTR_PER_UNIT_COMPOSITE = 1
LANE_INSTR_PER_COLUMN_PIXEL_COMPOSITE = 4
FORM_NAMES = {1: "binned", 2: "cells", 3: "fir", 4: "composite"}
WORKLOAD_C3 = ("C3 full visible range (BASELINE.json configs[2]): N=300, vsini=2 km/s, i=90, 310000 px 3800-6900 A, "
               "20 mu bins x {quiet,spot,facula}, 25000 lines, 3% facula + 1% spot, 25 phases, fp32")


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return dict(sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), hbm_gbs=float(d.get("hbm_gbs", 6650.0)), source="measured")
    return dict(sm_max_mhz=1965.0, hbm_gbs=6650.0, source="fallback")


def kernel_source_sha() -> str:
    """Hash of the CUDA sources the library is built from: ties an ncu capture under profiles/ to the build that ran."""
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2301_04259_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh")):
            with open(os.path.join(csrc, name), "rb") as fh:
                h.update(name.encode())
                h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_dram_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture
    (profiles/rNN_dram_traffic.csv of the newest round: kernel, bytes read, bytes written, source hash).  A row counts only if it was
    captured from the sources this run was built from; otherwise the figure is stale and `traffic` is null."""
    cands = sorted(f for f in os.listdir(os.path.join(ROOT, "profiles")) if f.endswith("_dram_traffic.csv"))
    out = {}
    if not cands:
        return out, "profiles/*_dram_traffic.csv missing: null"
    name = cands[-1]  # the newest round's
    path = os.path.join(ROOT, "profiles", name)
    sha = kernel_source_sha()
    with open(path) as fh:
        for row in csv.DictReader(fh):
            if row["source_sha"] == sha:
                out[row["kernel"]] = float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    if out:
        return out, f"profiles/{name}, captured from the sources of this build ({sha})"
    return out, f"profiles/{name} is of other sources than this build ({sha}): null"


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


# ------------------------------------------------------------------------------------------------------------------
# the oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------------------------
def oracle_full(wl):
    """ONE full-size run of the oracle (all cells, all pixels, all phases): (seconds, threads)."""
    import oracle
    oracle.build()
    t0 = time.perf_counter()
    oracle.run_workload(wl)
    return time.perf_counter() - t0, oracle.num_threads()


def oracle_sample(wl, px: int):
    """The oracle on a window of `px` pixels in the middle of the spectrum (all cells, all phases): seconds."""
    import oracle
    px = int(min(wl.n_pix, px))
    lo = (wl.n_pix - px) // 2
    t0 = time.perf_counter()
    oracle.run_workload(wl, lo, lo + px)
    return time.perf_counter() - t0, lo, px


def oracle_single_thread_c2():
    """the oracle's single-thread time on C2 (quiet + 100-phase time series)."""
    import oracle
    import workloads
    wl = workloads.make_config2()
    n = oracle.num_threads()
    oracle.set_threads(1)
    try:
        t0 = time.perf_counter()
        oracle.run_workload(wl)
        t = time.perf_counter() - t0
    finally:
        oracle.set_threads(n)
    return t, 1 + len(wl.phases)


def run_reference(args):
    """The tier's reference arm: the fp64 CPU oracle on C3.  The first timed step is ONE full-size run, measured as it
    is ("sample": "full") - `value` comes from it alone; the remaining steps (and the warm-ups) are bounded samples of the
    same workload so that the whole run ends within a few minutes, and `ms_per_step` is the mean wall time of the K timed
    steps that were actually run."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads
    wl = workloads.make_config3()
    n_spec = 1 + len(wl.phases)
    sample_px = 8192
    for _ in range(args.warmup):
        oracle_sample(wl, sample_px)
    t_full, threads = oracle_full(wl)
    step_s = [t_full]
    sample_rates = []
    for _ in range(max(0, args.steps - 1)):
        t, lo, px = oracle_sample(wl, sample_px)
        step_s.append(t)
        sample_rates.append(n_spec / (t * wl.n_pix / px))
    value = n_spec / t_full
    sample = "full: all 70688 cells x 310000 px x (1 quiet + 25 phases), one run, measured"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "spectra/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(step_s)), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_C3,
                   "note": "fp64 CPU oracle (oracle/soap_oracle.c, OpenMP over wavelength chunks). value = 26 spectra / the one "
                           "full-size step; the other timed steps and the warm-ups are %d-pixel samples (all cells, all phases); "
                           "ms_per_step = mean wall time of the timed steps as run" % sample_px,
                   "full_run_ms": 1e3 * t_full,
                   "sampled_steps_extrapolated_spectra_per_s": float(np.median(sample_rates)) if sample_rates else None},
        "cpu_baseline": {"value": value, "unit": "spectra/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "spectra/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------------------
# this repo's CUDA path
# ------------------------------------------------------------------------------------------------------------------
class Timer:
    def __init__(self, torch, flush_buf):
        self.torch, self.flush = torch, flush_buf

    def steps(self, fn, n, warm=3):
        """ms of n calls of fn, each bracketed by CUDA events on the current stream, L2 flushed before each."""
        torch = self.torch
        for _ in range(warm):
            self.flush.zero_()
            fn()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in ev:
            self.flush.zero_()
            a.record()
            fn()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]


def lane_instr(form: int, quiet_entries: int, active_entries: int, n_columns: int, P: int):
    """Algorithmic FP32 lane-instructions per launch of the two shift-interpolate-accumulate kernels."""
    if form == 4:
        q = (quiet_entries * LANE_INSTR_PER_UNIT_COMPOSITE + n_columns * LANE_INSTR_PER_COLUMN_PIXEL_COMPOSITE) * P
    else:
        q = quiet_entries * LANE_INSTR_PER_UNIT_BINNED * P
    return q, active_entries * LANE_INSTR_PER_UNIT_BINNED * P


def time_form(soap, torch, timer, wl, q, s, f, form, steps, dev_index, peak_instr):
    """Step time and the two kernels' durations of one evaluation form (SOAP_OPT_FORM) on a star of workload wl."""
    star = soap.soap_create(dev_index)
    if form is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, form)
    P, n_ph = wl.n_pix, len(wl.phases)
    dev = q.data.device
    Q = torch.empty(P, dtype=torch.float32, device=dev)
    D = torch.empty((n_ph, P), dtype=torch.float32, device=dev)

    def step():
        soap.soap_disk_geometry(star, wl, want_info=False)
        soap.soap_integrate_quiet(star, q, Q)
        soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D)

    ms = timer.steps(step, steps)
    soap.soap_set_option(star, soap.binding.SOAP_OPT_KERNEL_TIMING, 1)
    kq, ka = [], []
    for _ in range(max(5, min(steps, 20))):
        timer.flush.zero_()
        step()
        st = soap.soap_get_stats(star)
        kq.append(st["quiet_kernel_ms"])
        ka.append(st["active_kernel_ms"])
    soap.soap_set_option(star, soap.binding.SOAP_OPT_KERNEL_TIMING, 0)
    st = soap.soap_get_stats(star)
    iq, ia = lane_instr(st["form"], st["quiet_entries"], st["active_entries"], wl.grid_n, P)
    mq, ma, mm = float(np.mean(kq)), float(np.mean(ka)), float(np.mean(ms))
    out = {
        "form": FORM_NAMES[st["form"]], "ms_per_step": mm, "ms_per_step_median": float(np.median(ms)),
        "ms_per_step_best": float(np.min(ms)), "spectra_per_s": (1 + n_ph) / (mm * 1e-3),
        "quiet_kernel_ms": mq, "active_kernel_ms": ma,
        "quiet_entries": st["quiet_entries"], "active_entries": st["active_entries"],
        "quiet_lane_instr": iq, "active_lane_instr": ia,
        "quiet_alu_frac": iq / (mq * 1e-3) / peak_instr if mq > 0 else None,
        "active_alu_frac": ia / (ma * 1e-3) / peak_instr if ma > 0 else None,
        "step_alu_frac": (iq + ia) / (mm * 1e-3) / peak_instr,
    }
    return out, star, Q, D


def config_lines(soap, torch, timer, workloads, dev, steps, peak_instr):
    """Device-resident timing of the other BASELINE.json configs (parity-test cases beside the C3 headline)."""
    res = {}
    for name in ("C2", "C4", "C5"):
        if name == "C5":
            shared = workloads.make_config5_star(0)
            wls = [shared] + [workloads.make_config5_star(k, shared=shared) for k in range(1, 64)]
        else:
            wls = [{"C2": workloads.make_config2, "C4": workloads.make_config4}[name]()]
        w0 = wls[0]
        P, n_ph, n = w0.n_pix, len(w0.phases), len(wls)
        q = soap.to_device_spectra(w0.quiet, w0.lambda0, w0.dlambda, dev)
        sp = soap.to_device_spectra(w0.spot, w0.lambda0, w0.dlambda, dev, w0.spot_contrast, w0.spot_lb)
        fa = None if w0.facula is None else soap.to_device_spectra(w0.facula, w0.lambda0, w0.dlambda, dev, w0.facula_contrast, w0.facula_lb)
        stars = [soap.soap_create(dev.index) for _ in wls]
        Q = torch.empty((n, P), dtype=torch.float32, device=dev)
        D = torch.empty((n, n_ph, P), dtype=torch.float32, device=dev)

        def step():
            if n == 1:
                soap.soap_disk_geometry(stars[0], w0, want_info=False)
                soap.soap_integrate_quiet(stars[0], q, Q[0])
                soap.soap_active_timeseries(stars[0], q, sp, fa, w0.regions, w0.phases, D[0])
                return
            soap.soap_batch_disk_geometry(stars, wls)
            soap.soap_batch_integrate_quiet(stars, [q] * n, [Q[k] for k in range(n)])
            soap.soap_batch_active_timeseries(stars, [q] * n, [sp] * n, [fa] * n, [w.regions for w in wls],
                                              [w.phases for w in wls], [D[k] for k in range(n)])

        ms = timer.steps(step, max(3, min(steps, 10)))
        # kernel durations: the launches carry the whole batch and are timed on the first star's handle
        soap.soap_set_option(stars[0], soap.binding.SOAP_OPT_KERNEL_TIMING, 1)
        step()
        st = soap.soap_get_stats(stars[0])
        soap.soap_set_option(stars[0], soap.binding.SOAP_OPT_KERNEL_TIMING, 0)
        per = [soap.soap_get_stats(s_) for s_ in stars]
        q_ent = sum(p_["quiet_entries"] for p_ in per)
        a_ent = sum(p_["active_entries"] for p_ in per)
        iq, ia = lane_instr(st["form"], q_ent, a_ent, sum(w.grid_n for w in wls), P)
        launches0 = sum(p_["launches"] for p_ in per)
        step()
        torch.cuda.synchronize()
        launches = sum(soap.soap_get_stats(s_)["launches"] for s_ in stars) - launches0
        mm = float(np.mean(ms))
        graph_ms = None
        if n == 1 and len(w0.regions) * n_ph <= 192:  # a single star's step whose region centres travel as kernel arguments
            # enqueues kernels only and can be captured in a CUDA graph (include/soap_b200.h)
            try:
                side = torch.cuda.Stream()
                with torch.cuda.stream(side):
                    step()
                    side.synchronize()
                    graph = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(graph, stream=side):
                        step()
                torch.cuda.synchronize()
                graph_ms = float(np.mean(timer.steps(graph.replay, max(3, min(steps, 10)))))
            except Exception:
                graph_ms = None
        res[name] = {
            "workload": workloads.CONFIG_NAMES[int(name[1])], "stars": n, "ms_per_step": mm,
            "ms_per_step_median": float(np.median(ms)), "ms_per_step_best": float(np.min(ms)),
            "spectra_per_s": n * (1 + n_ph) / (mm * 1e-3), "launches_per_step": launches,
            "ms_per_step_cuda_graph": graph_ms,
            "quiet_form": FORM_NAMES[st["form"]], "quiet_entries": q_ent, "active_entries": a_ent,
            "quiet_kernel_ms": st["quiet_kernel_ms"], "active_kernel_ms": st["active_kernel_ms"],
            "quiet_alu_frac": iq / (st["quiet_kernel_ms"] * 1e-3) / peak_instr if st["quiet_kernel_ms"] > 0 else None,
            "active_alu_frac": ia / (st["active_kernel_ms"] * 1e-3) / peak_instr if st["active_kernel_ms"] > 0 else None,
        }
        for s_ in stars:
            soap.soap_destroy(s_)
        del Q, D, q, sp, fa
        torch.cuda.empty_cache()
    return res


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
    peak_instr = N_SM * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6   # FP32 lane-instructions (FMAs) per second
    peak_tflops = 2 * peak_instr / 1e12

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
    timer = Timer(torch, flush_buf)

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

    # ---- the same step captured once in a CUDA graph and replayed (a single star's step enqueues four kernels and nothing
    # else, so it can be captured; the host-side cost of the three calls drops out) ------------------------------------------
    graph_ms = None
    try:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            step()
            side.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                step()
        torch.cuda.synchronize()
        graph_ms = float(np.mean(timer.steps(graph.replay, max(5, min(args.steps, 20)))))
    except Exception as exc:  # reported, never fatal: the graph leg is informational
        graph_ms = None
        sys.stderr.write(f"cuda graph leg skipped: {exc}\n")

    # ---- the device's FP32 FMA rate, measured live with the inner loops' instruction forms ----------------
    from paper_2301_04259_b200 import benchlib  # libsoap_b200_bench.so: the probe is not part of the product library
    probe = {"ffma2_fma_per_s": benchlib.fp32_rate(local_rank, True), "ffma_fma_per_s": benchlib.fp32_rate(local_rank, False),
             "derived_fma_per_s": peak_instr}
    probe["ffma2_over_derived"] = probe["ffma2_fma_per_s"] / peak_instr
    probe["ffma_over_derived"] = probe["ffma_fma_per_s"] / peak_instr

    # ---- per-kernel durations (CUDA events inside the library, same stream), L2 flushed: the form that was timed above,
    # the north_star form (binned entries for both launches) and the run-collapsed form -------------------------------
    k_steps = max(5, min(args.steps, 20))
    forms = {}
    main_form, star_m, Qm, Dm = time_form(soap, torch, timer, wl, q, s, f, args.form, k_steps, local_rank, peak_instr)
    soap.soap_destroy(star_m)
    forms[main_form["form"]] = main_form
    for code in (1, 3):
        if FORM_NAMES[code] in forms:
            continue
        r, st_, Qx, Dx = time_form(soap, torch, timer, wl, q, s, f, code, k_steps, local_rank, peak_instr)
        r["max_abs_diff_of_quiet_vs_timed_form_over_sum_w"] = float((Qx - Qm).abs().max().item()) / info["sum_weights"]
        r["max_abs_diff_of_delta_vs_timed_form_over_max_delta"] = float((Dx - Dm).abs().max().item()) / float(Dm.abs().max().item())
        soap.soap_destroy(st_)
        forms[r["form"]] = r
        del Qx, Dx
    traffic, traffic_note = ncu_dram_traffic()
    kq_name = "composite_quiet_kernel" if main_form["form"] == "composite" else "sia_f32_kernel<quiet>"
    kern = {
        kq_name: dict(ms=main_form["quiet_kernel_ms"], instr=main_form["quiet_lane_instr"], units=main_form["quiet_entries"] * P),
        "sia_f32_kernel<active>": dict(ms=main_form["active_kernel_ms"], instr=main_form["active_lane_instr"],
                                       units=main_form["active_entries"] * P),
    }
    dom = max(kern, key=lambda k_: kern[k_]["ms"])
    other = [k_ for k_ in kern if k_ != dom][0]

    def tflops(k_):
        return 2 * kern[k_]["instr"] / (kern[k_]["ms"] * 1e-3) / 1e12

    step_instr = kern[dom]["instr"] + kern[other]["instr"]
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": tflops(dom), "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": tflops(dom) / peak_tflops, "traffic": traffic.get(dom), "traffic_source": traffic_note,
        "peak_source": f"148 SMs x 128 FP32 lanes x 2 FLOP x {peaks['sm_max_mhz']:.0f} MHz (sm_max_mhz, {peaks['source']} MEASURED_PEAKS.json); "
                       f"live FFMA2 probe on this device: {100 * probe['ffma2_over_derived']:.1f} % of it",
        "kernel_ms": kern[dom]["ms"], "units_per_launch": kern[dom]["units"], "lane_instr_per_launch": kern[dom]["instr"],
        "flop_per_lane_instr": 2,
        "other_kernel": {"kernel": other, "kernel_ms": kern[other]["ms"], "achieved": tflops(other), "frac": tflops(other) / peak_tflops,
                         "units_per_launch": kern[other]["units"], "lane_instr_per_launch": kern[other]["instr"],
                         "traffic": traffic.get(other)},
        "whole_step": {"lane_instr": step_instr, "frac": 2 * step_instr / (ms_per_step * 1e-3) / 1e12 / peak_tflops,
                       "frac_at_4_flop_per_binned_unit": 4 * (main_form["quiet_entries"] + main_form["active_entries"]) * P /
                                                         (ms_per_step * 1e-3) / 1e12 / peak_tflops},
        "fp32_probe": probe,
    }
    if clocks.get("sm_mhz"):
        roofline["frac_at_observed_clock"] = roofline["frac"] * peaks["sm_max_mhz"] / clocks["sm_mhz"]
    # the same figures as flat scalars (a record that keeps scalar fields only still carries them).  The roofline fraction of
    # the whole step counts the lane instructions of the forms that RAN; `whole_step_binned_equivalent` credits the composite
    # quiet launch with the binned form's 2 FMA per (entry, pixel), work it avoids: a throughput in binned units, not a
    # fraction of the roofline
    roofline.update({
        "quiet_kernel": kq_name, "quiet_kernel_ms": kern[kq_name]["ms"], "quiet_frac": tflops(kq_name) / peak_tflops,
        "active_kernel_ms": kern["sia_f32_kernel<active>"]["ms"], "active_frac": tflops("sia_f32_kernel<active>") / peak_tflops,
        "whole_step_frac_executed": roofline["whole_step"]["frac"],
        "whole_step_binned_equivalent": roofline["whole_step"]["frac_at_4_flop_per_binned_unit"],
        "ffma2_probe_frac": probe["ffma2_over_derived"], "ffma_probe_frac": probe["ffma_over_derived"],
    })

    # ---- the run-collapsed form against the memory roofline it moves the path to --------------
    fir = forms.get("fir")
    if fir is not None:
        q_bytes = wl.n_mu * P * 4 + P * 4
        a_bytes = 3 * wl.n_mu * P * 4 + P * 4 + n_ph * P * 4
        step_bytes = a_bytes + P * 4

        def hbm(nbytes, ms):
            g = nbytes / (ms * 1e-3) / 1e9
            return {"algorithmic_bytes": nbytes, "achieved": g, "frac": g / peaks["hbm_gbs"]}

        fir["roofline"] = {
            "bound": "hbm", "peak": peaks["hbm_gbs"], "unit": "GB/s",
            "quiet": hbm(q_bytes, fir["quiet_kernel_ms"]), "active": hbm(a_bytes, fir["active_kernel_ms"]),
            "whole_step": hbm(step_bytes, fir["ms_per_step"]),
            "traffic": {"quiet": traffic.get("sia_f32_kernel<quiet>/fir"), "active": traffic.get("sia_f32_kernel<active>/fir")},
            "note": "algorithmic bytes: every table read once and every output written once per launch (the quiet table is read by both "
                    "launches).  Executed FMAs are 2 per (run, pixel) instead of 2 per (entry, pixel); what is left is the per-run window "
                    "set-up and the producers' run building, so the form is still far from the HBM roofline it is re-baselined against",
        }

    # ---- resolution lowering of the 26 final spectra to R = 115 000 (HBM-bound: 1 read + 1 write)
    F = torch.empty((n_spec, P), dtype=torch.float32, device=dev)
    F[0] = Q
    F[1:] = Q.unsqueeze(0) + D
    Flow = torch.empty_like(F)
    lsf_ms = timer.steps(lambda: soap.soap_lower_resolution(star, F, P, wl.lambda0, wl.dlambda, 115000.0, Flow), 5)
    lsf_bytes = 2 * n_spec * P * 4
    lsf = {"kernel": "lower_resolution_p_kernel", "R": 115000, "rows": n_spec, "ms": float(np.mean(lsf_ms)),
           "bound": "hbm", "achieved": lsf_bytes / (float(np.mean(lsf_ms)) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
           "algorithmic_bytes": lsf_bytes, "traffic": traffic.get("lower_resolution_p_kernel")}
    lsf["frac"] = lsf["achieved"] / lsf["peak"]

    # ---- first-moment RV of every generated line in every lowered spectrum (the reduction after the path)
    centres = torch.from_numpy(wl.line_centres.astype(np.float64)).to(dev)
    halfw = torch.from_numpy((3.0 * np.maximum(wl.line_sigmas, 0.03)).astype(np.float64)).to(dev)
    norm = torch.full((n_spec,), float(info["sum_weights"]), dtype=torch.float64, device=dev)
    rvs_box = {}

    def rv_call():
        rvs_box["rv"] = soap.soap_line_rvs(star, Flow, P, wl.lambda0, wl.dlambda, centres, halfw, norm, 64)

    rv_ms = timer.steps(rv_call, 5)
    rv_bytes = n_spec * P * 4 + n_spec * len(wl.line_centres) * 8
    line_rv = {"kernel": "line_rv_kernel", "lines": int(len(wl.line_centres)), "rows": n_spec, "ms": float(np.mean(rv_ms)),
               "bound": "hbm", "achieved": rv_bytes / (float(np.mean(rv_ms)) * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
               "algorithmic_bytes": rv_bytes, "finite": int(torch.isfinite(rvs_box["rv"]).sum().item()),
               "traffic": traffic.get("line_rv_kernel")}
    line_rv["frac"] = line_rv["achieved"] / line_rv["peak"]

    # ---- total, flux-only and CB-only delta spectra (Eq. 1-3): one pass for the three against the total alone and against
    # a pass per effect (SOAP_OPT_EFFECT_PASSES); the workload's facula has a limb-brightening law, so its entries are walked twice
    def effects_leg():
        outs = [torch.empty((n_ph, P), dtype=torch.float32, device=dev) for _ in range(3)]

        def alone():
            soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, outs[0])

        def three():
            soap.soap_active_timeseries_effects(star, q, s, f, wl.regions, wl.phases, outs[0], outs[1], outs[2])

        t_alone = float(np.mean(timer.steps(alone, 5)))
        t_one = float(np.mean(timer.steps(three, 5)))
        soap.soap_set_option(star, soap.binding.SOAP_OPT_EFFECT_PASSES, 1)
        t_per = float(np.mean(timer.steps(three, 5)))
        soap.soap_set_option(star, soap.binding.SOAP_OPT_EFFECT_PASSES, 0)
        return {"total_alone_ms": t_alone, "three_effects_one_pass_ms": t_one, "three_effects_pass_per_effect_ms": t_per,
                "one_pass_over_total_alone": t_one / t_alone, "limb_brightening_laws": {"spot": list(wl.spot_lb), "facula": list(wl.facula_lb)},
                "note": "active map + shift-interpolate-accumulate launch(es) of soap_active_timeseries[_effects], L2 flushed between calls"}

    effects = effects_leg()

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
    if args.form is not None:
        soap.soap_set_option(star2, soap.binding.SOAP_OPT_FORM, args.form)
    e2e_steps = max(3, min(args.steps, 20))
    barrier()
    e2e_list = timer.steps(lambda: soap.soap_synthesize_host(star2, wl, hq, hs, hf, wl.regions, wl.phases, hQ, hD), e2e_steps)
    e2e_ms = sharding.max_over_ranks(float(sum(e2e_list)), dev)
    e2e_value = world * n_spec / (e2e_ms / e2e_steps * 1e-3)
    h2d = 3 * wl.n_mu * pitch * 4 + P * 4
    d2h = n_spec * P * 4
    # the host path computes wavelength chunks (different CTA ranges => different fp64 summation order): equal to rounding
    assert float((hQ.to(dev) - Q).abs().max()) <= 1e-6 * info["sum_weights"]
    assert float((hD.to(dev) - D).abs().max()) <= 1e-5 * float(D.abs().max())

    # the same with the (static) spectra tables resident: a time-series user uploads them once; per step only the region
    # list goes in and the 26 spectra come back to pinned host memory
    def resident_step():
        step()
        hQ.copy_(Q, non_blocking=True)
        hD.copy_(D, non_blocking=True)

    res_list = timer.steps(resident_step, e2e_steps)
    res_ms = sharding.max_over_ranks(float(sum(res_list)), dev) / e2e_steps

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    configs = {} if args.no_configs else config_lines(soap, torch, timer, workloads, dev, args.steps, peak_instr)

    n_vis = info["n_visible"]
    act_cells = int(n_active.sum())
    eff_interps = (n_vis + 2 * act_cells) * P  # what Alg. 1 / Alg. 5 would execute per star
    exec_units = (main_form["quiet_entries"] + main_form["active_entries"]) * P
    form_text = main_form["form"] + (" quiet launch + binned active launch (SOAP_FORM_AUTO)" if main_form["form"] == "composite" else "")
    line = {
        "metric": METRIC, "value": value, "unit": "spectra/s", "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(np.min(step_ms)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD_C3, "stars_per_gpu": 1, "spectra_per_step": n_spec, "form": form_text,
                   "l2": "512 MB buffer written before every timed step (inputs+outputs 106 MB < 126 MB L2)",
                   "timing": "sum of per-step CUDA-event intervals, max over ranks", "sharding": "independent stars per rank, no collective"},
        "cell_pixel_interps_per_s": world * eff_interps / (ms_per_step * 1e-3),
        "executed_lerp_accumulates_per_s": world * exec_units / (ms_per_step * 1e-3),
        "definitional": {"n_visible": n_vis, "active_cells_all_phases": act_cells, "quiet_entries": main_form["quiet_entries"],
                         "active_entries_all_phases": main_form["active_entries"], "columns": wl.grid_n},
        "roofline": roofline, "forms": forms, "fir_form": fir, "lower_resolution": lsf, "line_rvs": line_rv, "effects": effects,
        "configs": configs, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "spectra/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "api": "soap_synthesize_host (pinned host buffers)",
                "tables_resident": {"ms_per_step": res_ms, "value": world * n_spec / (res_ms * 1e-3),
                                    "h2d_bytes_per_step": 48 * len(wl.regions) * n_ph, "d2h_bytes_per_step": d2h,
                                    "note": "spectra tables uploaded once (a time series re-uses them); per step the region centres "
                                            "go in and the 26 spectra are copied to pinned host memory"}},
        "gpu_launches": launches, "wall_s_timed_region": wall,
        "cuda_graph": {"ms_per_step": graph_ms, "note": "the timed step captured once and replayed (4 kernel nodes with programmatic edges)"},
    }
    line["e2e"]["tables_resident_ms"] = res_ms
    line["e2e"]["tables_resident_value"] = world * n_spec / (res_ms * 1e-3)
    flat = {"cuda_graph_ms": graph_ms, "lsf_ms": lsf["ms"], "lsf_hbm_frac": lsf["frac"], "rv_ms": line_rv["ms"], "rv_hbm_frac": line_rv["frac"],
            "effects_one_pass_ratio": effects["one_pass_over_total_alone"], "effects_one_pass_ms": effects["three_effects_one_pass_ms"]}
    if fir is not None:
        flat.update({"fir_step_ms": fir["ms_per_step"], "fir_quiet_ms": fir["quiet_kernel_ms"], "fir_active_ms": fir["active_kernel_ms"],
                     "fir_quiet_hbm_frac": fir["roofline"]["quiet"]["frac"], "fir_active_hbm_frac": fir["roofline"]["active"]["frac"]})
    if "binned" in forms:
        flat.update({"binned_step_ms": forms["binned"]["ms_per_step"], "binned_quiet_ms": forms["binned"]["quiet_kernel_ms"],
                     "binned_quiet_frac": forms["binned"]["quiet_alu_frac"], "binned_active_frac": forms["binned"]["active_alu_frac"]})
    for name, c in configs.items():
        k_ = name.lower()
        flat.update({f"{k_}_ms": c.get("ms_per_step"), f"{k_}_quiet_alu_frac": c.get("quiet_alu_frac"),
                     f"{k_}_active_alu_frac": c.get("active_alu_frac")})
    line.update(flat)
    if world == 1 and not args.no_cpu_baseline:
        t_full, threads = oracle_full(wl)
        t_c2, n_c2 = oracle_single_thread_c2()
        line["cpu_baseline"] = {"value": n_spec / t_full, "unit": "spectra/s", "cores": threads, "kind": "oracle",
                                "sample": "full: all 70688 cells x 310000 px x (1 quiet + 25 phases), one run, measured",
                                "seconds": t_full, "c2_single_thread": {"seconds": t_c2, "spectra_per_s": n_c2 / t_c2, "cores": 1}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_configs(args):
    """--workload C2|C3|C4|C5 (with --vsini / --form): one JSON line with the step time and the two kernels' durations."""
    import torch

    import paper_2301_04259_b200 as soap
    import workloads

    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    peaks = load_peaks()
    peak_instr = N_SM * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6
    flush_buf = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)
    timer = Timer(torch, flush_buf)
    make = {"C2": workloads.make_config2, "C3": workloads.make_config3, "C4": workloads.make_config4,
            "C5": lambda: workloads.make_config5_star(0)}
    wl = make[args.workload]()
    if args.vsini is not None:
        wl.vsini_kms = args.vsini
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    sp = soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    fa = None if wl.facula is None else soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    r, star, _, _ = time_form(soap, torch, timer, wl, q, sp, fa, args.form, max(3, min(args.steps, 10)), dev.index, peak_instr)
    soap.soap_destroy(star)
    r["workload"] = workloads.CONFIG_NAMES[int(args.workload[1])] + (" (first star)" if args.workload == "C5" else "")
    r["vsini_kms"] = float(wl.vsini_kms)
    print(json.dumps(r))


def run_sweep(args):
    """--workload C5 --sweep [--gpus N]: the 64-star parameter sweep as ONE job dealt to the ranks (stars first).

    Rank r owns the contiguous block sharding.shard_range(64, r, N) and runs the three batch calls on it; nothing crosses
    NVLink while it computes.  Total work is fixed, so `scaling` is "strong"; value = 64 x 51 spectra / max-over-ranks
    device time.  Afterwards every star's checksum row (sum of Q, sum of |delta|) is gathered in star order
    (sharding.gather_unit_summaries).  The delta checksums do not depend on how the job was dealt (an item's result does not
    depend on which CTA, launch or rank computes it): `delta_checksums_sha16` must be the same for every N.  The quiet
    spectra agree to an fp32 rounding only (the batch launch groups its fp64 shares by CTA range), so their checksum is
    printed as a number, `quiet_checksum_sum`."""
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
    n_stars = 64
    b, e = sharding.shard_range(n_stars, rank, world)
    shared = workloads.make_config5_star(0)  # the spectra set is shared by all stars: every rank holds it
    wls = [shared if k == 0 else workloads.make_config5_star(k, shared=shared) for k in range(b, e)]
    n, P, n_ph = len(wls), shared.n_pix, len(shared.phases)
    q = soap.to_device_spectra(shared.quiet, shared.lambda0, shared.dlambda, dev)
    sp = soap.to_device_spectra(shared.spot, shared.lambda0, shared.dlambda, dev, shared.spot_contrast, shared.spot_lb)
    fa = soap.to_device_spectra(shared.facula, shared.lambda0, shared.dlambda, dev, shared.facula_contrast, shared.facula_lb)
    stars = [soap.soap_create(local_rank) for _ in wls]
    Q = torch.zeros((max(n, 1), P), dtype=torch.float32, device=dev)
    D = torch.zeros((max(n, 1), n_ph, P), dtype=torch.float32, device=dev)
    flush_buf = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)
    timer = Timer(torch, flush_buf)

    def step():
        if n == 0:
            return
        if n == 1:
            soap.soap_disk_geometry(stars[0], wls[0], want_info=False)
            soap.soap_integrate_quiet(stars[0], q, Q[0])
            soap.soap_active_timeseries(stars[0], q, sp, fa, wls[0].regions, wls[0].phases, D[0])
            return
        soap.soap_batch_disk_geometry(stars, wls)
        soap.soap_batch_integrate_quiet(stars, [q] * n, [Q[k] for k in range(n)])
        soap.soap_batch_active_timeseries(stars, [q] * n, [sp] * n, [fa] * n, [w.regions for w in wls],
                                          [w.phases for w in wls], [D[k] for k in range(n)])

    steps = max(3, min(args.steps, 10))
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ms = timer.steps(step, steps, warm=max(3, args.warmup))
    if world > 1:
        dist.barrier()
    total_ms = sharding.max_over_ranks(float(sum(ms)), dev)
    local = torch.stack([Q[:n].double().sum(dim=1), D[:n].double().abs().sum(dim=(1, 2))], dim=1) if n else torch.zeros((0, 2), dtype=torch.float64, device=dev)
    rows = sharding.gather_unit_summaries(local, n_stars)
    if rank == 0:
        ms_per_step = total_ms / steps
        rows_h = rows.cpu().numpy()
        digest = hashlib.sha256(np.ascontiguousarray(rows_h[:, 1]).tobytes()).hexdigest()[:16]
        print(json.dumps({
            "metric": METRIC, "value": n_stars * (1 + n_ph) / (ms_per_step * 1e-3), "unit": "spectra/s", "n_gpus": world,
            "steps": steps, "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workloads.CONFIG_NAMES[5], "stars": n_stars, "stars_on_rank0": n,
                       "sharding": "contiguous blocks of stars per rank (sharding.shard_range), no data-path collective",
                       "l2": "512 MB buffer written before every timed step"},
            "delta_checksums_sha16": digest, "quiet_checksum_sum": float(rows_h[:, 0].sum()), "stars_gathered": int(rows.shape[0]),
            "checksum_star0": [float(rows_h[0, 0]), float(rows_h[0, 1])]}))
    for s_ in stars:
        soap.soap_destroy(s_)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["graft", "reference"], default="graft")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the C2 / C4 / C5 timings of the `configs` object")
    ap.add_argument("--form", type=int, default=None, help="SOAP_OPT_FORM of the timed star (default: the library's AUTO)")
    ap.add_argument("--vsini", type=float, default=None, help="with --workload: override v sin i (km/s)")
    ap.add_argument("--workload", choices=["C2", "C3", "C4", "C5"], default=None,
                    help="print one per-config timing line instead of the bench contract (which is C3)")
    ap.add_argument("--sweep", action="store_true",
                    help="with --workload C5: the 64 stars as one job dealt to the --gpus ranks (strong scaling), one JSON line")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "C5" and args.sweep:
        run_sweep(args)
    elif args.workload is not None:
        run_configs(args)
    else:
        run_graft(args)


if __name__ == "__main__":
    main()
