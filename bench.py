#!/usr/bin/env python
"""bench.py -- throughput of the FDAS hot path on B200 (one step = one DM trial: prepare_spectrum ->
convolve_plane -> harmonic_sum_peaks on one synthetic SKA-like time series).

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores

Prints ONE JSON line (rank 0).  `value` = f-fdot plane points per second with the series resident in
HBM; `e2e` = the same through fdas_search_host with the series in pinned host memory (H2D + D2H
inside the timed region).  DM trials are independent, so N > 1 is N replicas on sharded trials
(weak scaling, no data-path collective).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import math
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "f-fdot plane points/s (SKA-like DM trial: real FFT + whitening + 193-template convolve+power + 16-harmonic sum/peaks)"
UNIT = "points/s"

# Algorithmic work of K2 per (segment, template) and per plane point -- DESIGN.md "Kernels / K2".
L_SEG = 2048
FLOP_IFFT = 5 * L_SEG * 11          # 5 L log2 L
FLOP_MUL = 6 * L_SEG
HBM_BYTES_PER_POINT = {"fp32": 4.05, "bf16": 4.02, "bf16_plane16": 2.02, "bf16_tc": 4.02, "bf16_tc_plane16": 2.02}
# ALU peak: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md unit counts/clocks)
N_SM, LANES, SM_MAX_GHZ = 148, 128, 1.965
ALU_PEAK_TFLOPS = N_SM * LANES * 2 * SM_MAX_GHZ / 1e3
TC_PRECISIONS = ("bf16_tc", "bf16_tc_plane16")
PROFILES = os.path.join(ROOT, "profiles")


# counters of an `ncu --set full` capture kept beside the DRAM traffic (write_traffic_json)
COUNTER_PREFIXES = ("sm__pipe_tensor_cycles_active", "sm__pipe_fma_cycles_active", "sm__pipe_alu_cycles_active",
                    "sm__pipe_fmaheavy_cycles_active", "smsp__issue_active", "l1tex__data_pipe_lsu_wavefronts.",
                    "l1tex__data_pipe_lsu_wavefronts_mem_shared.", "smsp__inst_executed.sum", "sm__warps_active",
                    "launch__registers_per_thread", "gpu__dram_throughput", "sm__throughput", "dram__throughput",
                    "sm__cycles_active.avg", "smsp__cycles_active.avg")


def ncu_traffic(workload: str, precision: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE K2 launch, from the committed
    profiles/*_traffic.json files (written by `bench.py --traffic-from-ncu` out of an `ncu --set full`
    capture; each names its kernel, command and commit).  The newest matching record wins; None if no
    capture exists for this (workload, precision)."""
    best = None
    try:
        names = sorted(f for f in os.listdir(PROFILES) if f.endswith("_traffic.json"))
    except OSError:
        return None
    for f in names:
        try:
            for rec in json.load(open(os.path.join(PROFILES, f)))["records"]:
                if rec["workload"] == workload and rec["precision"] == precision:
                    best = dict(rec, file="profiles/" + f)
        except Exception:
            continue
    return best


def write_traffic_json(rep: str, out: str, workload: str, precision: str, command: str):
    """`ncu -i rep --page raw --csv` -> profiles/<run>_traffic.json (appends one record per launch)."""
    import csv
    import subprocess
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units = rows[0], rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    commit = subprocess.run(["git", "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    recs = []
    for r in rows[2:]:
        def val(k):
            return float(r[hdr.index(k)]) * scale.get(units[hdr.index(k)], 1.0)
        rd, wr = val("dram__bytes_read.sum"), val("dram__bytes_write.sum")
        counters = {}
        for i, name in enumerate(hdr):
            if name.startswith(COUNTER_PREFIXES) and not any(t in name for t in (".max.", ".min.", ".sum.pct_of_peak", ".sum.per_cycle")):
                try:
                    counters[name] = [float(r[i].replace(",", "")), units[i]]
                except ValueError:
                    pass
        recs.append({"kernel": r[hdr.index("Kernel Name")], "workload": workload, "precision": precision,
                     "dram_bytes_read": rd, "dram_bytes_write": wr, "traffic": rd + wr, "counters": counters,
                     "duration_us_under_ncu": float(r[hdr.index("gpu__time_duration.sum")]) *
                     {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}[units[hdr.index("gpu__time_duration.sum")]],
                     "command": command,
                     "commit": commit})
    doc = {"records": []}
    if os.path.exists(out):
        doc = json.load(open(out))
    doc["records"] += recs
    json.dump(doc, open(out, "w"), indent=1)
    print(f"wrote {len(recs)} record(s) to {out}")


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


def measured_tensor_peak():
    """Dense bf16 TFLOP/s (cuBLAS burst figure: K2 is timed alone per launch), else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["bf16_tflops"]), "measured"
        except Exception:
            pass
    return 1590.0, "fallback"


def tc_mma_flops(info):
    """Tensor-core flops one K2-TC launch issues (padded operand shapes, K2-TC): per tile of
    128 bins 4 sub-tiles x ceil((2h+1)/16) K-steps x 2 bank images (Re T, Im T) of a 128 x 64 x 16 MMA
    (M = 128 template-pair lanes, N = 32 bins x {re, im})."""
    kp = (2 * int(info.halfwidth) + 1 + 15) // 16 * 16
    ntiles = int(info.nbins) // 128
    return ntiles * 4 * (kp // 16) * 2 * (2 * 128 * 64 * 16)


def workload_string(wl):
    """The same text in both arms' config.workload (the arms differ in config.precision / impl)."""
    return (f"{wl.name}: N={wl.n} samples at {wl.tsamp * 1e6:.0f} us, nfft={wl.nfft}, nz={wl.nz} (zmax={wl.zmax:g}, "
            f"zstep={wl.zstep:g}), seg_len={wl.seg_len}, H={wl.nharm}, {wl.nsigma:g} sigma, r_lo={wl.r_lo}")


def workload_for(name: str, inputs):
    if name == "ska":
        return inputs.ska()
    if name == "ska_half":
        return inputs.ska(half_res=True)
    if name == "ska_padded":
        return inputs.ska_padded()
    if name == "medium":
        return inputs.medium()
    if name == "tiny":
        return inputs.tiny()
    raise SystemExit(f"unknown workload {name}")


def trial_series(wl_name, trial, inputs):
    """Distinct seeded series per trial: configs[3] members for the SKA shapes."""
    if wl_name in ("ska", "ska_half"):
        w = inputs.batched_member(trial % 64, half_res=(wl_name == "ska_half"))
        if trial == 0:
            w = workload_for(wl_name, inputs)      # trial 0 is configs[2] itself (2 injected pulsars)
        return inputs.series_for(w)
    w = workload_for(wl_name, inputs)
    if wl_name == "ska_padded":
        return inputs.series_for(inputs.ska_padded(seed=3 + 7919 * trial))
    return inputs.make_series(w.n, w.seed + 7919 * trial, w.signals, w.red_knee)


class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons through NVML while the timed region runs; every sample
    carries its host time (time.perf_counter) so that it can be paired with CUDA-event times."""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.power, self.t = period, [], set(), [], []
        self.stop_flag = threading.Event()
        self.ok = False
        self.power_kind = "nvmlDeviceGetPowerUsage"
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
            self.instant = getattr(pynvml, "NVML_FI_DEV_POWER_INSTANT", None)
            if self.instant is not None and self._instant_power() is None:
                self.instant = None
            if self.instant is not None:
                self.power_kind = "NVML_FI_DEV_POWER_INSTANT"
        except Exception as e:   # no NVML: clocks are reported as unavailable
            self.err = repr(e)
            self.sm_max = None

    def _instant_power(self):
        try:
            v = self.nv.nvmlDeviceGetFieldValues(self.h, [self.instant])[0]
            if int(v.nvmlReturn) != 0:
                return None
            mw = float(v.value.uiVal)
            return mw / 1000.0 if mw > 0 else None
        except Exception:
            return None

    def energy_mj(self):
        try:
            return int(self.nv.nvmlDeviceGetTotalEnergyConsumption(self.h))
        except Exception:
            return None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown",
        }
        while not self.stop_flag.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                watts = self._instant_power() if self.instant is not None else None
                if watts is None:
                    watts = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.t.append(time.perf_counter())
                self.samples.append(mhz)
                self.power.append(watts)
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": int(statistics.median(self.samples)), "sm_max_mhz": self.sm_max,
                "sm_mhz_min": min(self.samples), "sm_mhz_max_seen": max(self.samples),
                "reasons": sorted(self.reasons), "power_w_mean": round(sum(self.power) / len(self.power), 1),
                "samples": len(self.samples)}


def sustained_loop(step, stream, torch, n_e, local_rank, every=16):
    """`n_e` identical steps back to back (seconds long: the NVML energy counter needs that, and the board
    settles at its power cap): J and ms per step, and -- from four CUDA events on every `every`-th step -- the
    per-call split of the SUSTAINED step and a table of step time, power and J per step binned by the SM clock
    NVML reported nearest to that step (the clock axis this pool allows: the power cap walks the clock by itself;
    locking clocks is unavailable here)."""
    es = ClockSampler(local_rank, period=0.01)
    if not es.ok:
        return None
    marks = list(range(0, n_e, every)) if every > 0 else []
    evs = {i: [torch.cuda.Event(enable_timing=True) for _ in range(4)] for i in marks}
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    es.start()
    j0 = es.energy_mj()
    t_host0 = time.perf_counter()
    ev0.record(stream)
    for i in range(n_e):
        step(i, evs.get(i))
    ev1.record(stream)
    torch.cuda.synchronize()
    j1 = es.energy_mj()
    es.stop_flag.set()
    es.join(timeout=2.0)
    sec = ev0.elapsed_time(ev1) * 1e-3
    if j0 is None or j1 is None or j1 <= j0:
        return None
    if not marks:    # a loop of one call only (energy_by_kernel): no per-step split
        return {"joules_per_step": (j1 - j0) / 1e3 / n_e, "mean_power_w": (j1 - j0) / 1e3 / sec, "steps": n_e,
                "seconds": sec, "ms_per_step": 1e3 * sec / n_e, "clocks": es.summary()}
    rows = []
    ts = np.array(es.t) - t_host0
    for i in marks:
        e = evs[i]
        rows.append((ev0.elapsed_time(e[0]) * 1e-3, e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2]),
                     e[2].elapsed_time(e[3])))
    rows = np.array(rows)
    out = {"joules_per_step": (j1 - j0) / 1e3 / n_e, "mean_power_w": (j1 - j0) / 1e3 / sec,
           "steps": n_e, "seconds": sec, "ms_per_step": 1e3 * sec / n_e,
           "source": "NVML total energy counter over a separate, sustained loop of identical steps",
           "kernel_ms_sustained": {"prepare_spectrum": float(rows[:, 1].mean()), "convolve_plane": float(rows[:, 2].mean()),
                                   "harmonic_sum_peaks": float(rows[:, 3].mean()),
                                   "sampled_steps": int(len(rows)), "every": every,
                                   "second_half": {"prepare_spectrum": float(rows[len(rows) // 2:, 1].mean()),
                                                   "convolve_plane": float(rows[len(rows) // 2:, 2].mean()),
                                                   "harmonic_sum_peaks": float(rows[len(rows) // 2:, 3].mean())}},
           "clocks": es.summary()}
    if len(ts) >= 2:
        mhz, watts = np.array(es.samples, dtype=float), np.array(es.power, dtype=float)
        near = np.abs(rows[:, 0][:, None] - ts[None, :]).argmin(axis=1)
        bins = {}
        for r, k in zip(rows, near):
            bins.setdefault(int(round(mhz[k] / 50.0) * 50), []).append((r[1] + r[2] + r[3], r[2], watts[k]))
        table = []
        for b in sorted(bins, reverse=True):
            a = np.array(bins[b])
            table.append({"sm_mhz": b, "n": int(len(a)), "ms_per_step": round(float(a[:, 0].mean()), 4),
                          "convolve_plane_ms": round(float(a[:, 1].mean()), 4), "power_w": round(float(a[:, 2].mean()), 1),
                          "joules_per_step": round(float(a[:, 0].mean() * a[:, 2].mean()) * 1e-3, 4)})
        out["clock_bins"] = {"bin_mhz": 50, "power": es.power_kind, "rows": table,
                             "note": "every 16th step of the sustained loop, paired with the NVML (SM MHz, W) sample "
                                     "nearest in time; J per step = W x ms of that bin.  The clock moves only as the "
                                     "1000 W cap moves it (locked clocks: unavailable on this pool)"}
    return out


# ------------------------------------------------------------------------------- CPU oracle arm
def oracle_sample(x, wl, budget_s=12.0):
    """Times the oracle, as it stands, on a bounded sample of one trial: O1+O2 on the whole series
    (prorated to the sample), O4 plane and O5/O6 harmonic sums + candidates over the first R bins
    of all nz rows.  Returns (points_per_s, cores, description, seconds)."""
    from oracle import fdas_oracle as orc
    t0 = time.perf_counter()
    X = orc.spectrum(x, wl.nfft)
    w = orc.whiten(X)
    t_spec = time.perf_counter() - t0
    bank = orc.template_bank(wl.zmax, wl.zstep)          # plan-time work, not counted
    nb = wl.nfft // 2
    nz = bank.shape[0]
    R = min(nb, 4096)
    t0 = time.perf_counter()
    orc.plane(w, bank, 0, R)
    t_probe = time.perf_counter() - t0
    R = int(min(nb, max(R, R * budget_s / max(t_probe, 1e-3))))
    R = max(4096, (R // 4096) * 4096)
    t0 = time.perf_counter()
    P = orc.plane(w, bank, 0, R)
    t_plane = time.perf_counter() - t0
    thr = orc.thresholds(wl.nharm, wl.nsigma)
    t0 = time.perf_counter()
    orc.candidates(P, wl.nharm, thr, min(wl.r_lo, R - 1))
    t_harm = time.perf_counter() - t0
    total = t_spec * (R / nb) + t_plane + t_harm
    desc = (f"oracle O1+O2 on the full {wl.nfft}-sample series (prorated by R/Nb), O4 plane and O5/O6 "
            f"harmonic sums over the first R={R} of {nb} bins x {nz} templates")
    return nz * R / total, orc.num_threads(), desc, total + t_spec * (1 - R / nb)


def run_reference(args):
    from paper_2211_13517_b200 import inputs
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = workload_for(args.workload, inputs)
    x = trial_series(args.workload, 0, inputs)
    budget = max(2.0, min(15.0, 120.0 / max(1, args.steps + args.warmup)))
    vals, secs = [], []
    cores, desc = 0, ""
    for i in range(args.warmup + args.steps):
        v, cores, desc, s = oracle_sample(x, wl, budget)
        if i >= args.warmup:
            vals.append(v)
            secs.append(s)
    value = len(vals) / sum(1.0 / v for v in vals)
    nb = wl.nfft // 2
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * wl.nz * nb / value, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(wl), "precision": "f64 (CPU oracle)",
                   "note": "ms_per_step is the oracle's time for a whole trial extrapolated from the sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------- CUDA arm
def time_path(plan, fdas, torch, wl, dev_pool, thr, steps, warmup, energy_seconds, local_rank, barrier,
              want_modes=True):
    """`steps` DM trials (prepare_spectrum -> convolve_plane -> harmonic_sum_peaks) of one plan on resident
    series: CUDA events on the launching stream around every call, NVML clocks during the timed region,
    and a second, seconds-long loop of the same steps for the energy per trial (the NVML counter needs
    seconds; that loop also shows the sustained step time)."""
    dev = dev_pool[0].device
    d_spec, d_plane = plan.alloc_spec(dev), plan.alloc_plane(dev)
    d_c, d_n = plan.alloc_cands(1 << 16, dev)
    stream = torch.cuda.current_stream()
    pool_n = len(dev_pool)

    def step(i, evs=None):
        x = dev_pool[i % pool_n]
        if evs is not None:
            evs[0].record(stream)
        plan.prepare_spectrum(x, d_spec, stream)
        if evs is not None:
            evs[1].record(stream)
        plan.convolve_plane(d_spec, d_plane, stream)
        if evs is not None:
            evs[2].record(stream)
        plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n, stream)
        if evs is not None:
            evs[3].record(stream)

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    n_cands = int(d_n.item())
    sampler = ClockSampler(local_rank, period=0.001)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    launches0 = plan.launch_count()
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    for i in range(steps):
        step(i, evs[i])
    torch.cuda.synchronize()
    sampler.stop_flag.set()
    barrier()
    t_total_ms = evs[0][0].elapsed_time(evs[-1][3])
    launches = plan.launch_count() - launches0
    sampler.join(timeout=2.0)
    res = {
        "total_ms": t_total_ms, "ms_per_step": t_total_ms / steps, "launches": launches, "candidates_last_step": n_cands,
        "kernel_ms": {"prepare_spectrum": statistics.mean(e[0].elapsed_time(e[1]) for e in evs),
                      "convolve_plane": statistics.mean(e[1].elapsed_time(e[2]) for e in evs),
                      "harmonic_sum_peaks": statistics.mean(e[2].elapsed_time(e[3]) for e in evs)},
        "clocks": sampler.summary(), "energy": None,
    }
    if sampler.ok and energy_seconds > 0:
        n_e = max(steps, int(energy_seconds * 1e3 / max(res["ms_per_step"], 1e-3)) + 1)
        res["energy"] = sustained_loop(step, stream, torch, n_e, local_rank)
    if not want_modes:
        res["buffers"] = (d_spec, d_plane)
        return res
    if res["energy"] is not None and energy_seconds > 0:
        # where the watts go (the sustained regime is power-bound): each call ALONE in its own seconds-long loop
        calls = {"prepare_spectrum": lambda i, evs=None: plan.prepare_spectrum(dev_pool[i % pool_n], d_spec, stream),
                 "convolve_plane": lambda i, evs=None: plan.convolve_plane(d_spec, d_plane, stream),
                 "harmonic_sum_peaks": lambda i, evs=None: plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo,
                                                                                  d_c, d_n, stream)}
        by = {}
        for name, fn in calls.items():
            n_k = int(energy_seconds * 1e3 / max(res["kernel_ms"][name], 1e-3)) + 1
            e = sustained_loop(fn, stream, torch, n_k, local_rank, every=0)
            if e is not None:
                by[name] = {"ms_per_call": e["ms_per_step"], "joules_per_call": e["joules_per_step"],
                            "mean_power_w": e["mean_power_w"], "sm_mhz": e["clocks"].get("sm_mhz"),
                            "reasons": e["clocks"].get("reasons"), "calls": e["steps"]}
        if len(by) == 3:
            by["sum_joules"] = sum(by[k]["joules_per_call"] for k in calls)
            by["step_joules"] = res["energy"]["joules_per_step"]
            by["note"] = ("each call of the step repeated alone for the same number of seconds (its own clock / power "
                          "equilibrium); the sum against the J of the whole step in the sustained loop")
            res["energy_by_kernel"] = by
    # both harmonic-sum modes on the plane of the last step: K3 alone, 10 launches each
    modes = {}
    for mode in ("plain", "neighbour_max"):
        plan.set_harmonic_mode(mode)
        t = thr if mode == "plain" else nbr_thresholds(thr)
        for _ in range(2):
            plan.harmonic_sum_peaks(d_plane, wl.nharm, t, wl.r_lo, d_c, d_n, stream)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(10):
            plan.harmonic_sum_peaks(d_plane, wl.nharm, t, wl.r_lo, d_c, d_n, stream)
        b.record(stream)
        torch.cuda.synchronize()
        modes[mode] = {"harmonic_sum_peaks_ms": a.elapsed_time(b) / 10, "candidates": int(d_n.item())}
    plan.set_harmonic_mode("plain")
    modes["note"] = ("neighbour_max: S'_h = sum_k max_{|d| <= k/2} P[k z][k r + d] (DESIGN.md reading A24), thresholds "
                     "= the plain ones raised by the growth of the noise mean")
    res["harmonic_modes"] = modes
    res["k3_stress"] = k3_stress(plan, fdas, torch, wl, d_plane, d_c, d_n, stream,
                                 res["kernel_ms"]["harmonic_sum_peaks"], n_cands)
    res["buffers"] = (d_spec, d_plane)
    return res


def k3_stress(plan, fdas, torch, wl, d_plane, d_c, d_n, stream, base_ms, base_cands):
    """K3 is a data-dependent branch-and-bound: the timed inputs (noise, about one candidate per trial at 6 sigma)
    are its best case.  The same kernel on the last step's plane under conditions that are not: thresholds low
    enough to list many fundamentals, low enough to overflow the prefilter's list (exact full scan), and a plane
    with RFI-like columns far above the saturation value of the block-max codes (127.875)."""
    def timed(thr, n):
        plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n, stream)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n):
            plan.harmonic_sum_peaks(d_plane, wl.nharm, thr, wl.r_lo, d_c, d_n, stream)
        b.record(stream)
        torch.cuda.synchronize()
        return {"harmonic_sum_peaks_ms": a.elapsed_time(b) / n, "candidates": int(d_n.item())}

    out = {"baseline_6_sigma": {"harmonic_sum_peaks_ms": base_ms, "candidates": base_cands}}
    for ns in (4.0, 3.0, 2.0):
        out[f"threshold_{ns:g}_sigma"] = timed(fdas.thresholds_from_sigma(wl.nharm, ns), 3)
    # RFI: 0.5 % of the columns (seeded) multiplied by 1000, in place; the block maxima are then rebuilt from the
    # plane on every call (fdas_plan_invalidate_plane), which is part of the time below
    g = torch.Generator(device="cpu")
    g.manual_seed(2211)
    nb = int(plan.info.nbins)
    cols = torch.randperm(nb, generator=g)[: nb // 200].to(d_plane.device)
    d_plane[:, cols] = d_plane[:, cols] * 1000.0
    plan.invalidate_plane()
    out["rfi_columns_6_sigma"] = dict(timed(fdas.thresholds_from_sigma(wl.nharm, wl.nsigma), 3),
                                      columns=int(cols.numel()), includes="the rebuild of the block maxima from the plane")
    out["note"] = ("candidate capacity 65536: `candidates` is the true count, only the first 65536 are stored and flagged; "
                   "2 sigma overflows the 2^22-entry prefilter list, so pass B scans every fundamental")
    return out


def nbr_thresholds(thr):
    """Thresholds for the neighbour-maximised sums in this benchmark: T_h + sum_{k<=h} (H_m - 1), m = 2 (k/2) + 1,
    H_m = mean of the maximum of m unit exponentials (the caller's choice; the library takes any)."""
    out, shift = [], 0.0
    for k, t in enumerate(thr, start=1):
        m = 2 * (k // 2) + 1
        shift += sum(1.0 / i for i in range(1, m + 1)) - 1.0
        out.append(t + shift)
    return np.array(out, dtype=np.float32)


def k2_rooflines(info, precision, workload, t_conv_ms, t_conv_sustained_ms=None, sustained_clocks=None):
    """The convolve kernel of one path against its binding roof and against HBM (north_star's yardstick).
    `t_conv_sustained_ms`: the same launch timed inside the seconds-long, power-capped loop (every 16th step)."""
    points = int(info.nz) * int(info.nbins)
    hbm_peak, peak_kind = measured_peaks()
    gbs = HBM_BYTES_PER_POINT[precision] * points / (t_conv_ms * 1e-3) / 1e9
    traffic = ncu_traffic(workload, precision)
    hbm = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
           "launch_ms": t_conv_ms,
           "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json)",
           "bytes_per_point": HBM_BYTES_PER_POINT[precision], "bytes_per_launch": HBM_BYTES_PER_POINT[precision] * points,
           "frac_of_8TBs_nominal": gbs / 8000.0,
           "traffic": None if traffic is None else traffic["traffic"],
           "traffic_source": None if traffic is None else {k: traffic[k] for k in ("file", "kernel", "commit", "command")}}
    if t_conv_sustained_ms:
        gbs_s = HBM_BYTES_PER_POINT[precision] * points / (t_conv_sustained_ms * 1e-3) / 1e9
        hbm.update({"launch_ms_sustained": t_conv_sustained_ms, "achieved_sustained": gbs_s,
                    "frac_sustained": gbs_s / hbm_peak,
                    "sustained_note": "the same launch inside the seconds-long loop of identical steps (board at its "
                                      "power cap; CUDA events around every 16th step)",
                    "sustained_clocks": sustained_clocks})
    if precision in TC_PRECISIONS:
        tpeak, tkind = measured_tensor_peak()
        tflops = tc_mma_flops(info) / (t_conv_ms * 1e-3) / 1e12
        main = dict(hbm, kernel="K2-TC convolve_tc_kernel",
                    tensor={"achieved": tflops, "peak": tpeak, "unit": "TFLOP/s", "frac": tflops / tpeak,
                            "peak_kind": f"{tkind} cuBLAS bf16 burst", "flops_per_launch": tc_mma_flops(info)})
    else:
        flops = int(info.nseg) * (int(info.nz) * (FLOP_IFFT + FLOP_MUL + 3 * int(info.valid)) + FLOP_IFFT)
        tflops = flops / (t_conv_ms * 1e-3) / 1e12
        main = {"kernel": "K2 convolve_kernel", "bound": "alu", "achieved": tflops, "peak": ALU_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": tflops / ALU_PEAK_TFLOPS,
                "peak_kind": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz", "flops_per_launch": flops,
                "launch_ms": t_conv_ms,
                "traffic": hbm["traffic"], "traffic_source": hbm["traffic_source"]}
        if t_conv_sustained_ms:
            main.update({"launch_ms_sustained": t_conv_sustained_ms,
                         "achieved_sustained": flops / (t_conv_sustained_ms * 1e-3) / 1e12,
                         "frac_sustained": flops / (t_conv_sustained_ms * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                         "sustained_clocks": sustained_clocks})
    return main, dict(hbm, kernel=main["kernel"])


def sustained_of(m):
    """(K2 launch ms inside the sustained loop, that loop's clocks) of a time_path result, or (None, None)."""
    e = m.get("energy")
    if not e or "kernel_ms_sustained" not in e:
        return None, None
    return e["kernel_ms_sustained"]["convolve_plane"], e.get("clocks")


def seg_len_sweep(fdas, torch, wl, precision, d_x, launches=10):
    """K2 (FFT formulation) alone at every segment length the kernel is built for: ms per launch by CUDA
    events, the segmentation, and the nominal flop count per plane point of that L."""
    out = []
    for L in (1024, 2048, 4096):
        plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, L, precision)
        info = plan.info
        d_spec, d_plane = plan.alloc_spec(), plan.alloc_plane()
        plan.prepare_spectrum(d_x, d_spec)
        for _ in range(3):
            plan.convolve_plane(d_spec, d_plane)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(launches):
            plan.convolve_plane(d_spec, d_plane)
        b.record()
        torch.cuda.synchronize()
        V = int(info.valid)
        flop_pt = (5.0 * L * math.log2(L) + 6.0 * L + 3.0 * V) / V
        out.append({"seg_len": L, "valid": V, "nseg": int(info.nseg), "threads_per_cta": L // 16,
                    "convolve_plane_ms": a.elapsed_time(b) / launches, "flop_per_point": round(flop_pt, 1)})
        del d_spec, d_plane
        plan.close()
        torch.cuda.empty_cache()
    return out


def survey_block(fdas, torch, inputs, precision, trials_each, pool, thr, local_rank):
    """configs[4]: DM trials of each resolution (64 us: N = 9,375,000; 128 us: N = 4,687,500) through
    fdas_search_batch from PINNED HOST memory (the H2D copy of every series and the D2H of every candidate list
    inside the timed region); series cycle a resident host pool.  trials_each < 0: the paper's counts, 3050 + 2875."""
    stream = torch.cuda.current_stream()
    cap = 1 << 12
    full = trials_each < 0
    counts_of = {False: inputs.SURVEY_TRIALS_FULL if full else trials_each,
                 True: inputs.SURVEY_TRIALS_HALF if full else trials_each}
    out = {"api": "fdas_search_batch, pinned host series in, candidates on the host out", "precision": precision,
           "trials": [counts_of[False], counts_of[True]], "whole_survey": full, "shapes": [],
           "note": f"the paper's survey is {inputs.SURVEY_TRIALS_FULL} + {inputs.SURVEY_TRIALS_HALF} trials "
                   f"(PAPER.md:35, BASELINE.json configs[4]); this block runs {counts_of[False]} + {counts_of[True]}, "
                   f"the {pool} distinct seeded series of each shape cycled.  The inputs are noise with at most one weak "
                   "signal (about one candidate per trial at 6 sigma): K3's branch-and-bound is at its best case here, "
                   "see `k3_stress` for planes that are not"}
    sampler = ClockSampler(local_rank, period=0.05)
    plans = []
    for half in (False, True):
        trials_each = counts_of[half]
        wl = inputs.ska(half_res=half)
        plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
        host = []
        for i in range(pool):
            ht = torch.empty(wl.n, dtype=torch.float32).pin_memory()
            ht.numpy()[:] = inputs.series_for(inputs.batched_member(i, half_res=half))
            host.append(ht)
        buf = np.empty((trials_each, cap), dtype=fdas.CAND_DTYPE)
        series = [host[i % pool] for i in range(trials_each)]
        plan.search_batch(series[:4], wl.nharm, thr, wl.r_lo, capacity=cap, out=buf, stream=stream)   # workspace + warm-up
        plans.append((wl, plan, series, buf))
    torch.cuda.synchronize()
    sampler.start()
    j0 = sampler.energy_mj() if sampler.ok else None
    t_all0 = time.perf_counter()
    for wl, plan, series, buf in plans:
        trials_each = len(series)
        t0 = time.perf_counter()
        counts, _, st = plan.search_batch(series, wl.nharm, thr, wl.r_lo, capacity=cap, out=buf, stream=stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        assert st in (fdas.FDAS_OK, fdas.FDAS_EOVERFLOW), st
        out["shapes"].append({"workload": workload_string(wl), "trials": trials_each, "seconds": dt,
                              "ms_per_trial": 1e3 * dt / trials_each,
                              "points_per_s": trials_each * int(plan.info.nz) * int(plan.info.nbins) / dt,
                              "h2d_bytes_per_trial": int(plan.info.nfft) * 4,
                              "candidates_per_trial": float(counts.mean())})
    total = time.perf_counter() - t_all0
    j1 = sampler.energy_mj() if sampler.ok else None
    sampler.stop_flag.set()
    sampler.join(timeout=2.0)
    ntot = counts_of[False] + counts_of[True]
    out["total_seconds"] = total
    out["ms_per_trial"] = 1e3 * total / ntot
    if j0 is not None and j1 is not None and j1 > j0:
        out["joules_per_trial"] = (j1 - j0) / 1e3 / ntot
        out["joules_total"] = (j1 - j0) / 1e3
        out["mean_power_w"] = (j1 - j0) / 1e3 / total
    if full:
        out["survey_total_s"] = total          # measured: every one of the 5925 trials was run
    else:
        out["survey_total_s_extrapolated"] = (inputs.SURVEY_TRIALS_FULL * out["shapes"][0]["ms_per_trial"]
                                              + inputs.SURVEY_TRIALS_HALF * out["shapes"][1]["ms_per_trial"]) * 1e-3
    out["clocks"] = sampler.summary()
    for _, plan, _, _ in plans:
        plan.close()
    return out


def run_cuda(args):
    import torch
    from paper_2211_13517_b200 import dist as fd, fdas, inputs

    ctx = fd.init_from_env("nccl")
    torch.cuda.set_device(ctx.local_rank)
    dev = torch.device("cuda", ctx.local_rank)
    wl = workload_for(args.workload, inputs)
    precision = args.precision
    plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
    info = plan.info
    points = int(info.nz) * int(info.nbins)

    # seeded pool of distinct series for this rank's trials (trial t -> pool[t % pool])
    pool_n = max(1, min(args.pool, args.steps))
    my_trials = [ctx.rank + ctx.world * i for i in range(pool_n)]
    host_pool = []
    for t in my_trials:
        ht = torch.empty(wl.n, dtype=torch.float32).pin_memory()
        ht.numpy()[:] = trial_series(args.workload, t, inputs)
        host_pool.append(ht)
    dev_pool = [h.to(dev, non_blocking=False) for h in host_pool]
    pool_bytes = pool_n * wl.n * 4
    cap = 1 << 16
    thr = fdas.thresholds_from_sigma(wl.nharm, wl.nsigma)
    stream = torch.cuda.current_stream()

    m = time_path(plan, fdas, torch, wl, dev_pool, thr, args.steps, args.warmup, args.energy_seconds,
                  ctx.local_rank, lambda: fd.barrier(ctx))
    d_spec, d_plane = m.pop("buffers")
    t_max_ms = fd.max_over_ranks(ctx, m["total_ms"])
    total_points = fd.sum_over_ranks(ctx, float(points * args.steps))
    value = total_points / (t_max_ms * 1e-3)
    launches_total = int(fd.sum_over_ranks(ctx, int(m["launches"])))

    # ---- end to end through the public API: pinned host series in, candidates on the host out, every
    # step.  fdas_search_batch is the call a user with many DM trials makes (the H2D copy of trial t+1
    # and the harmonic sum of trial t-1 overlap the convolution of trial t); fdas_search_host, one
    # synchronous trial per call, is timed beside it.
    e2e_steps = max(2, min(args.steps, args.e2e_steps))
    out = np.empty(cap, dtype=fdas.CAND_DTYPE)
    thr_c = thr.ctypes.data_as(C.POINTER(C.c_float))
    sp = int(stream.cuda_stream)
    for i in range(min(3, args.warmup)):
        plan.search_host_raw(host_pool[i % pool_n].data_ptr(), wl.nharm, thr_c, wl.r_lo, out.ctypes.data, cap, sp)
    fd.barrier(ctx)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        st, _cnt = plan.search_host_raw(host_pool[i % pool_n].data_ptr(), wl.nharm, thr_c, wl.r_lo,
                                        out.ctypes.data, cap, sp)
        assert st in (fdas.FDAS_OK, fdas.FDAS_EOVERFLOW), st
    torch.cuda.synchronize()
    t_sync = fd.max_over_ranks(ctx, time.perf_counter() - t0)
    e2e_sync_value = fd.sum_over_ranks(ctx, float(points * e2e_steps)) / t_sync

    bcap = 4096
    bout = np.empty((e2e_steps, bcap), dtype=fdas.CAND_DTYPE)
    series = [host_pool[i % pool_n] for i in range(e2e_steps)]
    plan.search_batch(series[:2], wl.nharm, thr, wl.r_lo, capacity=bcap, out=bout, stream=stream)   # workspace
    fd.barrier(ctx)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    counts, _, st = plan.search_batch(series, wl.nharm, thr, wl.r_lo, capacity=bcap, out=bout, stream=stream)
    torch.cuda.synchronize()
    t_e2e = fd.max_over_ranks(ctx, time.perf_counter() - t0)
    e2e_value = fd.sum_over_ranks(ctx, float(points * e2e_steps)) / t_e2e
    d2h = int(np.minimum(counts, bcap).sum()) * 16 + 8 * e2e_steps
    del d_spec, d_plane
    plan.close()
    torch.cuda.empty_cache()

    is_tc = precision in TC_PRECISIONS
    roofline, roofline_hbm = k2_rooflines(info, precision, args.workload, m["kernel_ms"]["convolve_plane"], *sustained_of(m))

    # ---- beside the tensor-core path: north_star's literal kernel (overlap-save FFT, bf16 storage, fp32
    # arithmetic, no tensor cores) as a FULL record in the same run: step, kernel split, energy, rooflines
    fft_path = None
    if is_tc and not args.no_fft_path and ctx.world == 1:
        fprec = "bf16_plane16" if precision.endswith("plane16") else "bf16"
        plan_f = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, fprec)
        mf = time_path(plan_f, fdas, torch, wl, dev_pool, thr, args.steps, args.warmup, args.energy_seconds,
                       ctx.local_rank, lambda: None, want_modes=False)
        mf.pop("buffers")
        rf, rf_hbm = k2_rooflines(plan_f.info, fprec, args.workload, mf["kernel_ms"]["convolve_plane"], *sustained_of(mf))
        fft_path = {"precision": fprec,
                    "kernel": "K2 convolve_kernel (overlap-save FFT, bf16 storage, fp32 arithmetic, no tensor cores): "
                              "north_star's literal convolve+power kernel",
                    "value": points * args.steps / (mf["total_ms"] * 1e-3), "unit": UNIT,
                    "ms_per_step": mf["ms_per_step"], "kernel_ms": mf["kernel_ms"], "energy": mf["energy"],
                    "gpu_launches": int(mf["launches"]), "candidates_last_step": mf["candidates_last_step"],
                    "roofline": rf, "roofline_hbm": rf_hbm, "clocks": mf["clocks"],
                    "ncu_counters": None if rf.get("traffic_source") is None else
                    dict(ncu_traffic(args.workload, fprec).get("counters") or {}, file=rf["traffic_source"]["file"])}
        plan_f.close()
        torch.cuda.empty_cache()
        # the same kernel at the other segment lengths (K2 alone, 10 launches each, same
        # spectrum; flop per plane point 5 L log2 L / (L - 2h) has its minimum near L = 1024-2048 for 129 taps)
        fft_path["seg_len_sweep"] = seg_len_sweep(fdas, torch, wl, fprec, dev_pool[0])

    # ---- SURVEY.md 8(f) #4, precision axis: sustained ms / J per trial of EVERY precision in one record (the two
    # paths above plus the three the line does not otherwise run), each with its sustained kernel split and its
    # table binned by the SM clock the power cap produced
    energy_grid = None
    if ctx.world == 1 and not args.no_energy_grid and args.energy_seconds > 0 and m["energy"] is not None:
        def grid_row(prec, burst_ms, e):
            return {"precision": prec, "ms_per_step_burst": burst_ms, "ms_per_step_sustained": e["ms_per_step"],
                    "joules_per_step": e["joules_per_step"], "mean_power_w": e["mean_power_w"],
                    "sm_mhz": e["clocks"].get("sm_mhz"), "reasons": e["clocks"].get("reasons"),
                    "kernel_ms_sustained": e["kernel_ms_sustained"], "clock_bins": e.get("clock_bins", {}).get("rows")}
        rows = [grid_row(precision, m["ms_per_step"], m["energy"])]
        if fft_path is not None and fft_path["energy"] is not None:
            rows.append(grid_row(fft_path["precision"], fft_path["ms_per_step"], fft_path["energy"]))
        for prec in ("bf16_tc", "bf16_tc_plane16", "bf16", "bf16_plane16", "fp32"):
            if any(r["precision"] == prec for r in rows):
                continue
            plan_g = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, prec)
            mg = time_path(plan_g, fdas, torch, wl, dev_pool, thr, args.steps, args.warmup, args.energy_seconds,
                           ctx.local_rank, lambda: None, want_modes=False)
            mg.pop("buffers")
            if mg["energy"] is not None:
                rows.append(grid_row(prec, mg["ms_per_step"], mg["energy"]))
            plan_g.close()
            torch.cuda.empty_cache()
        energy_grid = {"rows": rows, "seconds_each": args.energy_seconds,
                       "note": "one sustained loop of identical SKA-like steps per precision at default clocks; the clock "
                               "axis is what the 1000 W cap does by itself (clock_bins); locking clocks is unavailable "
                               "on this pool (PAPER.md:27, :33-45)"}

    survey = None
    if args.survey_trials != 0 and args.workload == "ska" and ctx.world == 1:
        del dev_pool
        torch.cuda.empty_cache()
        survey = survey_block(fdas, torch, inputs, precision, args.survey_trials, min(4, args.pool), thr, ctx.local_rank)

    plane_bytes = points * int(info.plane_elem_bytes)
    k3_gbs = int(info.nz) * (int(info.nbins) // 8) * 2 / (m["kernel_ms"]["harmonic_sum_peaks"] * 1e-3) / 1e9
    hbm_peak, peak_kind = measured_peaks()
    arith = "bf16 operands, fp32 accumulation on the tensor cores" if is_tc else "fp32 arithmetic"
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ctx.world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_max_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16 x bf16 -> f32 (tensor cores)" if is_tc else "f32", "data": "synthetic",
        "config": {
            "workload": workload_string(wl),
            "precision": f"{precision} ({arith})", "plane_points_per_step": points,
            "geometry": f"h={info.halfwidth}, V={info.valid}, S={info.nseg}, Nb={info.nbins}",
            "parallelism": f"dm-trial replicas x{ctx.world} (no data-path collective)",
            "l2": f"plane of {plane_bytes / 1e9:.2f} GB per step exceeds the 126 MB L2; input pool of "
                  f"{pool_n} series ({pool_bytes / 1e6:.0f} MB) cycled",
            "timed": "cuFFT R2C + K1a/K1b whitening + K2 convolve + K3 harmonic sum per step; CUDA events on the "
                     f"launching stream over {args.steps} steps; the `energy` loop ({args.energy_seconds:g} s of the "
                     "same steps) is the sustained figure",
        },
        "kernel_ms": m["kernel_ms"],
        "harmonic_modes": m["harmonic_modes"],
        "k3_stress": m["k3_stress"],
        "candidates_last_step": m["candidates_last_step"],
        "gpu_launches": launches_total,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(info.nfft) * 4,
                "d2h_bytes_per_step": d2h // e2e_steps, "steps": e2e_steps,
                "api": "fdas_search_batch (pinned host series -> candidates on host, copies pipelined with "
                       "compute), wall clock",
                "one_trial_per_call": {"value": e2e_sync_value, "api": "fdas_search_host, synchronous"}},
        "roofline": roofline,
        "roofline_hbm": roofline_hbm,
        "roofline_k3": {
            "kernel": "K3 prefilter kernels + exact_kernel + flag_kernel", "bound": "latency", "achieved": k3_gbs,
            "peak": hbm_peak, "unit": "GB/s", "frac": k3_gbs / hbm_peak,
            "note": "K3 is bound by the latency of its dependent loads and by the random 32-byte sector reads of its "
                    "exact pass, not by DRAM bandwidth (profiles/r02b_k3_seglen.md): `achieved` / `frac` are context only "
                    "-- one read of the block-max side plane (nz x Nb/8 16-bit codes, the bytes the branch-and-bound "
                    "prefilter has to scan) over the measured K3 time, against the HBM peak",
        },
        "clocks": m["clocks"],
    }
    if fft_path is not None:
        line["fft_path"] = fft_path
    if m["energy"] is not None:
        line["energy"] = m["energy"]
    if "energy_by_kernel" in m:
        line["energy_by_kernel"] = m["energy_by_kernel"]
    if energy_grid is not None:
        line["energy_grid"] = energy_grid
    if survey is not None:
        line["survey"] = survey
    if ctx.world > 1:
        line["config"]["omitted"] = ("with more than one rank the line carries no fft_path, energy_grid, survey or "
                                     "cpu_baseline block (they are single-GPU records)")
    if m["energy"] is not None:
        line["sustained"] = {"ms_per_step": m["energy"]["ms_per_step"],
                             "value": points / (m["energy"]["ms_per_step"] * 1e-3), "unit": UNIT,
                             "joules_per_step": m["energy"]["joules_per_step"],
                             "sm_mhz": m["energy"]["clocks"].get("sm_mhz"),
                             "note": "the honest per-DM-trial figure of a survey: the seconds-long loop at the power "
                                     "cap; `value` / `ms_per_step` of the line are the contract's K-step burst"}
    if ctx.rank == 0 and ctx.world == 1 and not args.no_cpu_baseline:
        v, cores, desc, _ = oracle_sample(host_pool[0].numpy(), wl, args.cpu_budget)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    if ctx.rank == 0:
        print(json.dumps(line), flush=True)
    fd.finalize(ctx)
    return 0


# ------------------------------------------------- configs[3] / configs[4]: pipelined DM trials
def run_batch(args):
    """BASELINE.json configs[3] (64 SKA-like trials) and configs[4] (3050 at 64 us + 2875 at 128 us)
    through fdas_search_batch: three streams, double-buffered planes.  One `step` = one DM trial."""
    import torch
    from paper_2211_13517_b200 import dist as fd, fdas, inputs

    ctx = fd.init_from_env("nccl")
    torch.cuda.set_device(ctx.local_rank)
    dev = torch.device("cuda", ctx.local_rank)
    precision = args.precision
    if args.workload == "batched":
        shapes = [("ska", False, args.trials or 64)]
    else:
        nf, nh = inputs.SURVEY_TRIALS_FULL, inputs.SURVEY_TRIALS_HALF
        if args.trials:
            nf = max(1, round(args.trials * nf / (nf + nh)))
            nh = max(1, args.trials - nf)
        shapes = [("ska", False, nf), ("ska_half", True, nh)]
    cap = 1 << 14
    parts = []
    for name, half, ntr in shapes:
        wl = inputs.ska(half_res=half)
        plan = fdas.Plan(wl.n, wl.tsamp, wl.zmax, wl.zstep, wl.seg_len, precision)
        pool_n = max(1, min(args.pool, ntr))
        host = []
        for i in range(pool_n):
            ht = torch.empty(wl.n, dtype=torch.float32).pin_memory()
            ht.numpy()[:] = inputs.series_for(inputs.batched_member((ctx.rank * pool_n + i) % 64, half_res=half))
            host.append(ht)
        devs = [h.to(dev) for h in host]
        out = np.empty((ntr, cap), dtype=fdas.CAND_DTYPE)
        parts.append(dict(name=name, wl=wl, plan=plan, ntr=ntr, host=host, dev=devs, out=out, pool=pool_n))
    thr = fdas.thresholds_from_sigma(16, 6.0)
    stream = torch.cuda.current_stream()

    def run_all(on_host, frac=1.0):
        counts = []
        for p in parts:
            n = max(1, int(p["ntr"] * frac))
            src = p["host"] if on_host else p["dev"]
            series = [src[i % p["pool"]] for i in range(n)]
            c, _, st = p["plan"].search_batch(series, p["wl"].nharm, thr, p["wl"].r_lo, capacity=cap,
                                              out=p["out"], stream=stream)
            assert st in (fdas.FDAS_OK, fdas.FDAS_EOVERFLOW), st
            counts.append(c)
        return counts

    warm_frac = min(1.0, max(args.warmup, 3) * 2.0 / min(p["ntr"] for p in parts))
    run_all(False, warm_frac)
    run_all(True, warm_frac)
    torch.cuda.synchronize()

    sampler = ClockSampler(ctx.local_rank, period=0.05)
    launches0 = sum(p["plan"].launch_count() for p in parts)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fd.barrier(ctx)
    torch.cuda.synchronize()
    sampler.start()
    j0 = sampler.energy_mj() if sampler.ok else None
    ev0.record(stream)
    counts = run_all(False)
    ev1.record(stream)
    torch.cuda.synchronize()
    j1 = sampler.energy_mj() if sampler.ok else None
    sampler.stop_flag.set()
    fd.barrier(ctx)
    sampler.join(timeout=2.0)
    t_ms = ev0.elapsed_time(ev1)
    launches = sum(p["plan"].launch_count() for p in parts) - launches0
    trials = sum(p["ntr"] for p in parts)
    points = sum(p["ntr"] * int(p["plan"].info.nz) * int(p["plan"].info.nbins) for p in parts)
    t_max_ms = fd.max_over_ranks(ctx, t_ms)
    value = fd.sum_over_ranks(ctx, float(points)) / (t_max_ms * 1e-3)

    # end to end: the same trials from pinned host memory (H2D of every series inside the region)
    fd.barrier(ctx)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    counts_h = run_all(True)
    torch.cuda.synchronize()
    t_e2e = fd.max_over_ranks(ctx, time.perf_counter() - t0)
    e2e_value = fd.sum_over_ranks(ctx, float(points)) / t_e2e
    assert all((a == b).all() for a, b in zip(counts, counts_h))
    h2d = sum(p["ntr"] * int(p["plan"].info.nfft) * 4 for p in parts) / trials
    d2h = sum(int(np.minimum(c, cap).sum()) * 16 + 8 * c.size for c in counts) / trials

    hbm_peak, peak_kind = measured_peaks()
    k2_flops = sum(p["ntr"] * int(p["plan"].info.nseg) * (int(p["plan"].info.nz) * (
        FLOP_IFFT + FLOP_MUL + 3 * int(p["plan"].info.valid)) + FLOP_IFFT) for p in parts)
    is_tc = precision in TC_PRECISIONS
    arith = "bf16 operands, fp32 accumulation on the tensor cores" if is_tc else "fp32 arithmetic"
    hbm_gbs = HBM_BYTES_PER_POINT[precision] * points / (t_max_ms * 1e-3) / 1e9
    if is_tc:
        batch_roofline = {"kernel": "K2-TC convolve_tc_kernel's algorithmic bytes of all trials over the whole pipelined time",
                          "bound": "hbm", "achieved": hbm_gbs, "peak": hbm_peak, "unit": "GB/s",
                          "frac": hbm_gbs / hbm_peak, "traffic": None,
                          "note": "per-kernel rooflines are reported by the single-trial workload (--workload ska)"}
    else:
        batch_roofline = {"kernel": "K2 convolve_kernel's algorithmic flops of all trials over the whole pipelined time",
                          "bound": "alu", "achieved": k2_flops / (t_max_ms * 1e-3) / 1e12, "peak": ALU_PEAK_TFLOPS,
                          "unit": "TFLOP/s", "frac": k2_flops / (t_max_ms * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                          "traffic": None,
                          "note": "per-kernel rooflines are reported by the single-trial workload (--workload ska)"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ctx.world, "steps": trials,
        "warmup": args.warmup, "ms_per_step": t_max_ms / trials, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16 x bf16 -> f32 (tensor cores)" if is_tc else "f32", "data": "synthetic",
        "config": {
            "workload": (f"{args.workload}: " + " + ".join(
                f"{p['ntr']} trials of N={p['wl'].n} at {p['wl'].tsamp * 1e6:.0f} us (nfft={p['plan'].info.nfft})"
                for p in parts) + f", nz=193, seg_len=2048, H=16, 6 sigma, storage={precision} ({arith})"),
            "precision": precision, "plane_points_total": points,
            "parallelism": f"dm-trial replicas x{ctx.world} (no data-path collective)",
            "pipeline": "fdas_search_batch: copy / prepare+K2 / K3+D2H streams, two slots of every per-trial buffer",
            "l2": "every trial writes a 3.24 GB (1.62 GB at 128 us) plane, far beyond the 126 MB L2; "
                  + ", ".join(f"{p['pool']} distinct {p['name']} series cycled" for p in parts),
            "timed": "all trials, series resident in HBM; CUDA events on the caller's stream around the batch calls",
        },
        "candidates_total": int(sum(int(c.sum()) for c in counts)),
        "gpu_launches": int(fd.sum_over_ranks(ctx, int(launches))),
        "total_seconds": t_max_ms * 1e-3,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": trials, "seconds": t_e2e,
                "api": "fdas_search_batch (pinned host series -> candidates on host), wall clock"},
        "roofline": batch_roofline,
        "roofline_hbm": {"bound": "hbm", "achieved": HBM_BYTES_PER_POINT[precision] * points / (t_max_ms * 1e-3) / 1e9,
                         "peak": hbm_peak, "unit": "GB/s", "peak_kind": f"{peak_kind} copy bandwidth",
                         "note": "K2's algorithmic bytes of all trials over the whole pipelined time"},
        "clocks": sampler.summary(),
    }
    line["roofline_hbm"]["frac"] = line["roofline_hbm"]["achieved"] / hbm_peak
    if j0 is not None and j1 is not None and j1 > j0:
        line["energy"] = {"joules_per_step": (j1 - j0) / 1e3 / trials, "joules_total": (j1 - j0) / 1e3,
                          "mean_power_w": (j1 - j0) / 1e3 / (t_ms * 1e-3), "seconds": t_ms * 1e-3,
                          "source": "NVML total energy counter over the timed region"}
    if ctx.rank == 0:
        print(json.dumps(line), flush=True)
    for p in parts:
        p["plan"].close()
    fd.finalize(ctx)
    return 0


def spawn_command(ngpus, argv):
    """`python bench.py --gpus N ...` without a launcher: one rank per GPU on this node through
    torch.distributed.run (the ranks then find WORLD_SIZE / RANK / LOCAL_RANK in their environment)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={ngpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000),
            os.path.abspath(__file__)] + list(argv)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="ska",
                    choices=["ska", "ska_half", "ska_padded", "medium", "tiny", "batched", "survey"])
    ap.add_argument("--energy-seconds", type=float, default=2.5,
                    help="length of the separate energy loop (0 = off)")
    ap.add_argument("--trials", type=int, default=0,
                    help="batched/survey: trials per rank (0 = 64 for batched, 3050+2875 for survey)")
    ap.add_argument("--precision", default="bf16_tc", choices=["fp32", "bf16", "bf16_plane16", "bf16_tc", "bf16_tc_plane16"])
    ap.add_argument("--pool", type=int, default=4, help="distinct series cycled per rank")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle plane work")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fft-path", action="store_true", help="skip the full record of the FFT K2 path")
    ap.add_argument("--survey-trials", type=int, default=-1,
                    help="ska workload, 1 GPU: DM trials of EACH resolution in the `survey` block "
                         "(-1 = the paper's 3050 + 2875, 0 = off)")
    ap.add_argument("--no-energy-grid", action="store_true",
                    help="skip the sustained ms / J per trial of the precisions the line does not otherwise run")
    ap.add_argument("--traffic-from-ncu", default=None, metavar="REP",
                    help="write the DRAM traffic of the launches in an ncu report to --traffic-out and exit")
    ap.add_argument("--traffic-out", default=os.path.join(PROFILES, "r03_traffic.json"))
    ap.add_argument("--traffic-command", default="", help="the command the ncu report was captured with")
    args = ap.parse_args()
    if args.traffic_from_ncu:
        write_traffic_json(args.traffic_from_ncu, args.traffic_out, args.workload, args.precision, args.traffic_command)
        return 0
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.impl == "cuda" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched plainly with --gpus N: start the N ranks ourselves, one per GPU (DM-trial replicas)
        import subprocess
        return subprocess.call(spawn_command(args.gpus, sys.argv[1:]),
                               env=dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "INFO")))
    if args.impl == "reference":
        if args.workload in ("batched", "survey"):
            args.workload = "ska"      # the oracle's per-trial rate is the same for every member
        return run_reference(args)
    if args.workload in ("batched", "survey"):
        return run_batch(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
