#!/usr/bin/env python
"""bench.py -- attempted spin flips / ns on B200 for the PT spin-glass hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]

A STEP is `--mcs-per-step` Monte Carlo steps (one Metropolis sweep of every replica, one Houdayer
cluster exchange per equal-temperature pair where the config enables it, one parallel-tempering pass, plus the overlap
measurement every k-th MCS where the config asks for it) of the whole workload, issued as one pt_mcs() /
pt_mcs_measure_device() call through the C ABI.

BASELINE.json's metric names no config, so the HEADLINE workload is the largest single-GPU configuration, C5 (2D L=128,
128 samples x 48 temperatures x 2 chains, Houdayer + PT every sweep: 2.0e12 attempted flips in its 10^4 MCS); with the
default K=200, 50 MCS per step the timed region is exactly the config's 10^4 MCS.  The other configs C1-C4 are timed in
the same run, each over `--config-steps` steps, and reported in the `per_config` block of the same JSON line (value,
ms_per_step, roofline, clocks, kernel and phase times).  Inputs are synthetic (seeded +-J samples) and
resident in HBM when the timed region starts; L2 is flushed between steps (untimed); each step is timed with CUDA events
on the library's stream; multi-GPU = independent sample shards (weak scaling, no data-path collective), max over ranks.

The timed region runs WITHOUT per-launch instrumentation; the per-kernel-class CUDA-event times and the phase clocks of
the fused kernel come from a second, instrumented pass of a few steps right after it (`roofline.kernel_ms_pass`).

`--impl reference` times the CPU oracle (oracle/, as it stands) on all host cores, one process per core on disjoint
sample ranges, each step a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "attempted_spin_flips_per_ns"
UNIT = "flips/ns"
SM_COUNT = 148
INT32_LANES_PER_SM_CLK = 128       # 4 SMSPs x 1 warp-instruction/clk x 32 lanes (fma + alu pipes, 64 each)
ALGO_OPS_PER_FLIP = {2: 20, 3: 22}  # Philox share 10 + 2d field terms + 6 decide/flip/accumulate
KERNEL_CLASSES = ["k_sweep", "k_houdayer", "k_exchange", "k_measure", "k_mcs"]
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from committed `ncu --set full` captures
# (never measured in this run: a number taken under a profiler is not a bench value).  (workload, kernel) -> (bytes, file)
NCU_TRAFFIC = {}
try:
    import csv as _csv
    with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as _f:
        NCU_TRAFFIC = {(r["workload"], r["kernel"]): (float(r["dram_bytes_per_launch"]), r["source"]) for r in _csv.DictReader(_f)}
except Exception:
    pass


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=sorted(wl.CONFIGS))
    ap.add_argument("--mcs-per-step", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--config-steps", type=int, default=20, help="timed steps of each per_config entry")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--gaussian", action="store_true", help="NEXT-3: Gaussian couplings in fixed point (16 fractional bits)")
    ap.add_argument("--track-round-trips", action="store_true", help="NEXT-1: tunnelling-time bookkeeping in every PT pass")
    ap.add_argument("--cluster", default="single", choices=["single", "counts", "multi"],
                    help="NEXT-4 cluster-move variant of a Houdayer workload: one single-cluster move per temperature (the paper's "
                         "MCS), per-temperature move counts 4..1 from the hot to the cold end, or the multi-cluster exchange")
    return ap.parse_args()


# --------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def window(self, t0, t1):
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.15 and len(r) >= 8] or [r for (_, r) in self.rows[-3:]]
        sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
        reasons = set()
        for r in rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(rows[0][1]) if rows else None,
                "power_w_max": max([float(r[2]) for r in rows if r[2].replace(".", "").isdigit()] or [0.0]),
                "samples": len(rows), "reasons": sorted(reasons)}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def shorten(x):
    """Floats to 5 significant digits (the JSON line is read by people and kept by its tail)."""
    if isinstance(x, float):
        return float("%.5g" % x)
    if isinstance(x, dict):
        return {k: shorten(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [shorten(v) for v in x]
    return x


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def gauss_fbits(w):
    """Fractional bits of the fixed-point Gaussian couplings (NEXT-3): 16 where the int32 energies allow it, else the most
    that keep d * N * max|Jq| below 2^31 with |J| < 6 sigma (C5's 2D L=128: 12)."""
    f = 16
    while f > 0 and w.d * w.N * 6.0 * (1 << f) >= 2.0 ** 31:
        f -= 1
    return f


def cluster_args(a, w):
    """(do_houdayer mode, per-temperature move counts or None) of the workload under --cluster."""
    hd = (2 if a.cluster == "multi" else 1) if w.houdayer else 0
    n_clu = None
    if w.houdayer and a.cluster == "counts":       # index 0 is the lowest beta = the hot end
        n_clu = np.array([1 + (3 * t) // max(w.T - 1, 1) for t in range(w.T)], dtype=np.int32)[::-1].copy()
    return hd, n_clu


# --------------------------------------------------------------------------------------------------------------
def oracle_rate(a, w, procs, samples_per_proc, target_flips_per_proc):
    """The oracle as it stands on `procs` host cores (one single-threaded process per core, disjoint sample ranges,
    PAPER.md:241).  Returns (aggregate flips/ns, seconds, flips, MCS)."""
    from oracle import pool as OP

    hd, n_clu = cluster_args(a, w)
    fixed = None
    if a.gaussian:
        fixed = (wl.gaussian_couplings_fixed(wl.SEED, procs * samples_per_proc, w.d, w.N, gauss_fbits(w)), gauss_fbits(w))
    n_mcs = max(1, int(target_flips_per_proc / w.flips_per_sweep(samples_per_proc)))
    po = OP.PersistentOracles(w, procs, samples_per_proc, houdayer_mode=hd, fixed=fixed,
                              n_clu=None if n_clu is None else n_clu.tolist())
    try:
        po.step(1)                                   # first touch of every page
        t0 = time.perf_counter()
        po.step(n_mcs)
        dt = time.perf_counter() - t0
    finally:
        po.close()
    flips = w.flips_per_sweep(procs * samples_per_proc) * n_mcs
    return flips / dt * 1e-9, dt, flips, n_mcs


def run_reference(a, w, rank):
    """--impl reference: the CPU oracle on all host cores; each step a bounded sample of the workload."""
    if rank != 0:
        return
    from oracle import pool as OP

    P = OP.n_cores()
    hd, n_clu = cluster_args(a, w)
    fixed = (wl.gaussian_couplings_fixed(wl.SEED, P, w.d, w.N, gauss_fbits(w)), gauss_fbits(w)) if a.gaussian else None
    ref_mcs = max(1, min(a.mcs_per_step, int(round(0.25 / (w.flips_per_sweep(1) * 30e-9)))))
    po = OP.PersistentOracles(w, P, 1, houdayer_mode=hd, fixed=fixed, n_clu=None if n_clu is None else n_clu.tolist())
    try:
        for _ in range(a.warmup):
            po.step(ref_mcs)
        t0 = time.perf_counter()
        for _ in range(a.steps):
            po.step(ref_mcs)
        dt = time.perf_counter() - t0
    finally:
        po.close()
    flips = w.flips_per_sweep(P) * ref_mcs * a.steps
    v = flips / dt * 1e-9
    sample = "%s restricted to %d samples (one oracle process per host core), %d MCS per step" % (w.name, P, ref_mcs)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": dt / a.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": config_of(a, w, a.gpus, sample=sample),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": P, "kind": "oracle", "sample": sample, "cpu": cpu_model()},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def config_of(a, w, n_gpus, sample=None):
    c = {"workload": "%s: %dD EA +-J, L=%d, %d samples x %d temperatures (beta %s %.1f..%.1f) x 2 chains per GPU" % (
             w.name, w.d, w.L, w.S, w.T, w.ladder, w.b_min, w.b_max),
         "mcs_per_step": a.mcs_per_step, "mcs_order": "sweep" + (", houdayer" if w.houdayer else "") + ", exchange",
         "measure_every": w.measure_every, "seed": wl.SEED, "parallelism": "samples sharded x%d" % n_gpus,
         "l2": "flushed between steps (512 MiB write, untimed)", "round_trip_tracking": bool(a.track_round_trips),
         "couplings": "gaussian, fixed point 2^-%d (NEXT-3)" % gauss_fbits(w) if a.gaussian else "+-J, p = 1/2",
         "cluster_move": {"single": "one single-cluster move per temperature", "counts": "single-cluster moves, counts 4..1 hot to cold (NEXT-4)",
                          "multi": "multi-cluster exchange (NEXT-4)"}[a.cluster] if w.houdayer else "none"}
    if sample:
        c["sample"] = sample
    return c


# --------------------------------------------------------------------------------------------------------------
class GpuRun:
    """One workload on this rank's GPU: the context, the step, the timed region, the instrumented pass."""

    def __init__(self, a, w, rank, world, dev, flush):
        import torch
        from paper_2003_04621_b200 import binding as B

        self.a, self.w, self.rank, self.world, self.dev, self.flush, self.B, self.torch = a, w, rank, world, dev, flush, B, torch
        self.Jq = wl.gaussian_couplings_fixed(wl.SEED, w.S, w.d, w.N, gauss_fbits(w), sample_offset=rank * w.S) if a.gaussian else None
        self.open()
        self.n_meas = (a.mcs_per_step // w.measure_every) if w.measure_every else 0
        self.Qrec = torch.empty((max(self.n_meas, 1), w.S, w.T), dtype=torch.int32, device=dev)
        self.QLrec = torch.empty_like(self.Qrec)
        self.flips_step = w.flips_per_sweep() * a.mcs_per_step

    def open(self):
        """pt_init of the workload (not timed): the state of MCS 0; same seed, same trajectory every time."""
        a, w, B = self.a, self.w, self.B
        B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, sample_offset=self.rank * w.S, device=self.dev,
                  track_round_trips=a.track_round_trips, fixed_couplings=a.gaussian, full_staging=True)
        if self.Jq is not None:
            B.pt_set_couplings_fixed(self.Jq, gauss_fbits(w))
        self.hd, n_clu = cluster_args(a, w)
        if n_clu is not None:
            B.pt_set_cluster_moves(n_clu)

    def from_mcs0(self, steps):
        """SURVEY 8(d) timing protocol: the same run timed FROM MCS 0 (a fresh pt_init, the kernels already loaded by
        the passes before it), next to the steady-state window (MCS >= 128) the warmed-up timed region covers."""
        torch = self.torch
        self.open()
        self.barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for k in range(steps):
            self.flush.fill_(k & 0xFF)
            evs[k][0].record()
            self.step()
            evs[k][1].record()
        self.barrier()
        ms = self.max_over_ranks(sum(e0.elapsed_time(e1) for e0, e1 in evs))
        return {"value": self.world * self.flips_step * steps / (ms * 1e6), "mcs": [0, steps * self.a.mcs_per_step]}

    def step(self):
        if self.n_meas == 0:
            self.B.pt_mcs(self.a.mcs_per_step, 1, self.hd, True)
        else:                                    # the MCS with the overlap records fused in (one launch where eligible)
            self.B.pt_mcs_measure_device(self.a.mcs_per_step, 1, self.hd, True, self.w.measure_every, self.Qrec, self.QLrec)

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
            self.torch.cuda.synchronize()

    def max_over_ranks(self, x):
        if self.world > 1:
            import torch.distributed as dist
            t = self.torch.tensor([x], dtype=self.torch.float64, device=self.dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return x

    def timed(self, steps, warmup, sampler):
        """W untimed warm-up steps, then exactly `steps` steps, each bracketed by CUDA events on the library's stream
        (the L2 flush between steps is outside the events); barrier + synchronize on both sides; max over ranks."""
        torch, B = self.torch, self.B
        for _ in range(warmup):
            self.step()
        self.barrier()
        launches0 = B.pt_get_launch_count()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        self.barrier()
        t0 = time.time()
        for k in range(steps):
            self.flush.fill_(k & 0xFF)
            evs[k][0].record()
            self.step()
            evs[k][1].record()
        self.barrier()
        t1 = time.time()
        ms_steps = [e0.elapsed_time(e1) for e0, e1 in evs]
        ms_total = self.max_over_ranks(sum(ms_steps))
        launches = B.pt_get_launch_count() - launches0
        assert B.pt_recompute_energy()[1] == 0, "tracked energies diverged from recomputed energies"
        # the steps are the repetitions (same work every step): median / min / max of this rank's per-step event times
        stats = {"median": float(np.median(ms_steps)), "min": float(np.min(ms_steps)), "max": float(np.max(ms_steps))}
        return {"value": self.world * self.flips_step * steps / (ms_total * 1e6), "ms_per_step": ms_total / steps,
                "ms_total": ms_total, "steps": steps, "gpu_launches": int(launches), "ms_step_stats": stats,
                "value_median_step": self.world * self.flips_step / (stats["median"] * 1e6),
                "mcs": [warmup * self.a.mcs_per_step, (warmup + steps) * self.a.mcs_per_step],
                "clocks": sampler.window(t0, t1) if sampler else None}

    def instrumented(self, steps, t):
        """Second pass (outside the timed region): every launch bracketed by CUDA events (per-class kernel times), the fused
        kernel's phase clocks on, then the Metropolis sweeps alone.  Returns the roofline block."""
        torch, B, a, w = self.torch, self.B, self.a, self.w
        peaks, peaks_kind = measured_peaks()
        B.pt_set_sample_groups(1)                 # one stream: per-class kernel times that do not overlap one another
        B.pt_set_profiling(True)
        B.pt_set_phase_clocks(True)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(steps):
            self.step()
        ev1.record()
        kms, kn = B.pt_get_kernel_times()
        pclk = B.pt_get_phase_clocks().astype(np.float64)
        B.pt_set_phase_clocks(False)
        B.pt_set_profiling(False)
        B.pt_set_sample_groups(-1)
        pass_ms = ev0.elapsed_time(ev1)
        fused = kn[4] > 0
        dom = 4 if fused else 0                   # the roofline is quoted for the kernel that does the Metropolis sweeps
        n_mcs_pass = a.mcs_per_step * steps
        if fused:                                 # one launch per step: the un-instrumented step time IS the launch time
            mcs_per_launch = max(1, n_mcs_pass // max(int(kn[4]), 1))
            dom_ms = t["ms_per_step"] * mcs_per_launch / a.mcs_per_step
        else:
            mcs_per_launch = 1
            dom_ms = kms[0] / max(int(kn[0]), 1)
        flips_per_launch = w.flips_per_sweep() * mcs_per_launch
        dom_flips_ns = flips_per_launch / (dom_ms * 1e6) if dom_ms > 0 else 0.0
        A = ALGO_OPS_PER_FLIP[w.d]
        f_max = peaks.get("sm_max_mhz", 1965.0) / 1e3
        peak_ops = SM_COUNT * INT32_LANES_PER_SM_CLK * f_max
        # ---- per-phase time per spin in the paper's normalisation, Eq. (11): t_update = t_kernel / (N_T N_R N_C N_B L^d)
        spins_mcs = float(w.flips_per_sweep())
        if fused:
            share = pclk / max(pclk.sum(), 1.0)
            per_mcs_us = t["ms_per_step"] / a.mcs_per_step * 1e3
            ph = {"metropolis": share[0] * per_mcs_us, "houdayer": share[1] * per_mcs_us, "exchange": share[2] * per_mcs_us,
                  "rest": share[3] * per_mcs_us}
            how = "fused launch: time per MCS x clock64() share of each phase"
        else:
            ph = {"metropolis": kms[0] / n_mcs_pass * 1e3, "houdayer": kms[1] / n_mcs_pass * 1e3,
                  "exchange": kms[2] / n_mcs_pass * 1e3, "rest": max(pass_ms - kms[:4].sum(), 0.0) / n_mcs_pass * 1e3}
            how = "separate launches: CUDA events per launch, instrumented pass on ONE stream; rest = gaps"
        phases = {"us_per_mcs": ph, "ns_per_spin": {k: v * 1e3 / spins_mcs for k, v in ph.items()},
                  "houdayer_over_metropolis": (ph["houdayer"] / ph["metropolis"]) if ph["metropolis"] > 0 else None,
                  "exchange_over_metropolis": (ph["exchange"] / ph["metropolis"]) if ph["metropolis"] > 0 else None,
                  "how": how}
        traffic = NCU_TRAFFIC.get((w.name, KERNEL_CLASSES[dom])) if not a.gaussian and a.cluster == "single" else None
        roofline = {
            "bound": "alu", "kernel": KERNEL_CLASSES[dom], "achieved": A * dom_flips_ns, "peak": peak_ops,
            "unit": "Gop/s (INT32 thread-ops)", "frac": A * dom_flips_ns / peak_ops,
            "traffic": traffic[0] if traffic else None,
            "traffic_source": traffic[1].split(":")[0] if traffic else None,        # the file; profiles/ncu_traffic.csv has the details
            "peak_how": "148 SMs x 128 INT32 lanes/clk x %.3f GHz; achieved = %d algorithmic ops/flip (SURVEY 8(d)) x flips per launch / "
                        "launch time; a %s launch = %d MCS = %d flips" % (f_max, A, KERNEL_CLASSES[dom], mcs_per_launch, flips_per_launch),
            "flips_per_ns": dom_flips_ns, "ms_per_launch": dom_ms,
            "whole_mcs_frac": A * t["value"] / self.world / peak_ops,
            "hbm": {"algorithmic_bytes_per_flip": 0.25 / mcs_per_launch, "achieved_gbs": 0.25 / mcs_per_launch * dom_flips_ns,
                    "peak_gbs": peaks.get("hbm_gbs"), "peak_kind": peaks_kind,
                    "frac": 0.25 / mcs_per_launch * dom_flips_ns / peaks.get("hbm_gbs", 6650.0)},
            "kernel_ms": {n: float(kms[i]) for i, n in enumerate(KERNEL_CLASSES)},
            "kernel_launches": {n: int(kn[i]) for i, n in enumerate(KERNEL_CLASSES)},
            "kernel_ms_pass": "%d instrumented steps (%d MCS) after the timed region, %.3f ms in all" % (steps, n_mcs_pass, pass_ms),
            "phases": phases,
        }
        # the Metropolis sweeps alone (a1-a3; Eq. (11) normalisation), same state, resident for mcs_per_step sweeps
        B.pt_set_profiling(True)
        for _ in range(3):
            B.pt_sweep(a.mcs_per_step)
        sms, sn = B.pt_get_kernel_times()
        B.pt_set_profiling(False)
        so = w.flips_per_sweep() * a.mcs_per_step / (sms[0] / max(int(sn[0]), 1) * 1e6)
        roofline["sweep_only"] = {"kernel": "k_sweep", "flips_per_ns": so, "frac": A * so / peak_ops,
                                  "what": "pt_sweep(%d) launches, no Houdayer / exchange" % a.mcs_per_step}
        assert B.pt_recompute_energy()[1] == 0
        return roofline

    def measurement_kernels(self):
        """The two measurement kernels alone (a6 and the NEXT-2 overlap profile), CUDA events around 20 calls each."""
        torch, B, w = self.torch, self.B, self.w
        prof_d = torch.empty((w.S, w.T, w.d, w.L), dtype=torch.int32, device=self.dev)
        out = {}
        for label, fn in (("overlap", lambda: B.pt_measure_overlap_device(self.Qrec[0], self.QLrec[0])),
                          ("overlap_profile", lambda: B.pt_measure_overlap_profile_device(prof_d))):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            m0.record()
            for _ in range(20):
                fn()
            m1.record()
            torch.cuda.synchronize()
            out[label] = m0.elapsed_time(m1) / 20 * 1e3
        return out

    def e2e(self, steps):
        """End to end through the C ABI with HOST buffers: H2D of the int8 spins, the step, D2H of the energies."""
        torch, B, w = self.torch, self.B, self.w
        assert B.pt_get_stage_bytes() == w.S * 2 * w.T * w.N, "PT_WS_FULL_STAGING not delivered"
        host_spins = torch.empty((w.S, 2, w.T, w.N), dtype=torch.int8).pin_memory()
        host_E = torch.empty((w.S, 2, w.T), dtype=torch.int32).pin_memory()
        hs, hE = host_spins.numpy(), host_E.numpy()
        B.pt_get_spins(out=hs)
        for _ in range(2):
            B.pt_set_spins_async(hs); self.step(); B.pt_get_energy(out=hE)
        self.barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            B.pt_set_spins_async(hs)           # sample-chunked copies; the steps of the first chunks overlap the later copies
            self.step()
            B.pt_get_energy(out=hE)            # synchronises
        self.barrier()
        dt = self.max_over_ranks(time.perf_counter() - t0)
        # the same loop through the bit-packed boundary (pt_set_spins_packed: one eighth of the bytes)
        host_bits = torch.empty((w.S, 2, w.T, (w.N + 31) // 32), dtype=torch.int32).pin_memory()
        hb = host_bits.numpy().view(np.uint32)
        B.pt_get_spins_packed(out=hb)
        for _ in range(2):
            B.pt_set_spins_packed(hb); self.step(); B.pt_get_energy(out=hE)
        self.barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            B.pt_set_spins_packed(hb)
            self.step()
            B.pt_get_energy(out=hE)
        self.barrier()
        dtp = self.max_over_ranks(time.perf_counter() - t0)
        packed = {"value": self.world * self.flips_step * steps / (dtp * 1e9), "unit": UNIT, "h2d_bytes_per_step": int(hb.nbytes),
                  "d2h_bytes_per_step": int(hE.nbytes), "what": "pt_set_spins_packed(host bit maps, pinned) + step + pt_get_energy(host)"}
        return {"value": self.world * self.flips_step * steps / (dt * 1e9), "unit": UNIT, "packed_boundary": packed,
                "h2d_bytes_per_step": int(hs.nbytes), "d2h_bytes_per_step": int(hE.nbytes),
                "steps": steps, "what": "pt_set_spins_async(host int8, pinned: sample-chunked H2D copies on the group streams) + step + "
                        "pt_get_energy(host, synchronises), wall clock; workspace with PT_WS_FULL_STAGING"}


# --------------------------------------------------------------------------------------------------------------
def main():
    a = parse()
    w = wl.CONFIGS[a.workload]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if a.impl == "reference":
        run_reference(a, w, rank)
        return

    import torch
    import torch.distributed as dist

    from paper_2003_04621_b200 import binding as B
    from paper_2003_04621_b200 import build as build_mod

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    if rank == 0:
        build_mod.build()
    assert B.pt_is_dev_build() == 0, "libptglass.so is a development build (PTG_DEV_LATTICE): rebuild the full library"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    flush = torch.empty(512 * 2 ** 20, dtype=torch.uint8, device=dev)
    sampler = ClockSampler(local) if rank == 0 else None

    # ---- headline: weak scaling, every rank holds the full per-GPU workload on its own range of global sample indices
    run = GpuRun(a, w, rank, world, dev, flush)
    t = run.timed(a.steps, a.warmup, sampler)
    roofline = run.instrumented(min(a.steps, 10), t) if rank == 0 or world > 1 else None
    e2e = None if a.no_e2e else run.e2e(a.e2e_steps)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    peaks, _ = measured_peaks()
    roofline["clock_ghz_during_run"] = (t["clocks"]["sm_mhz"] or peaks.get("sm_max_mhz", 1965.0)) / 1e3 if t["clocks"] else None
    philox_ops, _ = B.pt_microbench(4, 8, 1000, device=dev)     # measured live: Philox-only ceiling
    roofline["philox_only_flips_per_ns"] = philox_ops / 10.0
    roofline["measurement_us_per_call"] = run.measurement_kernels()
    fast_path = bool(B.pt_get_path())

    mcs0 = run.from_mcs0(max(a.warmup, 1))

    # ---- the other configs, same run, same protocol with fewer steps (N = 1 only: they are not part of the scaling line).
    # Numbers only (the prose that explains them is in the headline's roofline block and in DESIGN.md 9): the driver keeps
    # the TAIL of the line, so it is kept short and ends with `summary`.
    def compact(tc, rf, m0):
        ph = rf["phases"]["us_per_mcs"]
        return {"value": tc["value"], "ms_per_step": tc["ms_per_step"], "ms_step_stats": tc["ms_step_stats"], "steps": tc["steps"],
                "gpu_launches": tc["gpu_launches"], "sm_mhz": (tc["clocks"] or {}).get("sm_mhz"),
                "reasons": (tc["clocks"] or {}).get("reasons"), "kernel": rf["kernel"], "frac": rf["frac"],
                "whole_mcs_frac": rf["whole_mcs_frac"], "kernel_flips_per_ns": rf["flips_per_ns"], "ms_per_launch": rf["ms_per_launch"],
                "sweep_only_flips_per_ns": rf["sweep_only"]["flips_per_ns"], "from_mcs0": m0["value"],
                "us_per_mcs": [ph["metropolis"], ph["houdayer"], ph["exchange"], ph["rest"]]}

    per_config, summary = None, None
    if not a.no_per_config and world == 1:
        per_config = {w.name: dict(compact(t, roofline, mcs0), headline=True)}
        for name in sorted(wl.CONFIGS):
            if name == w.name:
                continue
            wc = wl.CONFIGS[name]
            rc = GpuRun(a, wc, rank, world, dev, flush)
            tc = rc.timed(a.config_steps, a.warmup, sampler)
            rf = rc.instrumented(min(a.config_steps, 5), tc)
            per_config[name] = compact(tc, rf, rc.from_mcs0(max(a.warmup, 1)))
        # [whole-MCS flips/ns, roofline frac of the dominant kernel, whole-MCS frac] per config; G2 / G5: the Gaussian
        # (fixed-point, NEXT-3) model on the two Houdayer shapes C2 and C5, whole-MCS flips/ns against the same op-count peak
        summary = {n: [per_config[n]["value"], per_config[n]["frac"], per_config[n]["whole_mcs_frac"]] for n in sorted(per_config)}
        if not a.gaussian and a.cluster == "single":
            import copy
            ag = copy.copy(a)
            ag.gaussian = True
            for n, key in (("C2", "G2"), ("C5", "G5")):
                rg = GpuRun(ag, wl.CONFIGS[n], rank, world, dev, flush)
                tg = rg.timed(a.config_steps, a.warmup, sampler)
                peak_ops = roofline["peak"]
                summary[key] = [tg["value"], None, ALGO_OPS_PER_FLIP[wl.CONFIGS[n].d] * tg["value"] / peak_ops]
    if sampler:
        sampler.stop()

    cpu = None
    if not a.no_cpu_baseline:
        from oracle import pool as OP

        P = OP.n_cores()
        v1, dt1, flips1, mcs1 = oracle_rate(a, w, 1, 1, 2.5e8)
        vP, dtP, flipsP, mcsP = oracle_rate(a, w, P, 1, 2.5e8)
        cpu = {"value": vP, "unit": UNIT, "cores": P, "kind": "oracle", "seconds": dtP, "cpu": cpu_model(),
               "sample": "%s restricted to %d samples (one single-threaded oracle process per host core on disjoint sample_offset "
                         "ranges, PAPER.md:241) x %d MCS (%.2e flips), same MCS order" % (w.name, P, mcsP, flipsP),
               "one_core": {"value": v1, "unit": UNIT, "cores": 1, "seconds": dt1,
                            "sample": "%s restricted to the first sample x %d MCS (%.2e flips)" % (w.name, mcs1, flips1)}}

    out = {
        "metric": METRIC, "value": t["value"], "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": t["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic", "config": config_of(a, w, world),
        "clocks": t["clocks"], "e2e": e2e, "gpu_launches": t["gpu_launches"], "roofline": roofline, "cpu_baseline": cpu,
        "ms_step_stats": t["ms_step_stats"], "value_median_step": t["value_median_step"],
        "timed_window_mcs": t["mcs"], "from_mcs0": mcs0, "fast_path": fast_path,
        "per_config": per_config, "summary": summary,           # `summary` stays the LAST key (the driver keeps the tail)
    }
    print(json.dumps(shorten(out)))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
