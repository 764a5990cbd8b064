#!/usr/bin/env python
"""bench.py -- attempted spin flips / ns on B200 for the PT spin-glass hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference]

A STEP is `--mcs-per-step` Monte Carlo steps (one Metropolis sweep of every replica, one
Houdayer cluster exchange per equal-temperature pair where the config enables it, one parallel-tempering pass,
plus the overlap measurement every k-th MCS where the config asks for it) of the whole workload, issued as one
pt_mcs() / pt_mcs_measure_device() call through the C ABI.  At N=1 the workload is BASELINE.json configs[1] (C2: 2D L=32, 1024 samples x
32 temperatures x 2 chains, Houdayer + PT every sweep).  With the default K=200, 50 MCS per step the timed region is
exactly the config's 10^4 MCS.  Inputs are synthetic (seeded +-J samples) and resident in HBM when the
timed region starts; L2 is flushed between steps (untimed); each step is timed with CUDA events on the library's
stream; multi-GPU = independent sample shards (weak scaling, no data-path collective), max over ranks.

`--impl reference` times the CPU oracle (oracle/, as it stands, one core) on a bounded sample of the same workload.
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

from paper_2003_04621_b200 import workloads as wl  # noqa: E402

METRIC = "attempted_spin_flips_per_ns"
UNIT = "flips/ns"
SM_COUNT = 148
INT32_LANES_PER_SM_CLK = 128       # 4 SMSPs x 1 warp-instruction/clk x 32 lanes (fma + alu pipes, 64 each)
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed ncu --set full
# capture of the same build (profiles/r1_v5_variants_and_gauss.md; r1_v4_final.md before it): the packed state of C2 is read once per k_mcs launch (10.68 MB,
# independent of the number of MCS per launch) and its write-back stays in L2 (0 B).  None where no capture exists.
NCU_DRAM_BYTES_PER_LAUNCH = {("C2", "k_mcs"): 10.68e6}
ALGO_OPS_PER_FLIP = {2: 20, 3: 22}  # Philox share 10 + 2d field terms + 6 decide/flip/accumulate


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=sorted(wl.CONFIGS))
    ap.add_argument("--mcs-per-step", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
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


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# --------------------------------------------------------------------------------------------------------------
def oracle_time(w, S, n_mcs, seed=wl.SEED, gaussian=False, cluster="single"):
    """Time the oracle as it stands on one host core; returns (flips/ns, seconds, flips)."""
    from oracle import ref

    o = ref.Oracle(w.L, w.d, S, w.T, w.betas(), seed)
    if gaussian:
        o.set_couplings_fixed(wl.gaussian_couplings_fixed(seed, S, w.d, w.N, 16), 16)
    hd = (2 if cluster == "multi" else 1) if w.houdayer else 0
    if w.houdayer and cluster == "counts":
        o.set_cluster_moves(np.array([1 + (3 * t) // max(w.T - 1, 1) for t in range(w.T)], dtype=np.int32)[::-1].copy())
    t0 = time.perf_counter()
    for m in range(1, n_mcs + 1):
        o.mcs(1, 1, hd, True)
        if w.measure_every and m % w.measure_every == 0:
            o.measure_overlap()
    dt = time.perf_counter() - t0
    flips = w.flips_per_sweep(S) * n_mcs
    o.close()
    return flips / dt * 1e-9, dt, flips


def run_reference(a, w, rank):
    """--impl reference: the CPU oracle, one core, each step a bounded sample (2 samples) of the workload."""
    if rank != 0:
        return
    S_ref = 2
    from oracle import ref

    o = ref.Oracle(w.L, w.d, S_ref, w.T, w.betas(), wl.SEED)
    if a.gaussian:
        o.set_couplings_fixed(wl.gaussian_couplings_fixed(wl.SEED, S_ref, w.d, w.N, 16), 16)

    hd = (2 if a.cluster == "multi" else 1) if w.houdayer else 0
    if w.houdayer and a.cluster == "counts":
        o.set_cluster_moves(np.array([1 + (3 * t) // max(w.T - 1, 1) for t in range(w.T)], dtype=np.int32)[::-1].copy())

    def step():
        o.mcs(a.mcs_per_step, 1, hd, True)
        if w.measure_every:
            for _ in range(a.mcs_per_step // w.measure_every):
                o.measure_overlap()

    for _ in range(a.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        step()
    dt = time.perf_counter() - t0
    flips = w.flips_per_sweep(S_ref) * a.mcs_per_step * a.steps
    v = flips / dt * 1e-9
    sample = "%s restricted to the first %d samples, %d MCS per step" % (w.name, S_ref, a.mcs_per_step)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": dt / a.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": config_of(a, w, a.gpus, sample=sample),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def config_of(a, w, n_gpus, sample=None):
    c = {"workload": "%s: %dD EA +-J, L=%d, %d samples x %d temperatures (beta %s %.1f..%.1f) x 2 chains per GPU" % (
             w.name, w.d, w.L, w.S, w.T, w.ladder, w.b_min, w.b_max),
         "mcs_per_step": a.mcs_per_step, "mcs_order": "sweep" + (", houdayer" if w.houdayer else "") + ", exchange",
         "measure_every": w.measure_every, "seed": wl.SEED, "parallelism": "samples sharded x%d" % n_gpus,
         "l2": "flushed between steps (512 MiB write, untimed)", "round_trip_tracking": bool(a.track_round_trips),
         "couplings": "gaussian, fixed point 2^-16 (NEXT-3)" if a.gaussian else "+-J, p = 1/2",
         "cluster_move": {"single": "one single-cluster move per temperature", "counts": "single-cluster moves, counts 4..1 hot to cold (NEXT-4)",
                          "multi": "multi-cluster exchange (NEXT-4)"}[a.cluster] if w.houdayer else "none"}
    if sample:
        c["sample"] = sample
    return c


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
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    # weak scaling: every rank holds the full per-GPU workload on its own range of global sample indices
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, sample_offset=rank * w.S, device=dev,
              track_round_trips=a.track_round_trips)
    if a.gaussian:
        B.pt_set_couplings_fixed(wl.gaussian_couplings_fixed(wl.SEED, w.S, w.d, w.N, 16, sample_offset=rank * w.S), 16)
    flush = torch.empty(512 * 2 ** 20, dtype=torch.uint8, device=dev)
    n_meas = (a.mcs_per_step // w.measure_every) if w.measure_every else 0
    hd = (2 if a.cluster == "multi" else 1) if w.houdayer else 0
    if w.houdayer and a.cluster == "counts":       # index 0 is the lowest beta = the hot end
        B.pt_set_cluster_moves(np.array([1 + (3 * t) // max(w.T - 1, 1) for t in range(w.T)], dtype=np.int32)[::-1].copy())

    Qrec = torch.empty((max(n_meas, 1), w.S, w.T), dtype=torch.int32, device=dev)
    QLrec = torch.empty_like(Qrec)

    def step():
        if n_meas == 0:
            B.pt_mcs(a.mcs_per_step, 1, hd, True)
        else:                                    # the MCS with the overlap records fused in (one launch where eligible)
            B.pt_mcs_measure_device(a.mcs_per_step, 1, hd, True, w.measure_every, Qrec, QLrec)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(a.warmup):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    B.pt_set_profiling(True)
    launches0 = B.pt_get_launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(a.steps)]
    barrier()
    t_wall0 = time.time()
    for k in range(a.steps):
        flush.fill_(k & 0xFF)                 # L2 flush, outside the timed events
        evs[k][0].record()
        step()
        evs[k][1].record()
    barrier()
    t_wall1 = time.time()
    ms_total = sum(e0.elapsed_time(e1) for e0, e1 in evs)
    kms, kn = B.pt_get_kernel_times()
    B.pt_set_profiling(False)
    launches = B.pt_get_launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    flips_step = w.flips_per_sweep() * a.mcs_per_step
    value = world * flips_step * a.steps / (ms_total * 1e6)
    assert B.pt_recompute_energy()[1] == 0, "tracked energies diverged from recomputed energies"

    # ---- end to end through the C ABI with HOST buffers: H2D of the int8 spins, the step, D2H of the energies
    e2e = None
    if not a.no_e2e:
        host_spins = torch.empty((w.S, 2, w.T, w.N), dtype=torch.int8).pin_memory()
        host_E = torch.empty((w.S, 2, w.T), dtype=torch.int32).pin_memory()
        hs, hE = host_spins.numpy(), host_E.numpy()
        B.pt_get_spins(out=hs)
        for _ in range(2):
            B.pt_set_spins(hs); step(); B.pt_get_energy(out=hE)
        barrier()
        t0 = time.perf_counter()
        for _ in range(a.e2e_steps):
            B.pt_set_spins(hs)
            step()
            B.pt_get_energy(out=hE)            # synchronises
        barrier()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * flips_step * a.e2e_steps / (dt * 1e9), "unit": UNIT,
               "h2d_bytes_per_step": int(hs.nbytes), "d2h_bytes_per_step": int(hE.nbytes),
               "steps": a.e2e_steps, "what": "pt_set_spins(host int8) + step + pt_get_energy(host), wall clock"}

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel of the timed region (INT32 issue; live CUDA-event launch times)
    peaks, peaks_kind = measured_peaks()
    f_ghz = (clocks["sm_mhz"] or peaks.get("sm_max_mhz", 1965.0)) / 1e3 if clocks else 1.965
    names = ["k_sweep", "k_houdayer", "k_exchange", "k_measure", "k_mcs"]
    dom = int(np.argmax(kms))
    if dom not in (0, 4):          # the roofline is quoted for the kernel that does the Metropolis sweeps
        dom = 4 if kn[4] > 0 else 0
    mcs_per_launch = 1 if dom == 0 else max(1, (a.mcs_per_step * a.steps) // max(int(kn[4]), 1))
    dom_ms = kms[dom] / max(int(kn[dom]), 1)
    flips_per_launch = w.flips_per_sweep() * mcs_per_launch
    dom_flips_ns = flips_per_launch / (dom_ms * 1e6) if dom_ms > 0 else 0.0
    A = ALGO_OPS_PER_FLIP[w.d]
    peak_ops = SM_COUNT * INT32_LANES_PER_SM_CLK * (peaks.get("sm_max_mhz", 1965.0) / 1e3)
    philox_ops, _ = B.pt_microbench(4, 8, 1000, device=dev)     # measured live: Philox-only ceiling
    roofline = {
        "bound": "alu", "kernel": names[dom], "achieved": A * dom_flips_ns, "peak": peak_ops,
        "unit": "Gop/s (INT32 thread-ops)", "frac": A * dom_flips_ns / peak_ops,
        "traffic": None if a.gaussian else NCU_DRAM_BYTES_PER_LAUNCH.get((w.name, names[dom])),
        "peak_how": "derived: 148 SMs x 128 INT32 lanes/clk (fma+alu pipes) x %.3f GHz max SM clock; A = %d algorithmic "
                    "ops/flip (Philox 10 + field 2d + decide 6); a %s launch = %d MCS = %d attempted flips" % (
                        peaks.get("sm_max_mhz", 1965.0) / 1e3, A, names[dom], mcs_per_launch, flips_per_launch),
        "flips_per_ns": dom_flips_ns, "ms_per_launch": dom_ms, "launches": int(kn[dom]),
        "philox_only_flips_per_ns": philox_ops / 10.0,
        "hbm": {"algorithmic_bytes_per_flip": 0.25 / mcs_per_launch, "achieved_gbs": 0.25 / mcs_per_launch * dom_flips_ns,
                "peak_gbs": peaks.get("hbm_gbs"), "peak_kind": peaks_kind,
                "frac": 0.25 / mcs_per_launch * dom_flips_ns / peaks.get("hbm_gbs", 6650.0)},
        "kernel_ms": {n: float(kms[i]) for i, n in enumerate(names)}, "step_total_ms": ms_total,
        "clock_ghz_during_run": f_ghz,
    }
    # the Metropolis sweeps alone (a1-a3; Eq. (11) normalisation), same state, after the timed region
    B.pt_set_profiling(True)
    for _ in range(5):
        B.pt_sweep(a.mcs_per_step)
    sms, sn = B.pt_get_kernel_times()
    B.pt_set_profiling(False)
    so = w.flips_per_sweep() * a.mcs_per_step / (sms[0] / max(int(sn[0]), 1) * 1e6)
    roofline["sweep_only"] = {"kernel": "k_sweep", "flips_per_ns": so, "frac": A * so / peak_ops,
                              "what": "pt_sweep(%d) launches, no Houdayer / exchange" % a.mcs_per_step}
    assert B.pt_recompute_energy()[1] == 0
    # the two measurement kernels alone (a6 and the NEXT-2 overlap profile), CUDA events around 20 calls each
    prof_d = torch.empty((w.S, w.T, w.d, w.L), dtype=torch.int32, device=dev)
    meas_us = {}
    for label, fn in (("overlap", lambda: B.pt_measure_overlap_device(Qrec[0], QLrec[0])),
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
        meas_us[label] = m0.elapsed_time(m1) / 20 * 1e3
    roofline["measurement_us_per_call"] = meas_us

    cpu = None
    if not a.no_cpu_baseline:
        S_cpu, mcs_cpu = 4, max(1, int(3.0e8 / (w.flips_per_sweep(4))))
        v, dt, flips = oracle_time(w, S_cpu, mcs_cpu, gaussian=a.gaussian, cluster=a.cluster)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": "%s restricted to the first %d samples x %d MCS (%.2e flips), same MCS order" % (w.name, S_cpu, mcs_cpu, flips)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms_total / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic", "config": config_of(a, w, world),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "fast_path": bool(B.pt_get_path()),
    }
    print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
