"""The CPU oracle on several host cores: independent oracle PROCESSES on disjoint ranges of the global sample index.

Every sample is a pure function of (seed, global sample index) (pin P8), so a run of S samples is the
concatenation of runs over any partition of [0, S) through `sample_offset` -- the paper's own way of using a multi-core
host ("24 disorder realizations in parallel").  The oracle itself stays single-threaded and untouched;
this module only starts processes and concatenates what they return.  TEST INFRASTRUCTURE ONLY (it imports oracle/).

Worker processes are *spawned* (not forked): the parent holds a CUDA context in the GPU tests.
"""
from __future__ import annotations

import multiprocessing as mp
import os
from concurrent.futures import ProcessPoolExecutor

import numpy as np

STATE_KEYS = ("spins", "energy", "temp_of_slot", "slot_of_temp", "attempts", "accepts", "last_size", "cum_size")


def n_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def run_chunk(job):
    """One oracle process: samples [g0, g0 + n) of a workload for n_mcs MCS in the paper's order,
    the overlap measurement after every measure_every-th MCS (R26).  Returns {checkpoint: state dict} for the MCS
    numbers in `checkpoints`, the overlap records, and the overlaps after the last MCS."""
    from oracle import ref

    (L, d, T, betas, seed, g0, n, n_mcs, houdayer, measure_every, checkpoints) = job
    o = ref.Oracle(L, d, n, T, np.asarray(betas, dtype=np.float64), seed, g0)
    states, recs = {}, []
    done = 0
    stops = sorted(set(int(c) for c in checkpoints if 0 < c <= n_mcs) | {n_mcs})
    for stop in stops:
        while done < stop:
            step = stop - done
            if measure_every:
                step = min(step, measure_every - done % measure_every)
            o.mcs(step, 1, int(houdayer), True)
            done += step
            if measure_every and done % measure_every == 0:
                recs.append(o.measure_overlap())
        st = o.state()
        st["Q"], st["QL"] = o.measure_overlap()
        states[stop] = st
    o.close()
    return g0, n, states, recs


class OraclePool:
    def __init__(self, procs: int | None = None):
        self.procs = procs or n_cores()
        self.ex = ProcessPoolExecutor(max_workers=self.procs, mp_context=mp.get_context("spawn"))

    def submit(self, w, g0, n, n_mcs, checkpoints=(), seed=None):
        from paper_2003_04621_b200 import workloads as wl

        job = (w.L, w.d, w.T, w.betas().tolist(), wl.SEED if seed is None else seed, int(g0), int(n), int(n_mcs),
               bool(w.houdayer), int(w.measure_every), tuple(checkpoints))
        return self.ex.submit(run_chunk, job)

    def submit_all_samples(self, w, n_mcs, chunks_per_proc=2):
        """All S samples of workload w in contiguous chunks; returns the list of futures."""
        n_chunks = min(w.S, self.procs * chunks_per_proc)
        edges = [round(k * w.S / n_chunks) for k in range(n_chunks + 1)]
        return [self.submit(w, a, b - a, n_mcs) for a, b in zip(edges[:-1], edges[1:]) if b > a]

    def close(self):
        self.ex.shutdown(wait=False, cancel_futures=True)


def gather(futures, n_mcs):
    """Concatenate the per-chunk results of submit_all_samples along the sample axis."""
    parts = sorted((f.result() for f in futures), key=lambda r: r[0])
    out = {k: np.concatenate([p[2][n_mcs][k] for p in parts], axis=0) for k in STATE_KEYS + ("Q", "QL")}
    n_rec = len(parts[0][3])
    recs = [(np.concatenate([p[3][r][0] for p in parts], axis=0), np.concatenate([p[3][r][1] for p in parts], axis=0))
            for r in range(n_rec)]
    return out, recs
