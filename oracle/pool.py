"""The CPU oracle on several host cores: independent oracle PROCESSES on disjoint ranges of the global sample index.

Every sample is a pure function of (seed, global sample index) (pin P8), so a run of S samples is the
concatenation of runs over any partition of [0, S) through `sample_offset` -- the paper's own way of using a multi-core
host ("24 disorder realizations in parallel").  The oracle itself stays single-threaded and untouched;
this module only starts processes and concatenates what they return.  TEST INFRASTRUCTURE ONLY, like the rest of
oracle/: tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it, the product
never does.  It holds none of the method's arithmetic.

Worker processes are *spawned* (not forked): the parent holds a CUDA context in the GPU tests and in bench.py.
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

    (L, d, T, betas, seed, g0, n, n_mcs, houdayer, measure_every, checkpoints) = job[:11]
    o = ref.Oracle(L, d, n, T, np.asarray(betas, dtype=np.float64), seed, g0)
    if len(job) > 11 and job[11] is not None:       # fixed-point couplings (NEXT-3): an input of the run, drawn per global sample
        import workloads as wl

        fbits = int(job[11])
        o.set_couplings_fixed(wl.gaussian_couplings_fixed(seed, n, d, L ** d, fbits, sample_offset=g0), fbits)
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

    def submit(self, w, g0, n, n_mcs, checkpoints=(), seed=None, gaussian_fbits=None):
        import workloads as wl

        job = (w.L, w.d, w.T, w.betas().tolist(), wl.SEED if seed is None else seed, int(g0), int(n), int(n_mcs),
               bool(w.houdayer), int(w.measure_every), tuple(checkpoints), gaussian_fbits)
        return self.ex.submit(run_chunk, job)

    def submit_all_samples(self, w, n_mcs, chunks_per_proc=2, gaussian_fbits=None):
        """All S samples of workload w in contiguous chunks; returns the list of futures."""
        n_chunks = min(w.S, self.procs * chunks_per_proc)
        edges = [round(k * w.S / n_chunks) for k in range(n_chunks + 1)]
        return [self.submit(w, a, b - a, n_mcs, gaussian_fbits=gaussian_fbits) for a, b in zip(edges[:-1], edges[1:]) if b > a]

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


# ---- persistent workers: P oracle processes that each keep one simulation alive and advance it on request (bench.py) ----

def _persistent_worker(conn, job):
    from oracle import ref

    (L, d, T, betas, seed, g0, n, houdayer, measure_every, fixed, n_clu) = job
    o = ref.Oracle(L, d, n, T, np.asarray(betas, dtype=np.float64), seed, g0)
    if fixed is not None:
        o.set_couplings_fixed(fixed[0], fixed[1])
    if n_clu is not None:
        o.set_cluster_moves(np.asarray(n_clu, dtype=np.int32))
    conn.send("ready")
    done = 0
    while True:
        msg = conn.recv()
        if msg is None:
            break
        for _ in range(int(msg)):                   # one MCS at a time, the measurement where the config asks for it (R26)
            o.mcs(1, 1, int(houdayer), True)
            done += 1
            if measure_every and done % measure_every == 0:
                o.measure_overlap()
        conn.send(done)
    o.close()
    conn.close()


class PersistentOracles:
    """P oracle processes on disjoint sample ranges [g0 + k n, g0 + (k + 1) n), each alive across step() calls."""

    def __init__(self, w, procs, samples_per_proc, houdayer_mode=None, fixed=None, n_clu=None, seed=None, g0=0):
        import workloads as wl

        ctx = mp.get_context("spawn")
        self.procs, self.conns = [], []
        hd = (1 if w.houdayer else 0) if houdayer_mode is None else houdayer_mode
        for k in range(procs):
            a, b = ctx.Pipe()
            fx = None if fixed is None else (fixed[0][k * samples_per_proc:(k + 1) * samples_per_proc], fixed[1])
            job = (w.L, w.d, w.T, w.betas().tolist(), wl.SEED if seed is None else seed, g0 + k * samples_per_proc,
                   samples_per_proc, hd, int(w.measure_every), fx, n_clu)
            p = ctx.Process(target=_persistent_worker, args=(b, job), daemon=True)
            p.start()
            self.procs.append(p)
            self.conns.append(a)
        for c in self.conns:
            assert c.recv() == "ready"

    def step(self, n_mcs):
        for c in self.conns:
            c.send(int(n_mcs))
        return [c.recv() for c in self.conns]

    def close(self):
        for c in self.conns:
            try:
                c.send(None)
            except Exception:
                pass
        for p in self.procs:
            p.join(timeout=5)
