"""SURVEY 8(d) parity subset (ii): samples {0, 1, S/2, S-1} (two for C5) of C2-C5 for the config's WHOLE run of 10^4 MCS,
at full S, L, T in bench.py's launch configuration (50 MCS per pt_mcs call; C3 with its overlap records fused into the
MCS launch), compared bit for bit with the oracle at MCS 10, 100, 1000 and 10^4 on the full state of the sample, and on
every one of C3's 1000 overlap records.

The oracle needs about 20 s (C2), 10 s (C3), 1.5 min (C4) and 8 min (C5) per sample on one host core, so all fourteen
oracle runs are started as separate processes (oracle/pool.py) when the test session starts (tests/conftest.py) and
this module -- collected last -- only waits for what is still running: about the C5 time on a host with >= 14 cores.
Run on the B200 box with `-m gpu`; deselect with `-m "gpu and not fulllength"` while iterating."""
import numpy as np
import pytest

from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod
import workloads as wl
from oracle import pool as OP
from tests.conftest import FULL_LENGTH_SAMPLES, full_length_jobs

pytestmark = [pytest.mark.gpu, pytest.mark.fulllength]
CHECKPOINTS = (10, 100, 1000, 10000)


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()
    yield
    B.pt_free()


@pytest.mark.parametrize("name", ["C3", "C2", "C4", "C5"])
def test_whole_run_of_sampled_samples_against_the_oracle(name):
    import torch

    w = wl.CONFIGS[name]
    assert w.n_mcs == CHECKPOINTS[-1]
    gs = FULL_LENGTH_SAMPLES[name](w.S)
    jobs = full_length_jobs()
    # ---- the GPU run: the whole config, 50 MCS per call as in bench.py
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    n_rec = 50 // w.measure_every if w.measure_every else 0
    Qr = torch.empty((max(n_rec, 1), w.S, w.T), dtype=torch.int32, device="cuda")
    QLr = torch.empty_like(Qr)
    gpu_states, gpu_recs = {}, []
    done = 0
    while done < w.n_mcs:
        n = min(50, min(c for c in CHECKPOINTS if c > done) - done)
        if w.measure_every:
            assert done % w.measure_every == 0 and n % w.measure_every == 0
            B.pt_mcs_measure_device(n, 1, w.houdayer, True, w.measure_every, Qr, QLr)
            q, ql = Qr.cpu().numpy(), QLr.cpu().numpy()
            gpu_recs += [(q[r][gs].copy(), ql[r][gs].copy()) for r in range(n // w.measure_every)]
        else:
            B.pt_mcs(n, 1, w.houdayer, True)
        done += n
        if done in CHECKPOINTS:
            st = B.state()
            st["Q"], st["QL"] = B.pt_measure_overlap()
            gpu_states[done] = {k: st[k][gs].copy() for k in OP.STATE_KEYS + ("Q", "QL")}
    assert B.pt_recompute_energy()[1] == 0
    assert tuple(B.pt_get_counters()) == (w.n_mcs, w.n_mcs, w.n_mcs if w.houdayer else 0)
    # ---- against the oracle processes, one per sampled sample
    for i, g in enumerate(gs):
        g0, n, states, recs = jobs[(name, g)].result()
        assert (g0, n) == (g, 1) and sorted(states) == list(CHECKPOINTS)
        for c in CHECKPOINTS:
            for k in OP.STATE_KEYS + ("Q", "QL"):
                assert np.array_equal(states[c][k][0], gpu_states[c][k][i]), "%s sample %d after %d MCS: %s differs" % (name, g, c, k)
        assert len(recs) == len(gpu_recs) == (w.n_mcs // w.measure_every if w.measure_every else 0)
        for r, ((qa, qla), (qb, qlb)) in enumerate(zip(recs, gpu_recs)):
            assert np.array_equal(qa[0], qb[i]) and np.array_equal(qla[0], qlb[i]), "%s sample %d: overlap record %d differs" % (name, g, r)
