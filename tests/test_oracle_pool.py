"""The multi-process oracle harness (oracle/pool.py) against the single-process oracle: a run over all samples
is the concatenation of runs over disjoint `sample_offset` ranges (pin P8)."""
import numpy as np

from oracle import ref
import workloads as wl
from oracle import pool as OP


def test_pool_of_oracle_processes_equals_one_oracle():
    w = wl.Workload("t", 2, 8, 6, 5, "geometric", 0.3, 1.5, 24, True, 10)
    pool = OP.OraclePool(3)
    try:
        futs = pool.submit_all_samples(w, 24)
        assert len(futs) == 6
        got, recs = OP.gather(futs, 24)
        one = pool.submit(w, 4, 2, 24, checkpoints=(10, 20)).result()
    finally:
        pool.close()
    o = ref.Oracle(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    want_recs = []
    for m in range(1, 25):
        o.mcs(1, 1, True, True)
        if m % 10 == 0:
            want_recs.append(o.measure_overlap())
        if m == 20:
            mid = o.state()
    want = o.state()
    for k in OP.STATE_KEYS:
        assert np.array_equal(got[k], want[k]), k
        assert np.array_equal(one[2][24][k], want[k][4:6]), k
        assert np.array_equal(one[2][20][k], mid[k][4:6]), k
    Q, QL = o.measure_overlap()
    assert np.array_equal(got["Q"], Q) and np.array_equal(got["QL"], QL)
    assert len(recs) == 2 and len(one[3]) == 2
    for (a, b), (c, e) in zip(recs, want_recs):
        assert np.array_equal(a, c) and np.array_equal(b, e)
    assert sorted(one[2]) == [10, 20, 24]


def test_persistent_oracle_processes_advance_like_one_oracle():
    w = wl.Workload("t", 3, 4, 4, 3, "geometric", 0.4, 1.1, 0, False, 0)
    po = OP.PersistentOracles(w, 2, 2)
    try:
        assert po.step(3) == [3, 3]
        assert po.step(2) == [5, 5]
    finally:
        po.close()
