import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# SURVEY 8(d) parity subset (ii): the samples whose whole 10^4-MCS run is recomputed by the oracle (two suffice for C5)
FULL_LENGTH_SAMPLES = {
    "C2": lambda S: [0, 1, S // 2, S - 1],
    "C3": lambda S: [0, 1, S // 2, S - 1],
    "C4": lambda S: [0, 1, S // 2, S - 1],
    "C5": lambda S: [0, S - 1],
}
_full_length = {"pool": None, "jobs": None}


def full_length_jobs():
    """{(config, global sample): future} of the oracle processes of tests/test_gpu_zz_fulllength.py.  Started once, as
    early as possible (at collection, when a GPU is there and such a test is selected), so that they run on otherwise
    idle host cores while the other GPU tests execute; longest first."""
    if _full_length["jobs"] is None:
        import workloads as wl
        from oracle import pool as OP
        from oracle import ref

        ref.build()                                  # once, before the workers race for it
        pool = OP.OraclePool(14)
        jobs = {}
        for name in ("C5", "C4", "C2", "C3"):
            w = wl.CONFIGS[name]
            for g in FULL_LENGTH_SAMPLES[name](w.S):
                jobs[(name, g)] = pool.submit(w, g, 1, w.n_mcs, checkpoints=(10, 100, 1000, w.n_mcs))
        _full_length["pool"], _full_length["jobs"] = pool, jobs
    return _full_length["jobs"]


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "fulllength: whole 10^4-MCS runs against the oracle (minutes of host time)")


@pytest.hookimpl(trylast=True)          # after the -m / -k deselection
def pytest_collection_modifyitems(config, items):
    import torch

    if torch.cuda.is_available():
        if any("fulllength" in item.keywords for item in items):
            full_length_jobs()
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_sessionfinish(session, exitstatus):
    if _full_length["pool"] is not None:
        _full_length["pool"].close()
