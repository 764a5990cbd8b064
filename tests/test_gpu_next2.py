"""GPU parity of the NEXT-2 row: overlap profiles per axis, bit for bit against the oracle, on the fast
and the general path, after real dynamics, plus its invariants at full size.  Run with `-m gpu`."""
import numpy as np
import pytest

from oracle import ref
from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod
import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()
    yield
    B.pt_free()


@pytest.mark.parametrize("L,d,S,T", [(8, 2, 3, 5), (16, 2, 2, 3), (32, 2, 2, 6), (64, 2, 2, 3), (128, 2, 1, 3), (256, 2, 1, 2),
                                     (8, 3, 2, 4), (16, 3, 2, 3), (32, 3, 1, 2),
                                     (2, 2, 2, 3), (6, 2, 2, 4), (10, 3, 1, 2), (4, 3, 2, 3)])
def test_profile_matches_oracle(L, d, S, T):
    betas = wl.betas_geometric(0.3, 1.5, T)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 2)
    B.pt_open(L, d, S, T, betas, wl.SEED, 2)
    assert np.array_equal(o.measure_overlap_profile(), B.pt_measure_overlap_profile())
    o.mcs(9, 1, True, True); B.pt_mcs(9, 1, True, True)
    prof = B.pt_measure_overlap_profile()
    assert np.array_equal(o.measure_overlap_profile(), prof)
    Q, _ = B.pt_measure_overlap()
    assert (prof.sum(axis=3) == Q[:, :, None]).all()
    assert B.pt_get_counters() == (9, 9, 9)              # a measurement advances nothing


@pytest.mark.parametrize("name", ["C3", "C5"])
def test_profile_full_size_invariants_and_sampled_parity(name):
    w = wl.CONFIGS[name]
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    B.pt_mcs(10, 1, w.houdayer, True)
    prof = B.pt_measure_overlap_profile()
    Q, _ = B.pt_measure_overlap()
    assert (prof.sum(axis=3) == Q[:, :, None]).all()
    plane = w.N // w.L
    assert ((prof - plane) % 2 == 0).all() and (abs(prof) <= plane).all()
    for g in (0, w.S - 1):
        o = ref.Oracle(w.L, w.d, 1, w.T, w.betas(), wl.SEED, g)
        o.mcs(10, 1, w.houdayer, True)
        assert np.array_equal(o.measure_overlap_profile()[0], prof[g])
