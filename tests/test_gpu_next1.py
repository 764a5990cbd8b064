"""GPU parity of the NEXT-1 row: round-trip bookkeeping inside the PT pass, on the schedule family of
Eq. (6)-(7), through the C ABI, bit for bit against the oracle -- separate kernels, fused kernel, chain-split fused
kernel, general-L path -- plus the equal-beta closed form on the device.  Run with `-m gpu`."""
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


def same_round_trips(o):
    for a, b, name in zip(o.get_round_trips(), B.pt_get_round_trips(), ("trips", "tau_sum", "tau_cnt")):
        assert np.array_equal(a, b), name


@pytest.mark.parametrize("L,d,S,T,phi,houd,general", [
    (8, 2, 3, 6, 0.7, True, False), (32, 2, 2, 12, 1.0, True, False), (8, 3, 2, 5, 1.6, False, False),
    (16, 3, 2, 40, 1.2, False, False),        # T*W >= 512: chain-split fused kernel
    (6, 2, 2, 5, 0.9, True, True), (64, 2, 1, 4, 2.0, True, False)])
def test_round_trips_match_oracle(L, d, S, T, phi, houd, general):
    _, betas = B.pt_schedule_family(0.6, 4.0, T, phi)          # hot ladder: many round trips in a short run
    _, betas_o = ref.schedule_family(0.6, 4.0, T, phi)
    assert np.array_equal(betas, betas_o)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 3)
    B.pt_open(L, d, S, T, betas, wl.SEED, 3, general=general, track_round_trips=True)
    for _ in range(10):                                        # separate kernels
        o.sweep(1); B.pt_sweep(1)
        if houd:
            o.houdayer_step(); B.houdayer_step()
        o.exchange(); B.pt_exchange()
    same_round_trips(o)
    for n in (1, 7, 150):                                      # fused where eligible
        o.mcs(n, 1, houd, True); B.pt_mcs(n, 1, houd, True)
        same_round_trips(o)
    if L == 8 and d == 2:
        assert B.pt_get_round_trips()[0].sum() > 0
    a, b = o.state(), B.state()
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_equal_betas_closed_form_on_device():
    T, S, n = 5, 3, 43
    B.pt_open(8, 2, S, T, np.full(T, 0.4), wl.SEED, track_round_trips=True)
    B.pt_mcs(n, 1, False, True)
    trips, tau_sum, tau_cnt = B.pt_get_round_trips()
    expect = np.array([(n - r) // T for r in range(T)], dtype=np.uint32)
    assert (trips == expect[None, None, :]).all()
    assert (tau_sum == tau_cnt * T).all() and tau_cnt.sum() == trips.sum()


def test_tracking_off_and_late_enable_are_state_errors():
    B.pt_open(8, 2, 1, 3, wl.betas_linear(0.2, 1.0, 3), wl.SEED)
    with pytest.raises(B.PTError) as e:
        B.pt_get_round_trips()
    assert e.value.code == B.PT_ERR_STATE
    with pytest.raises(B.PTError) as e:
        B.pt_set_round_trip_tracking(1)
    assert e.value.code == B.PT_ERR_STATE


def test_full_size_C2_round_trips_sampled():
    """C2 at full size in bench.py's launch configuration with tracking on: sampled samples against the oracle."""
    w = wl.C2
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, track_round_trips=True)
    B.pt_mcs(150, 1, True, True)
    trips, tau_sum, tau_cnt = B.pt_get_round_trips()
    assert np.array_equal(tau_cnt.sum(axis=2), trips.sum(axis=2))
    for g in (0, w.S - 1):
        o = ref.Oracle(w.L, w.d, 1, w.T, w.betas(), wl.SEED, g)
        o.mcs(150, 1, True, True)
        to, so, co = o.get_round_trips()
        assert np.array_equal(to[0], trips[g]) and np.array_equal(so[0], tau_sum[g]) and np.array_equal(co[0], tau_cnt[g])


# ---- NEXT-4: general p in Eq. (2) ------------------------------------------------------------------------------

@pytest.mark.parametrize("p", [0.0, 0.3, 0.5, 0.85, 1.0])
def test_general_p_couplings_and_dynamics_match_oracle(p):
    L, d, S, T = 16, 2, 3, 4
    betas = wl.betas_geometric(0.3, 1.2, T)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 1, p_ferro=p)
    B.pt_open(L, d, S, T, betas, wl.SEED, 1, p_ferro=p)
    assert np.array_equal(o.get_couplings(), B.pt_get_couplings())
    o.mcs(12, 1, True, True); B.pt_mcs(12, 1, True, True)
    a, b = o.state(), B.state()
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert B.pt_recompute_energy()[1] == 0
    if p == 0.5:
        o2 = ref.Oracle(L, d, S, T, betas, wl.SEED, 1)
        assert np.array_equal(o2.get_couplings(), B.pt_get_couplings())


def test_general_p_argument_and_state_errors():
    B.pt_open(8, 2, 1, 2, wl.betas_linear(0.2, 1.0, 2), wl.SEED)
    with pytest.raises(B.PTError) as e:
        B.pt_set_coupling_probability(0.3)                   # after pt_init
    assert e.value.code == B.PT_ERR_STATE
    import torch
    ws = torch.empty(B.pt_workspace_bytes(8, 2, 1, 2), dtype=torch.uint8, device="cuda:0")
    B.pt_bind(ws)
    with pytest.raises(B.PTError) as e:
        B.pt_set_coupling_probability(1.5)
    assert e.value.code == B.PT_ERR_ARG
