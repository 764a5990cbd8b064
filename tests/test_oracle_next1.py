"""Pins of the oracle's NEXT-1 parts: the temperature-schedule family of Eq. (6)-(7)
and the round-trip (tunnelling-time) bookkeeping (readings R27-R29 in DESIGN.md).
Pinned against closed forms and special cases, not against the oracle's own formula."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import ref
import workloads as wl


# ---- P11: schedule family ----------------------------------------------------------------------------------

def test_schedule_phi_one_is_linear_and_hits_both_ends():
    # "the case phi = 1 corresponds to a linear schedule"; Fig. 3's parameters
    T, b = ref.schedule_family(0.2, 1.5, 32, 1.0)
    lin = np.array([float(Fraction(2, 10) + Fraction(13, 10) * Fraction(i, 31)) for i in range(32)])
    assert np.allclose(T, lin, rtol=4e-16, atol=0)
    assert T[0] == 0.2 and abs(T[-1] - 1.5) <= 2e-16 * 1.5
    assert np.allclose(b * T, 1.0, rtol=4e-16)


@pytest.mark.parametrize("phi,num,den", [(2.0, 2, 1), (0.5, 1, 2), (3.0, 3, 1)])
def test_schedule_closed_forms_for_rational_exponents(phi, num, den):
    # T_i = (i / (N_T - 1))^phi (T_max - T_min) + T_min, evaluated exactly with rationals / integer roots
    NT, Tmin, Tmax = 17, Fraction(1, 5), Fraction(3, 2)
    T, _ = ref.schedule_family(float(Tmin), float(Tmax), NT, phi)
    for i in range(NT):
        x = Fraction(i, NT - 1) ** num
        exact = float(x) ** (1.0 / den) * float(Tmax - Tmin) + float(Tmin)
        assert abs(T[i] - exact) <= 1e-14
    assert T[0] == float(Tmin) and abs(T[-1] - float(Tmax)) < 1e-15


def test_schedule_density_moves_with_phi_as_in_fig3():
    # phi < 1: spacing denser towards higher temperatures; phi > 1: denser towards lower
    for phi in (0.5, 0.8):
        T, _ = ref.schedule_family(0.2, 1.5, 32, phi)
        d = np.diff(T)
        assert (d > 0).all() and (np.diff(d) < 0).all()
    for phi in (1.5, 3.0):
        T, _ = ref.schedule_family(0.2, 1.5, 32, phi)
        d = np.diff(T)
        assert (d > 0).all() and (np.diff(d) > 0).all()
    T1, _ = ref.schedule_family(0.7, 0.7, 1, 1.3)
    assert T1.tolist() == [0.7]
    for bad in [(0.0, 1.0, 4, 1.0), (1.0, 0.5, 4, 1.0), (0.2, 1.5, 0, 1.0), (0.2, 1.5, 4, 0.0), (0.2, 1.5, 4, -1.0)]:
        with pytest.raises(ValueError):
            ref.schedule_family(*bad)


# ---- P12: round trips --------------------------------------------------------------------------------------

@pytest.mark.parametrize("T", [2, 3, 5, 8])
def test_round_trips_equal_betas_closed_form(T):
    """All betas equal => every proposal is accepted and a pass is a cyclic shift (pin P4): the slot at index 0
    jumps to index T-1, every other slot moves down one index.  Slot r therefore first sits at index 0 after pass
    n = r, reaches the far end one pass later and completes a round trip every T passes:
    trips[r] = floor((n - r) / T), every round-trip time equals T."""
    S, n_pass = 2, 37
    o = ref.Oracle(4, 2, S, T, np.full(T, 0.3), wl.SEED)
    for n in range(1, n_pass + 1):
        o.exchange()
        trips, tau_sum, tau_cnt = o.get_round_trips()
        expect = np.array([(n - r) // T if n >= r else 0 for r in range(T)], dtype=np.uint32)
        assert (trips == expect[None, None, :]).all(), (n, trips[0, 0], expect)
        assert (tau_sum == tau_cnt * T).all()
    # completions happen at n = r + kT (k >= 1): count them per bin floor(log2 n)
    cnt = np.zeros(32, dtype=np.uint64)
    for r in range(T):
        for n in range(r + T, n_pass + 1, T):
            cnt[int(np.log2(n))] += 1
    assert (tau_cnt == cnt[None, None, :]).all()


def test_round_trips_single_temperature_and_no_passes():
    o = ref.Oracle(4, 2, 1, 1, np.array([0.5]), wl.SEED)
    o.mcs(5, 1, False, True)
    trips, tau_sum, tau_cnt = o.get_round_trips()
    assert trips.sum() == 0 and tau_sum.sum() == 0 and tau_cnt.sum() == 0
    o = ref.Oracle(4, 2, 1, 4, wl.betas_linear(0.2, 1.0, 4), wl.SEED)
    o.sweep(3)
    assert o.get_round_trips()[0].sum() == 0


def test_round_trips_replay_from_the_permutation_history():
    """On a real run the statistics must equal a replay of the definition from the recorded slot_of_temp history
    (a different route: numpy on history arrays, one replica followed at a time), and the trips of a chain tile
    disjoint time intervals, so sum(tau) <= T * n."""
    L, d, S, T, n_pass = 4, 2, 3, 5, 400
    betas = wl.betas_geometric(0.1, 0.6, T)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED)
    hist = [o.get_perm()[0].copy()]                       # temp_of_slot after 0, 1, ... passes
    for _ in range(n_pass):
        o.mcs(1, 1, True, True)
        hist.append(o.get_perm()[0].copy())
    hist = np.stack(hist)                                 # [n+1][S][2][T(slot)]
    trips, tau_sum, tau_cnt = o.get_round_trips()
    assert trips.sum() > 0
    exp_trips = np.zeros_like(trips)
    exp_sum = np.zeros_like(tau_sum)
    exp_cnt = np.zeros_like(tau_cnt)
    for s in range(S):
        for c in range(2):
            for r in range(T):
                path = hist[:, s, c, r]                   # temperature index of this replica over time
                started, far, t0 = False, False, 0
                for n, t in enumerate(path):
                    if t == T - 1 and started:
                        far = True
                    if t == 0:
                        if started and far:
                            exp_trips[s, c, r] += 1
                            exp_sum[s, c, int(np.log2(n))] += n - t0
                            exp_cnt[s, c, int(np.log2(n))] += 1
                            t0, far = n, False
                        elif not started:
                            started, t0 = True, n
    assert np.array_equal(trips, exp_trips)
    assert np.array_equal(tau_sum, exp_sum) and np.array_equal(tau_cnt, exp_cnt)
    assert (tau_sum.sum(axis=2) <= T * n_pass).all()
    assert np.array_equal(tau_cnt.sum(axis=2), trips.sum(axis=2))


def test_round_trips_do_not_depend_on_sharding():
    T, n = 4, 120
    betas = wl.betas_geometric(0.1, 0.5, T)
    full = ref.Oracle(4, 2, 4, T, betas, wl.SEED, 0)
    part = ref.Oracle(4, 2, 2, T, betas, wl.SEED, 2)
    full.mcs(n, 1, False, True)
    part.mcs(n, 1, False, True)
    for a, b in zip(full.get_round_trips(), part.get_round_trips()):
        assert np.array_equal(a[2:], b)
