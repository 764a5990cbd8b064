"""Pins P1-P4, P6-P9 of the CPU oracle: known answers, closed forms, invariants, special
cases, brute force and library routines -- each chosen so that a plausible mistake in the oracle (dropped term,
wrong sign or index, transposed operand) fails at least one.  CPU only."""
import json
import math
import os

import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SEED = wl.SEED


def hexs(v):
    return ["%08x" % int(x) for x in v]


# ------------------------------------------------------------------ P1 Philox known answers

def test_p1_philox_known_answers():
    with open(os.path.join(GOLD, "philox_known_answers.json")) as f:
        vecs = json.load(f)["vectors"]
    for v in vecs:
        out = ref.philox([int(k, 16) for k in v["key"]], [int(c, 16) for c in v["ctr"]])
        assert hexs(out) == v["out"]


def test_p1_philox_against_independent_numpy():
    rng = np.random.default_rng(1)
    ctr = rng.integers(0, 2 ** 32, size=(64, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=2, dtype=np.uint64).astype(np.uint32)
    want = H.philox_np(key, ctr)
    for n in range(64):
        assert (ref.philox(key, ctr[n]) == want[n]).all()


# ------------------------------------------------------------------ P2 energy / indexing, P9 init

@pytest.mark.parametrize("L,d", [(2, 2), (4, 2), (6, 2), (8, 2), (2, 3), (4, 3), (6, 3)])
def test_p2_energy_bruteforce_gauge_flip(L, d):
    T = 3
    o = ref.Oracle(L, d, 2, T, [0.3, 0.7, 1.1], SEED)
    J, s = o.get_couplings(), o.get_spins()
    E, bad = o.recompute_energy()
    assert bad == 0
    N = L ** d
    for smp in range(2):
        for c in range(2):
            for r in range(T):
                assert E[smp, c, r] == H.energy_bruteforce(J[smp], s[smp, c, r], L, d)
    # (v) E = dN (mod 2); replicas of one sample agree mod 4 (R22b)
    assert ((E - d * N) % 2 == 0).all()
    for smp in range(2):
        assert len(set((E[smp].ravel() % 4).tolist())) == 1
    # (iii) global flip
    o.set_spins(-s)
    assert (o.recompute_energy()[0] == E).all()
    # (i) gauge invariance: s_i -> eps_i s_i, J_ij -> eps_i eps_j J_ij
    rng = np.random.default_rng(5)
    eps = (rng.integers(0, 2, size=N) * 2 - 1).astype(np.int8)
    nbr = H.neighbour_list(L, d)
    Jg = J.copy()
    for mu in range(d):
        Jg[:, mu, :] = J[:, mu, :] * eps[None, :] * eps[nbr[:, 2 * mu]][None, :]
    o.set_couplings(Jg)
    o.set_spins(s * eps[None, None, None, :])
    assert (o.recompute_energy()[0] == E).all()


@pytest.mark.parametrize("L,d", [(2, 2), (4, 2), (8, 2), (2, 3), (4, 3)])
def test_p2_ferromagnet_ground_state(L, d):
    o = ref.Oracle(L, d, 1, 2, [0.5, 1.0], SEED)
    N = L ** d
    o.set_couplings(np.ones((1, d, N), dtype=np.int8))
    o.set_spins(np.ones((1, 2, 2, N), dtype=np.int8))
    assert (o.recompute_energy()[0] == -d * N).all()
    # one flipped spin costs 2 per bond touching it: 2 * 2d
    s = np.ones((1, 2, 2, N), dtype=np.int8)
    s[..., N // 2] = -1
    o.set_spins(s)
    assert (o.recompute_energy()[0] == -d * N + 4 * d).all()


def test_p9_init_balance_and_key_independence():
    o = ref.Oracle(16, 2, 8, 4, [0.1, 0.2, 0.3, 0.4], SEED)
    J, s = o.get_couplings(), o.get_spins()
    assert abs(int(J.sum())) < 5 * math.sqrt(J.size)
    assert abs(int(s.sum())) < 5 * math.sqrt(s.size)
    assert set(np.unique(J).tolist()) == {-1, 1} and set(np.unique(s).tolist()) == {-1, 1}
    # J of (sample g, mu, i) does not depend on L, S, T (the counter has no such field)
    o2 = ref.Oracle(4, 2, 3, 2, [0.5, 0.6], SEED)
    assert (o2.get_couplings()[:, :, :16] == J[:3, :, :16]).all()
    assert (o2.get_spins()[:, :, :, :16] == s[:3, :, :2, :16]).all()
    # different seed -> different couplings
    o3 = ref.Oracle(16, 2, 8, 4, [0.1, 0.2, 0.3, 0.4], SEED + 1)
    assert (o3.get_couplings() != J).mean() > 0.4


def test_init_rejects_bad_arguments():
    b = np.array([0.5, 1.0])
    for args in [(3, 2, 1, 2), (8, 4, 1, 2), (8, 2, 0, 2), (0, 2, 1, 2), (8, 1, 1, 2)]:
        with pytest.raises(ValueError):
            ref.Oracle(*args, b, SEED)
    with pytest.raises(ValueError):
        ref.Oracle(8, 2, 1, 2, np.array([0.5, -1.0]), SEED)
    with pytest.raises(ValueError):
        ref.Oracle(8, 2, 1, 2, np.array([0.5, float("nan")]), SEED)


# ------------------------------------------------------------------ P3 Metropolis half-sweeps

@pytest.mark.parametrize("L,d", [(4, 2), (8, 2), (4, 3), (2, 3)])
def test_p3_beta_zero_flips_everything(L, d):
    o = ref.Oracle(L, d, 2, 2, [0.0, 0.0], SEED)
    s0, E0 = o.get_spins(), o.recompute_energy()[0]
    assert (o.get_thresholds(2)[0] == 2 ** 32 - 1).all()
    o.sweep(1)
    assert (o.get_spins() == -s0).all()          # every site flips (barring a 2^-32 event)
    assert (o.recompute_energy()[0] == E0).all()
    assert o.recompute_energy()[1] == 0
    o.sweep(1)
    assert (o.get_spins() == s0).all()
    assert o.get_counters() == (2, 0, 0)


@pytest.mark.parametrize("L,d", [(8, 2), (4, 3)])
def test_p3_beta_large_is_deterministic_descent(L, d):
    o = ref.Oracle(L, d, 3, 2, [50.0, 50.0], SEED)
    assert (o.get_thresholds(2)[0] == 0).all()
    J = o.get_couplings()
    nbr, col = H.neighbour_list(L, d), H.colours(L, d)
    N = L ** d
    prev = o.get_energy()
    for _ in range(6):
        s = o.get_spins().astype(np.int64)
        # independent restatement: with all thresholds 0 a site flips iff a = s_i * h_i <= 0, colour by colour
        for p in (0, 1):
            h = np.zeros_like(s)
            for mu in range(d):
                up, dn = nbr[:, 2 * mu], nbr[:, 2 * mu + 1]
                h += J[:, None, None, mu, :] * s[..., up] + J[:, None, None, mu, :][..., dn] * s[..., dn]
            flip = (s * h <= 0) & (col == p)[None, None, None, :]
            s = np.where(flip, -s, s)
        o.sweep(1)
        assert (o.get_spins() == s).all()
        E = o.get_energy()
        assert (E <= prev).all()                  # energy never increases at T = 0
        assert o.recompute_energy()[1] == 0
        prev = E


def test_p3_incremental_energy_matches_recompute_and_threshold_values():
    w = wl.C1
    o = ref.Oracle(w.L, w.d, w.S, w.T, w.betas(), SEED)
    for _ in range(20):
        o.sweep(3)
        assert o.recompute_energy()[1] == 0
    thrM, _ = o.get_thresholds(2)
    for t, b in enumerate(w.betas()):
        for k in (1, 2):
            p = math.exp(-4 * k * b)
            assert 0 <= p - thrM[t, k - 1] / 2.0 ** 32 < 2.0 ** -32 + 1e-18


def test_p3_sweep_against_vectorised_restatement():
    """One whole sweep re-derived with numpy (simultaneous update of a colour => also shows order independence
    within a colour, P3(v)) and the test-side Philox.  A second reading of 8(c).3, not the oracle's code."""
    L, d, S, T = 6, 3, 2, 3
    betas = np.array([0.3, 0.6, 0.9])
    o = ref.Oracle(L, d, S, T, betas, SEED, sample_offset=7)
    o.exchange()  # make temp_of_slot non-trivial first
    J, s = o.get_couplings().astype(np.int64), o.get_spins().astype(np.int64)
    tos, _ = o.get_perm()
    thrM, _ = o.get_thresholds(2)
    nbr, col = H.neighbour_list(L, d), H.colours(L, d)
    N = L ** d
    i = np.arange(N)
    key = (SEED & 0xFFFFFFFF, SEED >> 32)
    for n in range(2):
        for p in (0, 1):
            for smp in range(S):
                for c in range(2):
                    for r in range(T):
                        ctr = np.stack([i >> 3, np.full(N, n), np.full(N, 7 + smp),
                                        np.full(N, (3 << 28) | (p << 24) | (c << 16) | r)], axis=-1).astype(np.uint32)
                        u = H.philox_np(key, ctr)[i, (i >> 1) & 3].astype(np.int64)
                        sp = s[smp, c, r]
                        h = np.zeros(N, dtype=np.int64)
                        for mu in range(d):
                            up, dn = nbr[:, 2 * mu], nbr[:, 2 * mu + 1]
                            h += J[smp, mu] * sp[up] + J[smp, mu][dn] * sp[dn]
                        a = sp * h
                        thr = thrM[tos[smp, c, r]].astype(np.int64)[np.clip(a // 2 - 1, 0, d - 1)]
                        flip = ((a <= 0) | (u < thr)) & (col == p)
                        s[smp, c, r] = np.where(flip, -sp, sp)
        o.sweep(1)
        assert (o.get_spins() == s).all()


# ------------------------------------------------------------------ P4 PT pass

def test_p4_equal_betas_is_cyclic_shift():
    T = 6
    o = ref.Oracle(4, 2, 3, T, [0.7] * T, SEED)
    s0, E0 = o.get_spins(), o.recompute_energy()[0]
    o.exchange()
    tos, sot = o.get_perm()
    assert (sot == np.array([1, 2, 3, 4, 5, 0])).all()
    assert (tos == np.array([5, 0, 1, 2, 3, 4])).all()
    att, acc = o.get_swap_counts()
    assert (att == 1).all() and (acc == 1).all()
    assert (o.get_spins() == s0).all() and (o.recompute_energy()[0] == E0).all()


def test_p4_maps_stay_inverse_and_single_temperature_noop():
    w = wl.C1
    o = ref.Oracle(w.L, w.d, w.S, w.T, w.betas()[::-1].copy(), SEED)   # decreasing betas also legal (R7)
    ar = np.arange(w.T)
    for _ in range(50):
        o.sweep(1)
        o.exchange()
        tos, sot = o.get_perm()
        assert (np.take_along_axis(tos, sot, axis=2) == ar).all()
        assert (np.sort(sot, axis=2) == ar).all()
    att, acc = o.get_swap_counts()
    assert (att == 50).all() and (acc <= att).all()
    # energies by temperature are a permutation of energies by slot
    E_slot, _ = o.recompute_energy()
    assert (o.get_energy() == np.take_along_axis(E_slot, sot, axis=2)).all()
    o1 = ref.Oracle(4, 2, 2, 1, [0.5], SEED)
    o1.exchange()
    assert o1.get_counters() == (0, 1, 0)
    assert (o1.get_perm()[0] == 0).all()


def test_p4_decision_equals_eq5_in_double():
    """thrX within 2^-32 of exp(-4m|dbeta|); and one pass re-derived from Eq. (5) with the test-side Philox."""
    betas = np.array([0.2, 0.9, 0.5, 0.5, 1.7])
    T = len(betas)
    o = ref.Oracle(6, 2, 4, T, betas, SEED, sample_offset=3)
    _, thrX = o.get_thresholds(40)
    for t in range(T - 1):
        for m in range(40):
            p = math.exp(-4 * m * abs(betas[t + 1] - betas[t]))
            got = thrX[t, m] / 2.0 ** 32
            assert (p - got < 2.0 ** -32 + 1e-18) and (got <= p)
    key = (SEED & 0xFFFFFFFF, SEED >> 32)
    o.sweep(2)
    for n in range(30):
        E_slot, _ = o.recompute_energy()
        tos, sot = o.get_perm()
        want = sot.copy()
        for smp in range(4):
            for c in range(2):
                for t in range(T - 1):
                    ra, rb = want[smp, c, t], want[smp, c, t + 1]
                    u = int(H.philox_np(key, np.array([t, n, 3 + smp, (4 << 28) | (c << 16)], dtype=np.uint32))[0])
                    x = (betas[t] - betas[t + 1]) * float(E_slot[smp, c, ra] - E_slot[smp, c, rb])
                    p = 1.0 if x >= 0 else math.exp(x)          # Eq. (5)
                    thr = 2 ** 32 if p >= 1.0 else min(2 ** 32 - 1, math.floor(p * 2.0 ** 32))
                    if x >= 0 or u < thr:
                        want[smp, c, t], want[smp, c, t + 1] = rb, ra
        o.exchange()
        assert (o.get_perm()[1] == want).all()
        o.sweep(1)


# ------------------------------------------------------------------ P6 Houdayer, P7 overlap

@pytest.mark.parametrize("L,d", [(8, 2), (16, 2), (4, 3), (6, 3), (2, 2), (2, 3)])
def test_p6_houdayer_invariants_and_component(L, d):
    T = 4
    betas = np.array([0.3, 0.8, 1.3, 2.0])
    o = ref.Oracle(L, d, 3, T, betas, SEED)
    key = (SEED & 0xFFFFFFFF, SEED >> 32)
    N = L ** d
    for n in range(8):
        o.sweep(1)
        o.exchange()
        s0 = o.get_spins()
        E0 = o.get_energy()
        Q0, QL0 = o.measure_overlap()
        tos, sot = o.get_perm()
        o.houdayer_step()
        s1 = o.get_spins()
        assert o.recompute_energy()[1] == 0                       # (i) each energy equals its from-scratch value
        E1 = o.get_energy()
        assert (E1.sum(axis=1) == E0.sum(axis=1)).all()           # (i) E1+E2 unchanged
        Q1, QL1 = o.measure_overlap()
        assert (Q1 == Q0).all() and (QL1 == QL0).all()            # (ii)
        last, _ = o.get_cluster_sizes()
        for smp in range(3):
            for t in range(T):
                ra, rb = sot[smp, 0, t], sot[smp, 1, t]
                A, B = s0[smp, 0, ra], s0[smp, 1, rb]
                neg = (A * B) == -1
                n_neg = int(neg.sum())
                changedA = s1[smp, 0, ra] != A
                changedB = s1[smp, 1, rb] != B
                assert (changedA == changedB).all()
                if n_neg == 0:
                    assert last[smp, t] == 0 and not changedA.any()
                    continue
                u = int(H.philox_np(key, np.array([0, n, smp, (5 << 28) | t], dtype=np.uint32))[0])
                i0 = np.nonzero(neg)[0][(u * n_neg) >> 32]         # (vii) k-th negative site in index order
                comp = H.component_of(neg, i0, L, d)              # (v) library connected components
                assert (changedA == comp).all()
                assert last[smp, t] == comp.sum() <= n_neg        # (vi)
        # untouched slots: none (every slot is at some temperature); chains stay +-1
        assert set(np.unique(s1).tolist()) <= {-1, 1}


def test_p6_special_cases_and_involution():
    L, d, T = 8, 2, 3
    o = ref.Oracle(L, d, 2, T, [0.4, 0.9, 1.5], SEED)
    N = L * L
    s = o.get_spins()
    # (iv) B = -A: whole lattice is one cluster, configurations are exchanged, energies unchanged
    s2 = s.copy()
    s2[:, 1] = -s2[:, 0]
    o.set_spins(s2)
    E0 = o.get_energy()
    o.houdayer_step()
    assert (o.get_cluster_sizes()[0] == N).all()
    s3 = o.get_spins()
    assert (s3[:, 0] == s2[:, 1]).all() and (s3[:, 1] == s2[:, 0]).all()
    assert (o.get_energy() == E0).all()
    Q, QL = o.measure_overlap()
    assert (Q == -N).all() and (QL == d * N).all()               # P7
    # B = A: no negative site, size 0, no change
    s4 = s.copy()
    s4[:, 1] = s4[:, 0]
    o.set_spins(s4)
    o.houdayer_step()
    assert (o.get_cluster_sizes()[0] == 0).all() and (o.get_spins() == s4).all()
    Q, QL = o.measure_overlap()
    assert (Q == N).all() and (QL == d * N).all()
    # (iii) involution: two contexts at the same counter value; applying the step to the stepped state restores it
    a = ref.Oracle(L, d, 2, T, [0.4, 0.9, 1.5], SEED)
    b = ref.Oracle(L, d, 2, T, [0.4, 0.9, 1.5], SEED)
    a.sweep(3)
    b.sweep(3)
    before = a.get_spins()
    a.houdayer_step()
    b.set_spins(a.get_spins())
    b.houdayer_step()            # b's Houdayer counter is still 0 -> same draw u; same q=-1 set -> same cluster
    assert (b.get_spins() == before).all()


@pytest.mark.parametrize("L,d", [(4, 2), (8, 2), (4, 3), (2, 3)])
def test_p7_overlap_bruteforce_and_parity(L, d):
    T = 3
    o = ref.Oracle(L, d, 2, T, [0.2, 0.5, 0.8], SEED)
    o.mcs(5, 1, False, True)
    N = L ** d
    Q, QL = o.measure_overlap()
    s = o.get_spins()
    _, sot = o.get_perm()
    for smp in range(2):
        for t in range(T):
            q, ql = H.overlap_bruteforce(s[smp, 0, sot[smp, 0, t]], s[smp, 1, sot[smp, 1, t]], L, d)
            assert (Q[smp, t], QL[smp, t]) == (q, ql)
    assert ((Q - N) % 2 == 0).all() and ((QL - d * N) % 2 == 0).all()


# ------------------------------------------------------------------ P8 sharding / call-sequence invariance

def test_p8_sharding_invariance():
    w = wl.C1
    full = ref.Oracle(w.L, w.d, 4, w.T, w.betas(), SEED, 0)
    part = ref.Oracle(w.L, w.d, 2, w.T, w.betas(), SEED, 2)
    for o in (full, part):
        o.mcs(40, 1, True, True)
    a, b = full.state(), part.state()
    for k in a:
        if k == "counters":
            continue
        assert (a[k][2:] == b[k]).all(), k


def test_p8_mcs_equals_separate_calls():
    a = ref.Oracle(4, 3, 2, 4, wl.betas_geometric(0.4, 1.1, 4), SEED)
    b = ref.Oracle(4, 3, 2, 4, wl.betas_geometric(0.4, 1.1, 4), SEED)
    a.mcs(25, 2, True, True)
    for _ in range(25):
        b.sweep(1)
        b.sweep(1)
        b.houdayer_step()
        b.exchange()
    sa, sb = a.state(), b.state()
    for k in sa:
        assert (sa[k] == sb[k]).all(), k


# ------------------------------------------------------------------ survey worked examples W1-W3

def test_survey_worked_examples():
    with open(os.path.join(GOLD, "survey_worked_examples.json")) as f:
        G = json.load(f)
    g = G["W1"]
    b = wl.C1.betas()
    assert b[1].hex() == g["betas_hex"]["1"] and float(b[7]).hex() == g["betas_hex"]["7"]
    o = ref.Oracle(8, 2, 4, 8, b, SEED)
    J, s = o.get_couplings(), o.get_spins()
    assert J[0, 0, :16].tolist() == g["J_s0_mu0_first16"] and J[0, 1, :16].tolist() == g["J_s0_mu1_first16"]
    assert s[0, 0, 0, :16].tolist() == g["spin_s0_c0_r0_first16"]
    assert H.crc(J) == g["crc_J"] and H.crc(s) == g["crc_spins_init"]
    thrM, thrX = o.get_thresholds(32)
    # thresholds depend on libm's exp in the last unit: allow +-1
    assert np.abs(thrM.astype(np.int64) - np.array(g["thrM"])).max() <= 1
    assert np.abs(thrX[0, 1:5].astype(np.int64) - np.array(g["thrX_0_m1to4"])).max() <= 1
    assert (thrX[0, g["thrX_0_zero_from_m"]:] == 0).all() and thrX[0, g["thrX_0_zero_from_m"] - 1] > 0
    E = o.recompute_energy()[0]
    assert E[0, 0].tolist() == g["E_init_s0_c0"]
    assert E[1, 0, :3].tolist() == g["E_init_s1_c0_first3"] and E[2, 0, :3].tolist() == g["E_init_s2_c0_first3"]
    o.sweep(1)
    assert H.crc(o.get_spins()) == g["after_sweep1"]["crc_spins"]
    assert o.recompute_energy()[0][0, 0].tolist() == g["after_sweep1"]["E_s0_c0_slot"]
    o.exchange()
    sot = o.get_perm()[1]
    assert sot[0, 0].tolist() == g["after_exchange1"]["slot_of_temp_s0_c0"]
    assert sot[0, 1].tolist() == g["after_exchange1"]["slot_of_temp_s0_c1"]
    assert int(o.get_swap_counts()[1].sum()) == g["after_exchange1"]["accepts_total"]
    o.mcs(999, 1, False, True)
    f1 = g["after_1000_mcs"]
    assert H.crc(o.get_spins()) == f1["crc_spins"]
    assert o.get_energy()[0, 0].tolist() == f1["E_by_temp_s0_c0"] and o.get_energy()[0, 1].tolist() == f1["E_by_temp_s0_c1"]
    assert o.get_perm()[1][0, 0].tolist() == f1["slot_of_temp_s0_c0"]
    assert o.get_swap_counts()[1].sum(axis=(0, 1)).tolist() == f1["accepts_per_pair"]
    Q, QL = o.measure_overlap()
    assert Q[0].tolist() == f1["Q_s0"] and QL[0].tolist() == f1["QL_s0"]

    g = G["W2"]
    o = ref.Oracle(8, 2, 4, 8, b, SEED)
    o.mcs(200, 1, True, True)
    assert H.crc(o.get_spins()) == g["crc_spins"]
    assert o.get_energy()[0, 0].tolist() == g["E_by_temp_s0_c0"]
    last, cum = o.get_cluster_sizes()
    assert last[0].tolist() == g["last_cluster_sizes_s0"] and int(cum.sum()) == g["cum_cluster_size_total"]
    assert int(o.get_swap_counts()[1].sum()) == g["accepts_total"]

    g = G["W3"]
    b3 = np.array([0.4 * pow(1.1 / 0.4, t / 3.0) for t in range(4)])
    assert b3[1].hex() == g["betas_hex"]["1"] and b3[2].hex() == g["betas_hex"]["2"]
    o = ref.Oracle(4, 3, 2, 4, b3, SEED)
    assert H.crc(o.get_couplings()) == g["crc_J"] and H.crc(o.get_spins()) == g["crc_spins_init"]
    assert o.recompute_energy()[0].ravel().tolist() == g["E_init_flat"]
    assert np.abs(o.get_thresholds(2)[0][3].astype(np.int64) - np.array(g["thrM_3"])).max() <= 1
    o.mcs(100, 1, True, True)
    f3 = g["after_100_mcs_with_houdayer"]
    assert H.crc(o.get_spins()) == f3["crc_spins"]
    assert o.get_energy().ravel().tolist() == f3["E_by_temp_flat"]
    Q, QL = o.measure_overlap()
    assert Q.ravel().tolist() == f3["Q_flat"] and QL.ravel().tolist() == f3["QL_flat"]
    last, cum = o.get_cluster_sizes()
    assert last.ravel().tolist() == f3["last_cluster_sizes_flat"] and int(cum.sum()) == f3["cum_cluster_size_total"]
    assert o.get_swap_counts()[1].sum(axis=(0, 1)).tolist() == f3["accepts_per_pair"]
