"""Pins P16-P17 of the oracle's cluster-move variants (readings R36, R37).

R36  ref_set_cluster_moves: n_clu[t] single-cluster moves per Houdayer call at temperature index t.
R37  ref_houdayer_multi: every q = -1 component is exchanged with probability 1/2.
Pinned by: reduction to the default move, a test-side reconstruction of every move from scipy's connected components
and an independent numpy Philox, conservation laws, and exact enumeration at 2D L = 4."""
import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H

SEED = wl.SEED
KEY = (SEED & 0xFFFFFFFF, SEED >> 32)


def _labels(neg, L, d):
    """Component label of every site (library routine), -1 outside negmask."""
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components

    N = L ** d
    nbr = H.neighbour_list(L, d)
    rows, cols = [], []
    for k in range(2 * d):
        ok = neg & neg[nbr[:, k]]
        rows.append(np.nonzero(ok)[0])
        cols.append(nbr[ok, k])
    rows, cols = np.concatenate(rows), np.concatenate(cols)
    g = coo_matrix((np.ones(len(rows), dtype=np.int8), (rows, cols)), shape=(N, N))
    _, lab = connected_components(g, directed=False)
    return np.where(neg, lab, -1)


# ------------------------------------------------------------------ P16: per-temperature move counts (R36)

def test_p16_all_ones_is_the_default_move_bit_for_bit():
    b = wl.betas_linear(0.2, 2.0, 6)
    a = ref.Oracle(8, 2, 3, 6, b, SEED)
    c = ref.Oracle(8, 2, 3, 6, b, SEED)
    c.set_cluster_moves(np.ones(6, dtype=np.int32))
    a.mcs(25, 1, 1, True)
    c.mcs(25, 1, 1, True)
    sa, sc = a.state(), c.state()
    for k in sa:
        assert np.array_equal(sa[k], sc[k]), k
    c.set_cluster_moves(None)
    a.mcs(5, 1, 1, True)
    c.mcs(5, 1, 1, True)
    assert np.array_equal(a.get_spins(), c.get_spins())


def test_p16_rejects_bad_counts():
    o = ref.Oracle(4, 2, 1, 3, [0.5, 0.7, 0.9], SEED)
    with pytest.raises(RuntimeError):
        o.set_cluster_moves(np.array([1, -1, 1], dtype=np.int32))
    with pytest.raises(RuntimeError):
        o.set_cluster_moves(np.array([1, 65536, 1], dtype=np.int32))


@pytest.mark.parametrize("L,d", [(8, 2), (16, 2), (4, 3), (6, 3), (2, 2)])
def test_p16_every_move_reconstructed_from_library_components(L, d):
    T, S = 4, 3
    betas = np.array([0.3, 0.8, 1.3, 2.0])
    n_clu = np.array([3, 0, 2, 1], dtype=np.int32)
    o = ref.Oracle(L, d, S, T, betas, SEED)
    o.set_cluster_moves(n_clu)
    for n in range(6):
        o.sweep(1)
        o.exchange()
        s0 = o.get_spins()
        E0 = o.get_energy()
        Q0, QL0 = o.measure_overlap()
        _, cum0 = o.get_cluster_sizes()
        _, sot = o.get_perm()
        o.houdayer_step()
        s1 = o.get_spins()
        assert o.recompute_energy()[1] == 0
        assert (o.get_energy().sum(axis=1) == E0.sum(axis=1)).all()       # E1 + E2 unchanged
        Q1, QL1 = o.measure_overlap()
        assert (Q1 == Q0).all() and (QL1 == QL0).all()
        last, cum = o.get_cluster_sizes()
        for smp in range(S):
            for t in range(T):
                ra, rb = sot[smp, 0, t], sot[smp, 1, t]
                A, B = s0[smp, 0, ra].copy(), s0[smp, 1, rb].copy()
                sizes = []
                for j in range(n_clu[t]):
                    neg = (A * B) == -1
                    n_neg = int(neg.sum())
                    if n_neg == 0:
                        sizes.append(0)
                        continue
                    u = int(H.philox_np(KEY, np.array([j, n, smp, (5 << 28) | t], dtype=np.uint32))[0])
                    i0 = np.nonzero(neg)[0][(u * n_neg) >> 32]
                    comp = H.component_of(neg, i0, L, d)
                    A[comp] = -A[comp]
                    B[comp] = -B[comp]
                    sizes.append(int(comp.sum()))
                assert np.array_equal(s1[smp, 0, ra], A) and np.array_equal(s1[smp, 1, rb], B), (smp, t)
                assert last[smp, t] == (sizes[-1] if sizes else 0)
                assert cum[smp, t] - cum0[smp, t] == sum(sizes)


def test_p16_zero_moves_leave_the_temperature_alone():
    L, d, S, T = 8, 2, 2, 3
    o = ref.Oracle(L, d, S, T, [0.4, 0.9, 1.5], SEED)
    o.set_cluster_moves(np.array([0, 0, 0], dtype=np.int32))
    o.sweep(2)
    before = o.state()
    o.houdayer_step()
    after = o.state()
    assert np.array_equal(before["spins"], after["spins"]) and np.array_equal(before["energy"], after["energy"])
    assert (after["last_size"] == 0).all() and np.array_equal(before["cum_size"], after["cum_size"])
    assert after["counters"][2] == before["counters"][2] + 1          # the step is still counted


# ------------------------------------------------------------------ P17: multi-cluster variant (R37)

@pytest.mark.parametrize("L,d", [(8, 2), (16, 2), (4, 3), (6, 3), (2, 2), (2, 3)])
def test_p17_multi_cluster_reconstructed_from_library_components(L, d):
    T, S = 4, 3
    betas = np.array([0.3, 0.8, 1.3, 2.0])
    o = ref.Oracle(L, d, S, T, betas, SEED)
    n_flipped_clusters = n_kept_clusters = 0
    for n in range(6):
        o.sweep(1)
        o.exchange()
        s0 = o.get_spins()
        E0 = o.get_energy()
        Q0, QL0 = o.measure_overlap()
        _, cum0 = o.get_cluster_sizes()
        _, sot = o.get_perm()
        o.houdayer_multi_step()
        s1 = o.get_spins()
        assert o.recompute_energy()[1] == 0
        assert (o.get_energy().sum(axis=1) == E0.sum(axis=1)).all()       # E1 + E2 unchanged
        Q1, QL1 = o.measure_overlap()
        assert (Q1 == Q0).all() and (QL1 == QL0).all()
        last, cum = o.get_cluster_sizes()
        for smp in range(S):
            for t in range(T):
                ra, rb = sot[smp, 0, t], sot[smp, 1, t]
                A, B = s0[smp, 0, ra], s0[smp, 1, rb]
                neg = (A * B) == -1
                lab = _labels(neg, L, d)
                flip = np.zeros(L ** d, dtype=bool)
                for lb in np.unique(lab[lab >= 0]):
                    members = np.nonzero(lab == lb)[0]
                    i_min = int(members.min())
                    w = H.philox_np(KEY, np.array([i_min >> 2, n, smp, (5 << 28) | (1 << 24) | t], dtype=np.uint32))
                    if int(w[i_min & 3]) >> 31:
                        flip[members] = True
                        n_flipped_clusters += 1
                    else:
                        n_kept_clusters += 1
                assert np.array_equal(s1[smp, 0, ra], np.where(flip, -A, A)), (smp, t)
                assert np.array_equal(s1[smp, 1, rb], np.where(flip, -B, B)), (smp, t)
                assert last[smp, t] == flip.sum()
                assert cum[smp, t] - cum0[smp, t] == flip.sum()
    tot = n_flipped_clusters + n_kept_clusters
    if tot > 400:                                                        # fair coin, 5 sigma
        assert abs(n_flipped_clusters - tot / 2) < 2.5 * np.sqrt(tot)


def test_p17_special_cases():
    L, d, T = 8, 2, 3
    N = L * L
    o = ref.Oracle(L, d, 4, T, [0.4, 0.9, 1.5], SEED)
    s = o.get_spins()
    # B = -A: one component, root site 0 -> exchanged as a whole or not at all, by the bit of site 0
    s2 = s.copy()
    s2[:, 1] = -s2[:, 0]
    o.set_spins(s2)
    E0 = o.get_energy()
    o.houdayer_multi_step()
    last, _ = o.get_cluster_sizes()
    s3 = o.get_spins()
    for smp in range(4):
        for t in range(T):
            w = H.philox_np(KEY, np.array([0, 0, smp, (5 << 28) | (1 << 24) | t], dtype=np.uint32))
            if int(w[0]) >> 31:
                assert last[smp, t] == N and np.array_equal(s3[smp, 0, t], s2[smp, 1, t])
            else:
                assert last[smp, t] == 0 and np.array_equal(s3[smp, 0, t], s2[smp, 0, t])
    assert (o.get_energy() == E0).all()
    assert set(np.unique(last).tolist()) == {0, N}                      # 12 fair coins: both outcomes occur
    # B = A: nothing to exchange
    s4 = s.copy()
    s4[:, 1] = s4[:, 0]
    o.set_spins(s4)
    o.houdayer_multi_step()
    assert (o.get_cluster_sizes()[0] == 0).all() and (o.get_spins() == s4).all()


def test_p17_mcs_mode_2_equals_separate_calls():
    b = wl.betas_linear(0.2, 2.0, 5)
    a = ref.Oracle(8, 2, 2, 5, b, SEED)
    c = ref.Oracle(8, 2, 2, 5, b, SEED)
    a.mcs(7, 2, 2, True)
    for _ in range(7):
        c.sweep(2)
        c.houdayer_multi_step()
        c.exchange()
    sa, sc = a.state(), c.state()
    for k in sa:
        assert np.array_equal(sa[k], sc[k]), k


@pytest.mark.parametrize("mode", ["multi", "counts"])
def test_p17_exact_enumeration_2d_L4(mode):
    """Both variants keep the canonical ensemble: time averages against exact enumeration (as pin P5)."""
    L, d, S = 4, 2, 2
    betas = wl.betas_linear(0.2, 1.5, 6)
    T = len(betas)
    o = ref.Oracle(L, d, S, T, betas, SEED)
    if mode == "counts":
        o.set_cluster_moves(np.array([3, 2, 2, 1, 0, 1], dtype=np.int32))
    hd = 2 if mode == "multi" else 1
    n_mcs = 30000
    o.mcs(2000, 1, hd, True)
    Es = np.zeros((n_mcs, S, 2, T))
    Qs = np.zeros((n_mcs, S, T))
    for n in range(n_mcs):
        o.mcs(1, 1, hd, True)
        Es[n] = o.get_energy()
        Qs[n] = o.measure_overlap()[0]
    J = o.get_couplings()
    N = L ** d
    zs = []
    for s in range(S):
        E_exact, q2_exact, _ = H.enumerate_2d_L4(J[s], betas)
        for t in range(T):
            m, e = H.binned_mean_err(Es[:, s, :, t].mean(axis=1))
            zs.append((m - E_exact[t]) / e)
            m, e = H.binned_mean_err((Qs[:, s, t] / N) ** 2)
            zs.append((m - q2_exact[t]) / e)
    zs = np.array(zs)
    assert np.abs(zs).max() < 4.5, zs
    assert np.sqrt((zs ** 2).mean()) < 1.8, zs
