"""Pins of the oracle's NEXT-3 part (readings R33-R35): couplings as fixed-point
numbers J = Jq * 2^-fbits (a rounded standard-normal sample is an INPUT), integer fields and energies, acceptance
probabilities from double exp.  Pinned by (a) the reduction to the +-J model, which P1-P9 pin, bit for bit; (b) exact
enumeration of the canonical averages for Gaussian couplings at 2D L = 4; (c) invariants."""
import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H


@pytest.mark.parametrize("L,d,fbits", [(8, 2, 0), (8, 2, 16), (4, 3, 9), (6, 2, 20)])
def test_pm_one_couplings_in_fixed_point_reproduce_the_pmJ_run_bit_for_bit(L, d, fbits):
    """Jq = J * 2^fbits with J = +-1: fields, energies and energy differences are the +-J ones times 2^fbits, and
    ldexp(2a * 2^fbits, -fbits) = 2a exactly, so every threshold equals the +-J table entry: same trajectory."""
    S, T = 2, 5
    betas = wl.betas_geometric(0.3, 1.8, T)
    a = ref.Oracle(L, d, S, T, betas, wl.SEED, 4)
    b = ref.Oracle(L, d, S, T, betas, wl.SEED, 4)
    b.set_couplings_fixed(a.get_couplings().astype(np.int32) << fbits, fbits)
    assert np.array_equal(b.get_energy(), a.get_energy().astype(np.int64) << fbits)
    for _ in range(25):
        a.mcs(1, 2, True, True); b.mcs(1, 2, True, True)
    sa, sb = a.state(), b.state()
    for k in sa:
        if k == "energy":
            assert np.array_equal(sb[k], sa[k].astype(np.int64) << fbits)
        else:
            assert np.array_equal(sa[k], sb[k]), k
    assert b.recompute_energy()[1] == 0


def _run(o, n_mcs, houdayer, burn=2000):
    o.mcs(burn, 1, houdayer, True)
    Es = np.zeros((n_mcs, o.S, 2, o.T)); Qs = np.zeros((n_mcs, o.S, o.T))
    for n in range(n_mcs):
        o.mcs(1, 1, houdayer, True)
        Es[n] = o.get_energy(); Qs[n] = o.measure_overlap()[0]
    return Es, Qs


@pytest.mark.parametrize("houdayer", [False, True])
def test_gaussian_couplings_sample_the_canonical_ensemble_2d_L4(houdayer):
    """Exact enumeration (2^16 states) of <E> and <q^2> with the SAME fixed-point couplings as real numbers."""
    L, d, S, fbits = 4, 2, 2, 12
    betas = wl.betas_linear(0.2, 1.6, 6)
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, d, L ** d, fbits)
    o = ref.Oracle(L, d, S, len(betas), betas, wl.SEED)
    o.set_couplings_fixed(Jq, fbits)
    Es, Qs = _run(o, 40000, houdayer)
    scale = float(1 << fbits)
    zs = []
    for s in range(S):
        E_exact, q2_exact, _ = H.enumerate_any(Jq[s] / scale, betas, L, d)
        for t in range(len(betas)):
            m, e = H.binned_mean_err(Es[:, s, :, t].mean(axis=1) / scale)
            zs.append((m - E_exact[t]) / e)
            m, e = H.binned_mean_err((Qs[:, s, t] / L ** d) ** 2)
            zs.append((m - q2_exact[t]) / e)
    zs = np.array(zs)
    assert np.abs(zs).max() < 4.5, zs
    assert np.sqrt((zs ** 2).mean()) < 1.8, zs


def test_gaussian_invariants_and_argument_checks():
    L, d, S, T, fbits = 6, 3, 2, 4, 16
    betas = wl.betas_geometric(0.4, 1.1, T)
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, d, L ** d, fbits)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED)
    o.set_couplings_fixed(Jq, fbits)
    j2, f2 = o.get_couplings_fixed()
    assert np.array_equal(j2, Jq) and f2 == fbits
    sp = o.get_spins()
    for s in range(S):                                    # energy against a numpy restatement with real couplings
        e = H.energy_bruteforce(Jq[s].astype(np.float64), sp[s, 0, 1].astype(np.float64), L, d)
        assert o.recompute_energy()[0][s, 0, 1] == e
    for _ in range(10):
        E0 = o.get_energy().astype(np.int64)
        Q0, QL0 = o.measure_overlap()
        o.houdayer_step()
        assert np.array_equal(E0.sum(axis=1), o.get_energy().astype(np.int64).sum(axis=1))   # E1 + E2 conserved
        Q1, QL1 = o.measure_overlap()
        assert np.array_equal(Q0, Q1) and np.array_equal(QL0, QL1)
        o.sweep(1); o.exchange()
        assert o.recompute_energy()[1] == 0
    with pytest.raises(RuntimeError):
        o.set_couplings_fixed(np.full((S, d, L ** d), 2 ** 24, dtype=np.int32), 16)        # would overflow int32 energies
    with pytest.raises(RuntimeError):
        o.set_couplings_fixed(Jq, 30)
    # beta = 0 flips everything whatever the couplings; thresholds are monotone in a
    z = ref.Oracle(4, 2, 1, 2, np.array([0.0, 0.0]), wl.SEED)
    z.set_couplings_fixed(wl.gaussian_couplings_fixed(1, 1, 2, 16, 10), 10)
    s0 = z.get_spins(); z.sweep(1)
    assert np.array_equal(z.get_spins(), -s0)
