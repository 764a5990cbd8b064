"""Pins of the oracle's NEXT-2 part ("spin-glass susceptibility and the modes for the
correlation length"; reading R31): the overlap profile prof[mu][x] = sum of q_i over the plane x_mu = x, from which
chi_SG = <Q^2>/N and the axis Fourier modes q(k e_mu) follow."""
import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H


@pytest.mark.parametrize("L,d", [(4, 2), (6, 2), (8, 2), (4, 3), (6, 3)])
def test_profile_brute_force_sums_and_special_cases(L, d):
    S, T = 2, 3
    o = ref.Oracle(L, d, S, T, wl.betas_linear(0.2, 1.0, T), wl.SEED)
    o.mcs(7, 1, True, True)
    prof = o.measure_overlap_profile()
    Q, _ = o.measure_overlap()
    sp = o.get_spins(); _, sot = o.get_perm()
    for s in range(S):
        for t in range(T):
            q = (sp[s, 0, sot[s, 0, t]].astype(np.int64) * sp[s, 1, sot[s, 1, t]]).reshape(H.lattice_shape(L, d))
            for mu in range(d):
                axes = tuple(a for a in range(d) if a != H.axis_of(mu, d))
                assert np.array_equal(prof[s, t, mu], q.sum(axis=axes))          # numpy plane sums
                assert prof[s, t, mu].sum() == Q[s, t]                             # every axis sums to Q
    assert ((prof - L ** (d - 1)) % 2 == 0).all() and (abs(prof) <= L ** (d - 1)).all()
    # identical chains: q = +1 everywhere; negated chain: q = -1 everywhere (fresh state: identity permutations)
    o = ref.Oracle(L, d, S, T, wl.betas_linear(0.2, 1.0, T), wl.SEED)
    s0 = o.get_spins()
    s1 = s0.copy(); s1[:, 1] = s1[:, 0]
    o.set_spins(s1)
    assert (o.measure_overlap_profile() == L ** (d - 1)).all()
    s1[:, 1] = -s1[:, 0]
    o.set_spins(s1)
    assert (o.measure_overlap_profile() == -(L ** (d - 1))).all()


def test_profile_of_a_plane_wave_pattern_and_its_fourier_mode():
    """A = +1 everywhere, B = +1 on the half x < L/2 and -1 on the other half (temperature order = slot order at
    init): prof[x-axis] = +-L^(d-1) by half, the other axes see exactly zero; the k_min mode along x is the known
    square-wave coefficient and along y it vanishes."""
    L, d, S, T = 8, 3, 1, 2
    o = ref.Oracle(L, d, S, T, np.array([0.5, 0.6]), wl.SEED)
    x = np.arange(L ** d) % L
    A = np.ones((S, 2, T, L ** d), dtype=np.int8)
    A[:, 1] = np.where(x < L // 2, 1, -1).astype(np.int8)
    o.set_spins(A)
    prof = o.measure_overlap_profile()[0, 0]
    assert prof[0].tolist() == [L * L] * (L // 2) + [-L * L] * (L // 2)
    assert (prof[1] == 0).all() and (prof[2] == 0).all()
    k = 2 * np.pi / L
    qk = (prof * np.exp(1j * k * np.arange(L))[None, :]).sum(axis=1)
    exact = L * L * 2 / (1 - np.exp(1j * k))             # sum_{x<L/2} e^{ikx} - sum_{x>=L/2} e^{ikx} = 2 (1 - e^{ikL/2}) / (1 - e^{ik}) ... = 4 / (1 - e^{ik})
    assert abs(qk[0] - 2 * exact) < 1e-9 and abs(qk[1]) < 1e-9 and abs(qk[2]) < 1e-9
