"""Pin P5: the whole chain (checkerboard Metropolis + Houdayer + PT, readings R1, R4, R9, R13) samples the
canonical ensemble.  Brute force: exact enumeration of <E> and <q^2> for 2D L=4 (2^16 states per sample) and of
<E> for 3D L=2 (2^8 states, double bonds, R3), against time averages of the oracle.  This replaces the paper's
own check against an exact Pfaffian calculation (Fig. 8), which is not reproducible here."""
import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H


def _run(L, d, S, betas, n_mcs, houdayer, burn=2000):
    T = len(betas)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED)
    o.mcs(burn, 1, houdayer, True)
    Es = np.zeros((n_mcs, S, 2, T))
    Qs = np.zeros((n_mcs, S, T))
    for n in range(n_mcs):
        o.mcs(1, 1, houdayer, True)
        Es[n] = o.get_energy()
        Qs[n] = o.measure_overlap()[0]
    return o, Es, Qs


@pytest.mark.parametrize("houdayer", [False, True])
def test_p5_exact_enumeration_2d_L4(houdayer):
    L, d, S = 4, 2, 2
    betas = wl.betas_linear(0.2, 1.5, 6)
    o, Es, Qs = _run(L, d, S, betas, 40000, houdayer)
    J = o.get_couplings()
    N = L ** d
    zs = []
    for s in range(S):
        E_exact, q2_exact, _ = H.enumerate_2d_L4(J[s], betas)
        for t in range(len(betas)):
            m, e = H.binned_mean_err(Es[:, s, :, t].mean(axis=1))
            zs.append((m - E_exact[t]) / e)
            m, e = H.binned_mean_err((Qs[:, s, t] / N) ** 2)
            zs.append((m - q2_exact[t]) / e)
    zs = np.array(zs)
    assert np.abs(zs).max() < 4.5, zs
    assert np.sqrt((zs ** 2).mean()) < 1.8, zs       # 24 values: an rms well above 1 would mean a biased sampler


def test_p5_energy_histogram_2d_L4():
    """Stronger form: the sampled energy histogram against g(E) exp(-beta E) / Z at one temperature."""
    L, d, S = 4, 2, 1
    betas = wl.betas_linear(0.3, 1.2, 4)
    o, Es, _ = _run(L, d, S, betas, 30000, True)
    J = o.get_couplings()
    _, _, Eall = H.enumerate_2d_L4(J[0], betas)
    levels, g = np.unique(Eall, return_counts=True)
    for t in (0, 2):
        w = g * np.exp(-betas[t] * (levels - levels.min()))
        w /= w.sum()
        x = Es[:, 0, :, t].ravel()
        # thin by 10 MCS to tame autocorrelation, then compare frequencies of the populated levels
        x = x.reshape(-1, 2)[::10].ravel()
        obs = np.array([(x == lv).sum() for lv in levels], dtype=np.float64)
        exp_ = w * len(x)
        keep = exp_ > 20
        chi2 = ((obs[keep] - exp_[keep]) ** 2 / exp_[keep]).sum()
        assert chi2 < 3.0 * keep.sum(), (t, chi2, keep.sum())
        assert set(np.unique(x).tolist()) <= set(levels.tolist())


def test_p5_exact_energy_3d_L2():
    L, d, S = 2, 3, 3
    betas = wl.betas_linear(0.2, 1.0, 4)
    o, Es, _ = _run(L, d, S, betas, 30000, False)
    J = o.get_couplings()
    zs = []
    for s in range(S):
        E_exact, _, _ = H.enumerate_any(J[s], betas, L, d)
        for t in range(len(betas)):
            m, e = H.binned_mean_err(Es[:, s, :, t].mean(axis=1))
            zs.append((m - E_exact[t]) / max(e, 1e-12))
    assert np.abs(np.array(zs)).max() < 4.5, zs
