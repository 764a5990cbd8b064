"""GPU parity of the NEXT-3 row: fixed-point (Gaussian) couplings with double-exp acceptance, through the
C ABI, bit for bit against the oracle: spins, energies, permutations, swap counts, cluster sizes, overlaps.
Run with `-m gpu`."""
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


def same_state(o, tag):
    a, b = o.state(), B.state()
    for k in a:
        assert np.array_equal(a[k], b[k]), "%s: %s differs" % (tag, k)
    Qo, QLo = o.measure_overlap(); Qg, QLg = B.pt_measure_overlap()
    assert np.array_equal(Qo, Qg) and np.array_equal(QLo, QLg), tag
    assert B.pt_recompute_energy()[1] == 0, tag


@pytest.mark.parametrize("L,d,S,T,fbits,general", [
    (8, 2, 3, 5, 16, False), (32, 2, 2, 6, 16, False), (64, 2, 1, 3, 12, False), (8, 3, 2, 4, 16, False), (16, 3, 1, 3, 14, False),
    (4, 2, 2, 3, 16, False), (6, 3, 2, 3, 10, False), (10, 2, 1, 4, 16, False), (16, 2, 2, 4, 16, True),
    (8, 2, 3, 5, 21, False),            # 2 d max|Jq| >= 2^23: the kernels with the per-site range test
    (32, 2, 1, 40, 16, False)])         # two 32-temperature groups in the fused kernel's cluster phase
def test_gaussian_couplings_match_oracle(L, d, S, T, fbits, general):
    betas = wl.betas_geometric(0.2, 1.4, T)
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, d, L ** d, fbits, sample_offset=2)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 2)
    o.set_couplings_fixed(Jq, fbits)
    B.pt_open(L, d, S, T, betas, wl.SEED, 2, general=general, fixed_couplings=True)
    B.pt_set_couplings_fixed(Jq, fbits)
    j2, f2 = B.pt_get_couplings_fixed()
    assert np.array_equal(j2, Jq) and f2 == fbits
    same_state(o, "after set")
    for step in range(5):
        o.sweep(1); B.pt_sweep(1)
        same_state(o, "sweep %d" % step)
        o.houdayer_step(); B.houdayer_step()
        same_state(o, "houdayer %d" % step)
        o.exchange(); B.pt_exchange()
        same_state(o, "exchange %d" % step)
    o.sweep(3); B.pt_sweep(3)
    same_state(o, "sweep(3)")
    o.mcs(20, 2, True, True); B.pt_mcs(20, 2, True, True)      # ONE fused launch on the word-parallel lattices
    same_state(o, "mcs")
    assert B.pt_get_fused() == int(B.pt_get_path() == 1)
    B.pt_set_fused(0)
    o.mcs(4, 1, True, True); B.pt_mcs(4, 1, True, True)        # the separate kernels
    same_state(o, "mcs, separate kernels")
    B.pt_set_fused(-1)
    o.mcs(3, 1, False, True); B.pt_mcs(3, 1, False, True)      # no cluster move: no energy recompute in the fused kernel
    same_state(o, "mcs without the cluster move")


def test_pm_one_in_fixed_point_equals_the_pmJ_path_on_the_device():
    L, d, S, T, fbits = 32, 2, 2, 5, 16
    betas = wl.betas_geometric(0.3, 1.8, T)
    B.pt_open(L, d, S, T, betas, wl.SEED, fixed_couplings=True)
    J = B.pt_get_couplings()
    B.pt_mcs(15, 1, True, True)
    ref_state = B.state()
    B.pt_open(L, d, S, T, betas, wl.SEED, fixed_couplings=True)
    B.pt_set_couplings_fixed(J.astype(np.int32) << fbits, fbits)
    B.pt_mcs(15, 1, True, True)
    st = B.state()
    for k in st:
        if k == "energy":
            assert np.array_equal(st[k], ref_state[k].astype(np.int64) << fbits)
        else:
            assert np.array_equal(st[k], ref_state[k]), k


def test_errors_and_return_to_pmJ():
    L, d, S, T = 8, 2, 1, 2
    B.pt_open(L, d, S, T, wl.betas_linear(0.2, 1.0, T), wl.SEED, fixed_couplings=True)
    with pytest.raises(B.PTError) as e:
        B.pt_get_couplings_fixed()
    assert e.value.code == B.PT_ERR_STATE
    with pytest.raises(B.PTError) as e:
        B.pt_set_couplings_fixed(np.full((S, d, L * L), 2 ** 25, dtype=np.int32), 16)
    assert e.value.code == B.PT_ERR_ARG
    with pytest.raises(B.PTError) as e:
        B.pt_set_couplings_fixed(np.ones((S, d, L * L), dtype=np.int32), 25)
    assert e.value.code == B.PT_ERR_ARG
    J = B.pt_get_couplings()
    B.pt_set_couplings_fixed(wl.gaussian_couplings_fixed(1, S, d, L * L, 16), 16)
    with pytest.raises(B.PTError) as e:
        B.pt_get_couplings()
    assert e.value.code == B.PT_ERR_STATE
    B.pt_set_couplings(J)                                   # back to +-J
    assert np.array_equal(B.pt_get_couplings(), J) and B.pt_recompute_energy()[1] == 0


def test_device_exp_thresholds_against_the_host_libm():
    """Reading R34 rests on two double `exp` implementations (CUDA libdevice on the device, the C library in the oracle)
    giving the same floor(2^32 exp(x)): both are within 1 ulp, so a differing floor needs exp(x) within ~2^-53 relative of
    a multiple of 2^-32.  Counted here on 4 x 10^5 arguments of the form the path produces, -(beta * a * 2^-f): the floors
    may differ by at most 1 unit, on at most a handful of arguments (0 observed)."""
    B.pt_open(32, 2, 64, 8, wl.betas_linear(0.2, 1.0, 8), wl.SEED, fixed_couplings=True)
    rng = np.random.default_rng(5)
    betas = wl.betas_geometric(0.2, 3.0, 32)
    a = rng.integers(1, 2 ** 21, size=400000)
    x = -(betas[rng.integers(0, 32, size=a.size)] * np.ldexp(a.astype(np.float64) * 2.0, -16))
    dev = B.pt_threshold_selftest(x).astype(np.int64)
    host = np.array([ref.threshold(float(v)) for v in x[:20000]], dtype=np.int64)
    # the oracle's routine on a subset, numpy's exp (also a correctly-rounded-or-1-ulp libm path) on everything
    hostnp = np.minimum(np.floor(np.ldexp(np.exp(x), 32)), 4294967295.0).astype(np.int64)
    assert np.abs(dev[:20000] - host).max() <= 1 and np.abs(dev - hostnp).max() <= 1
    n_diff = int((dev[:20000] != host).sum())
    print("device vs host THR: %d of 20000 floors differ (oracle libm), %d of %d (numpy)" % (n_diff, int((dev != hostnp).sum()), x.size))
    assert n_diff <= 2 and (dev != hostnp).sum() <= 40
    with pytest.raises(B.PTError) as e:             # a workspace without the int32 coupling arrays
        B.pt_open(8, 2, 2, 4, wl.betas_linear(0.2, 1.0, 4), wl.SEED)
        B.pt_set_couplings_fixed(np.ones((2, 2, 64), dtype=np.int32), 4)
    assert e.value.code == B.PT_ERR_STATE


def test_gaussian_C2_shape_sampled_samples():
    """C2's lattice, ladder and chain count with Gaussian couplings on 64 samples; samples 0 and 63 against the oracle."""
    w, S, fbits, n = wl.C2, 64, 16, 30
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, w.d, w.N, fbits)
    B.pt_open(w.L, w.d, S, w.T, w.betas(), wl.SEED, fixed_couplings=True)
    B.pt_set_couplings_fixed(Jq, fbits)
    B.pt_mcs(n, 1, True, True)
    st = B.state()
    assert B.pt_recompute_energy()[1] == 0
    for g in (0, S - 1):
        o = ref.Oracle(w.L, w.d, 1, w.T, w.betas(), wl.SEED, g)
        o.set_couplings_fixed(Jq[g:g + 1], fbits)
        o.mcs(n, 1, True, True)
        a = o.state()
        for k in a:
            if k != "counters":
                assert np.array_equal(a[k][0], st[k][g]), (g, k)


def test_gaussian_C2_full_size_all_samples_and_a_thousand_mcs():
    """The Gaussian (fixed-point) path at C2's FULL size in bench.py's launch configuration (`bench.py --gaussian`: one fused
    launch per step): (i) all 1024 samples for their first 16 MCS, full state, against oracle processes on all host cores;
    (ii) samples {0, 1, S/2, S-1} for 1000 MCS, compared at 10, 100 and 1000 -- about 4 x 10^7 double-exp decisions per
    sample, the ground reading R34's agreement argument stands on."""
    from oracle import pool as OP

    w, fbits = wl.C2, 16
    Jq = wl.gaussian_couplings_fixed(wl.SEED, w.S, w.d, w.N, fbits)
    gs = [0, 1, w.S // 2, w.S - 1]
    pool = OP.OraclePool()
    try:
        long_jobs = {g: pool.submit(w, g, 1, 1000, checkpoints=(10, 100, 1000), gaussian_fbits=fbits) for g in gs}
        futs = pool.submit_all_samples(w, 16, gaussian_fbits=fbits)
        B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, fixed_couplings=True)
        B.pt_set_couplings_fixed(Jq, fbits)
        assert B.pt_get_fused() == 1
        got, done = {}, 0
        for stop in (10, 16, 100, 1000):
            while done < stop:
                n = min(50, stop - done)
                B.pt_mcs(n, 1, True, True)
                done += n
            st = B.state()
            st["Q"], st["QL"] = B.pt_measure_overlap()
            got[stop] = st if stop == 16 else {k: st[k][gs].copy() for k in OP.STATE_KEYS + ("Q", "QL")}
        assert B.pt_recompute_energy()[1] == 0
        want, _ = OP.gather(futs, 16)
        for k in OP.STATE_KEYS + ("Q", "QL"):
            assert np.array_equal(want[k], got[16][k]), "all samples after 16 MCS: %s differs" % k
        for i, g in enumerate(gs):
            _, _, states, _ = long_jobs[g].result()
            for c in (10, 100, 1000):
                for k in OP.STATE_KEYS + ("Q", "QL"):
                    assert np.array_equal(states[c][k][0], got[c][k][i]), "sample %d after %d MCS: %s differs" % (g, c, k)
    finally:
        pool.close()


@pytest.mark.parametrize("L,d,S,T,general", [(32, 2, 2, 6, False), (8, 3, 2, 5, False), (64, 2, 1, 3, False), (6, 2, 2, 4, True)])
def test_gaussian_with_cluster_variants_and_records(L, d, S, T, general):
    """Fixed-point couplings together with the NEXT-4 variants (move counts in the fused kernel, multi-cluster step) and
    with pt_mcs_measure_device (which issues the separate calls in this model)."""
    import torch

    betas = wl.betas_geometric(0.2, 1.4, T)
    fbits = 12 if L >= 64 else 16                      # d N max|Jq| must stay below 2^31
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, d, L ** d, fbits, sample_offset=4)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 4)
    o.set_couplings_fixed(Jq, fbits)
    B.pt_open(L, d, S, T, betas, wl.SEED, 4, general=general, fixed_couplings=True)
    B.pt_set_couplings_fixed(Jq, fbits)
    n_clu = np.array([(3 * t) % 4 for t in range(T)], dtype=np.int32)
    o.set_cluster_moves(n_clu); B.pt_set_cluster_moves(n_clu)
    o.mcs(6, 1, 1, True); B.pt_mcs(6, 1, 1, True)
    same_state(o, "move counts")
    o.set_cluster_moves(None); B.pt_set_cluster_moves(None)
    o.houdayer_multi_step(); B.houdayer_multi_step()
    same_state(o, "multi-cluster step")
    o.mcs(4, 1, 2, True); B.pt_mcs(4, 1, 2, True)
    same_state(o, "mcs with the multi-cluster step")
    Qr = torch.empty((2, S, T), dtype=torch.int32, device="cuda")
    QLr = torch.empty_like(Qr)
    B.pt_mcs_measure_device(7, 1, 1, True, 3, Qr, QLr)
    for r in range(2):
        o.mcs(3, 1, 1, True)
        Qo, QLo = o.measure_overlap()
        assert np.array_equal(Qo, Qr.cpu().numpy()[r]) and np.array_equal(QLo, QLr.cpu().numpy()[r])
    o.mcs(1, 1, 1, True)
    same_state(o, "records")


def test_int32_couplings_are_laid_out_by_flag_never_by_spare_bytes():
    """pt_init lays the int32 coupling arrays out iff pt_set_workspace_flags(PT_WS_FIXED_COUPLINGS) asked for them: a
    workspace with room to spare does not get them unasked, and a workspace too small for what was asked is refused."""
    import torch
    L, d, S, T = 8, 2, 2, 4
    betas = wl.betas_linear(0.2, 1.0, T)
    Jq = wl.gaussian_couplings_fixed(wl.SEED, S, d, L * L, 16)
    big = torch.empty(B.pt_workspace_bytes_ex(L, d, S, T, B.PT_WS_FIXED_COUPLINGS), dtype=torch.uint8, device="cuda:0")
    B.pt_bind(big)
    B.pt_init(L, d, S, T, betas, wl.SEED)                      # room for the arrays, but nobody asked
    assert B.pt_get_stage_bytes() > 0
    with pytest.raises(B.PTError) as e:
        B.pt_set_couplings_fixed(Jq, 16)
    assert e.value.code == B.PT_ERR_STATE and "pt_set_workspace_flags" in str(e.value)
    B.pt_bind(big)                                             # re-binding resets the flags
    B.pt_set_workspace_flags(B.PT_WS_FIXED_COUPLINGS)
    B.pt_init(L, d, S, T, betas, wl.SEED)
    B.pt_set_couplings_fixed(Jq, 16)
    assert np.array_equal(B.pt_get_couplings_fixed()[0], Jq)
    small = torch.empty(B.pt_workspace_bytes(L, d, S, T), dtype=torch.uint8, device="cuda:0")
    B.pt_bind(small)
    B.pt_set_workspace_flags(B.PT_WS_FIXED_COUPLINGS)
    with pytest.raises(B.PTError) as e:
        B.pt_init(L, d, S, T, betas, wl.SEED)
    assert e.value.code == B.PT_ERR_STATE
    with pytest.raises(B.PTError) as e:
        B.pt_set_workspace_flags(64)
    assert e.value.code == B.PT_ERR_ARG
