"""GPU parity of the cluster-move variants (readings R36, R37): the
per-temperature single-cluster move counts (separate kernels, fused kernel lane- and warp-per-pair, general-L path)
and the multi-cluster exchange (label propagation in shared memory), through the C ABI, bit for bit against the
oracle; plus C2 and C5 at full size with sampled samples.  Run with `-m gpu`."""
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


def same_state(o, tag=""):
    a, b = o.state(), B.state()
    for k in a:
        assert np.array_equal(a[k], b[k]), (tag, k)
    qa, qb = o.measure_overlap(), B.pt_measure_overlap()
    assert np.array_equal(qa[0], qb[0]) and np.array_equal(qa[1], qb[1]), tag


def counts_for(T, kind):
    if kind == "window":                       # moves only in a temperature window (ref. [39])
        c = np.zeros(T, dtype=np.int32)
        c[T // 3: 2 * T // 3 + 1] = 1
        return c
    if kind == "hot":                          # more moves where clusters are small
        return np.array([1 + (3 * (T - 1 - t)) // max(T - 1, 1) for t in range(T)], dtype=np.int32)[::-1].copy()
    rng = np.random.default_rng(T)
    return rng.integers(0, 4, size=T).astype(np.int32)


SHAPES = [
    (8, 2, 3, 6, False), (16, 2, 2, 5, False), (32, 2, 2, 12, False), (32, 2, 1, 40, False),   # lane-per-pair fused
    (64, 2, 2, 4, False), (128, 2, 1, 3, False),                                               # warp-per-pair
    (8, 3, 2, 5, False), (16, 3, 1, 4, False),
    (6, 2, 2, 5, True), (10, 2, 1, 4, True), (4, 3, 2, 4, True), (6, 3, 1, 3, True), (2, 2, 2, 3, True),
]


@pytest.mark.parametrize("L,d,S,T,general", SHAPES)
@pytest.mark.parametrize("kind", ["window", "hot", "random"])
def test_cluster_move_counts_match_oracle(L, d, S, T, general, kind):
    betas = wl.betas_geometric(0.2, 2.5, T) if d == 2 else wl.betas_geometric(0.4, 1.1, T)
    n_clu = counts_for(T, kind)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 5)
    B.pt_open(L, d, S, T, betas, wl.SEED, 5, general=general)
    o.set_cluster_moves(n_clu)
    B.pt_set_cluster_moves(n_clu)
    for n in range(4):                                        # separate kernels, state compared after every call
        o.sweep(1); B.pt_sweep(1)
        o.houdayer_step(); B.houdayer_step()
        same_state(o, "houdayer %d" % n)
        o.exchange(); B.pt_exchange()
    for n in (1, 9):                                          # fused where eligible
        o.mcs(n, 1, 1, True); B.pt_mcs(n, 1, 1, True)
        same_state(o, "mcs %d" % n)
    assert B.pt_recompute_energy()[1] == 0
    last, _ = B.pt_get_cluster_sizes()
    assert (last[:, n_clu == 0] == 0).all()
    # back to the default: one move everywhere
    o.set_cluster_moves(None); B.pt_set_cluster_moves(None)
    o.mcs(3, 1, 1, True); B.pt_mcs(3, 1, 1, True)
    same_state(o, "default again")


def test_all_ones_is_the_default_on_the_device():
    L, d, S, T = 32, 2, 4, 16
    betas = wl.betas_geometric(0.2, 3.0, T)
    B.pt_open(L, d, S, T, betas, wl.SEED)
    B.pt_mcs(20, 1, 1, True)
    ref_state = B.state()
    B.pt_open(L, d, S, T, betas, wl.SEED)
    B.pt_set_cluster_moves(np.ones(T, dtype=np.int32))
    B.pt_mcs(20, 1, 1, True)
    st = B.state()
    for k in st:
        assert np.array_equal(st[k], ref_state[k]), k


def test_cluster_move_arguments():
    B.pt_open(8, 2, 1, 3, [0.5, 0.7, 0.9], wl.SEED)
    with pytest.raises(B.PTError):
        B.pt_set_cluster_moves(np.array([1, -1, 1], dtype=np.int32))
    with pytest.raises(B.PTError):
        B.pt_set_cluster_moves(np.array([1, 65536, 1], dtype=np.int32))
    with pytest.raises(B.PTError):
        B.pt_mcs(1, 1, 3, True)


@pytest.mark.parametrize("L,d,S,T,general", SHAPES + [(12, 2, 1, 3, True), (20, 2, 1, 2, True), (2, 3, 2, 3, True)])
def test_multi_cluster_matches_oracle(L, d, S, T, general):
    betas = wl.betas_geometric(0.2, 2.5, T) if d == 2 else wl.betas_geometric(0.4, 1.1, T)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 2)
    B.pt_open(L, d, S, T, betas, wl.SEED, 2, general=general)
    for n in range(4):
        o.sweep(1); B.pt_sweep(1)
        o.houdayer_multi_step(); B.houdayer_multi_step()
        same_state(o, "multi %d" % n)
        o.exchange(); B.pt_exchange()
    for n in (1, 8):
        o.mcs(n, 1, 2, True); B.pt_mcs(n, 1, 2, True)
        same_state(o, "mcs %d" % n)
    assert B.pt_recompute_energy()[1] == 0
    # mixing the variants in one run keeps parity (they share the Houdayer counter)
    o.houdayer_step(); B.houdayer_step()
    o.houdayer_multi_step(); B.houdayer_multi_step()
    same_state(o, "mixed")


@pytest.mark.parametrize("T", [32, 40, 5])
def test_fused_multi_cluster_on_register_strips(T):
    """2D L = 32: pt_mcs(..., 2, ...) is ONE launch (houdayer_multi_quad: roots by a tournament over the index bits, one Philox
    coin per root, one growth from the chosen roots) -- against the oracle's component labelling and against the separate
    label-equivalence kernel, for one and two groups of 32 temperatures."""
    L, d, S = 32, 2, 3
    betas = wl.betas_geometric(0.2, 3.0, T)
    o = ref.Oracle(L, d, S, T, betas, wl.SEED, 7)
    B.pt_open(L, d, S, T, betas, wl.SEED, 7)
    assert B.pt_get_fused() == 1
    n0 = B.pt_get_launch_count()
    o.mcs(12, 1, 2, True); B.pt_mcs(12, 1, 2, True)
    assert B.pt_get_launch_count() - n0 == 1
    same_state(o, "fused multi, T = %d" % T)
    o.mcs(3, 2, 1, True); B.pt_mcs(3, 2, 1, True)              # the single-cluster move in between: one Houdayer counter
    o.mcs(5, 1, 2, False); B.pt_mcs(5, 1, 2, False)
    same_state(o, "fused multi after mixing, T = %d" % T)
    fused = B.state()
    try:
        B.pt_open(L, d, S, T, betas, wl.SEED, 7)
        B.pt_set_fused(0)
        B.pt_mcs(12, 1, 2, True); B.pt_mcs(3, 2, 1, True); B.pt_mcs(5, 1, 2, False)
        sep = B.state()
    finally:
        B.pt_set_fused(-1)
    for k in fused:
        assert np.array_equal(fused[k], sep[k]), k
    o.close()


def test_multi_cluster_special_cases_on_device():
    L, d, S, T = 16, 2, 3, 4
    N = L * L
    B.pt_open(L, d, S, T, [0.3, 0.6, 0.9, 1.2], wl.SEED)
    s = B.pt_get_spins()
    s2 = s.copy()
    s2[:, 1] = -s2[:, 0]                       # B = -A: one component rooted at site 0: all or nothing
    B.pt_set_spins(s2)
    E0 = B.pt_get_energy()
    B.houdayer_multi_step()
    last, _ = B.pt_get_cluster_sizes()
    assert set(np.unique(last).tolist()) <= {0, N}
    s3 = B.pt_get_spins()
    for smp in range(S):
        for t in range(T):
            exp = s2[smp, 1, t] if last[smp, t] == N else s2[smp, 0, t]
            assert np.array_equal(s3[smp, 0, t], exp)
    assert np.array_equal(B.pt_get_energy(), E0)
    s4 = s.copy()
    s4[:, 1] = s4[:, 0]                        # B = A: nothing to exchange
    B.pt_set_spins(s4)
    B.houdayer_multi_step()
    assert (B.pt_get_cluster_sizes()[0] == 0).all() and np.array_equal(B.pt_get_spins(), s4)


def test_multi_cluster_label_array_must_fit_shared_memory():
    B.pt_open(256, 2, 1, 2, [0.5, 0.9], wl.SEED)          # 65 536 sites: 256 KiB of labels per pair
    st0 = B.state()
    for fn in (B.houdayer_multi_step, lambda: B.pt_mcs(1, 1, 2, True)):
        with pytest.raises(B.PTError) as e:
            fn()
        assert e.value.code == B.PT_ERR_ARG
    st1 = B.state()
    for k in st0:
        assert np.array_equal(st0[k], st1[k]), k           # a refused call leaves the state and the counters alone
    B.houdayer_step()                                      # the single-cluster move still runs at this size
    assert B.pt_recompute_energy()[1] == 0


@pytest.mark.parametrize("name,n_mcs", [("C2", 30), ("C5", 8)])
def test_variants_full_size_sampled(name, n_mcs):
    """Full L, T, S of the config; samples {0, S/2, S-1} recomputed by the oracle through sample_offset."""
    w = wl.CONFIGS[name]
    n_clu = counts_for(w.T, "hot")
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    B.pt_set_cluster_moves(n_clu)
    E0 = B.pt_get_energy().sum(axis=1)
    B.pt_mcs(n_mcs, 1, 1, True)
    B.pt_set_cluster_moves(None)
    B.pt_mcs(n_mcs // 2, 1, 2, True)
    st = B.state()
    assert B.pt_recompute_energy()[1] == 0
    Ea = B.pt_get_energy().sum(axis=1)
    B.houdayer_multi_step()
    assert np.array_equal(B.pt_get_energy().sum(axis=1), Ea)      # E1 + E2 conserved on every sample
    assert B.pt_recompute_energy()[1] == 0
    assert E0.shape == Ea.shape
    for g in (0, w.S // 2, w.S - 1):
        o = ref.Oracle(w.L, w.d, 1, w.T, w.betas(), wl.SEED, g)
        o.set_cluster_moves(n_clu)
        o.mcs(n_mcs, 1, 1, True)
        o.set_cluster_moves(None)
        o.mcs(n_mcs // 2, 1, 2, True)
        a = o.state()
        for k in ("spins", "energy", "temp_of_slot", "slot_of_temp", "accepts", "last_size", "cum_size"):
            assert np.array_equal(a[k][0], st[k][g]), (g, k)
