"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit, on the same seeded
inputs: spins, couplings, thresholds, energies, both permutation arrays, swap counts, cluster sizes, overlaps.
Run on the B200 box with `-m gpu`."""
import numpy as np
import pytest

from oracle import ref
from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod
import workloads as wl
from tests import helpers as H

pytestmark = pytest.mark.gpu
SEED = wl.SEED


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()
    yield
    B.pt_free()


def assert_same_state(o, tag=""):
    a, b = o.state(), B.state()
    for k in a:
        if not np.array_equal(a[k], b[k]):
            bad = np.argwhere(a[k] != b[k])
            raise AssertionError("%s %s differs at %d places, first %s: oracle %s gpu %s" % (
                tag, k, len(bad), bad[0], a[k][tuple(bad[0])], b[k][tuple(bad[0])]))
    Qo, QLo = o.measure_overlap()
    Qg, QLg = B.pt_measure_overlap()
    assert np.array_equal(Qo, Qg) and np.array_equal(QLo, QLg), tag + " overlaps differ"
    assert B.pt_recompute_energy()[1] == 0, tag + " tracked energy != recomputed"


def open_both(L, d, S, T, betas, offset=0, general=False):
    o = ref.Oracle(L, d, S, T, betas, SEED, offset)
    B.pt_open(L, d, S, T, betas, SEED, offset, general=general)
    return o


def test_philox_device_known_answers_and_oracle():
    import json, os
    B.pt_open(32, 2, 8, 8, wl.betas_linear(0.2, 1.0, 8), SEED)      # staging area doubles as the scratch
    with open(os.path.join(os.path.dirname(__file__), "golden", "philox_known_answers.json")) as f:
        vecs = json.load(f)["vectors"]
    for v in vecs:
        out = B.pt_philox_selftest([int(k, 16) for k in v["key"]], [[int(c, 16) for c in v["ctr"]]])
        assert ["%08x" % x for x in out[0]] == v["out"]
    rng = np.random.default_rng(3)
    ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    key = np.array([0xdeadbeef, 0x12345678], dtype=np.uint32)
    got = B.pt_philox_selftest(key, ctr)
    assert np.array_equal(got, H.philox_np(key, ctr))
    for n in range(0, 1000, 97):
        assert np.array_equal(got[n], ref.philox(key, ctr[n]))


def test_philox_device_against_the_toolkits_curand_philox():
    """Pin P1, second half (PAPER.md:167 refs [70, 71]): the library's device Philox, the oracle's and the
    CUDA toolkit's own curand_Philox4x32_10(ctr, key) give the same four words, in the same order (R25), for the known
    answers and for counters laid out like the method's five domains."""
    import json, os
    from tests import native

    B.pt_open(32, 2, 8, 8, wl.betas_linear(0.2, 1.0, 8), SEED)
    with open(os.path.join(os.path.dirname(__file__), "golden", "philox_known_answers.json")) as f:
        for v in json.load(f)["vectors"]:
            out = native.curand_philox([int(k, 16) for k in v["key"]], [[int(c, 16) for c in v["ctr"]]])
            assert ["%08x" % x for x in out[0]] == v["out"]
    rng = np.random.default_rng(11)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    # counters shaped like the method's: (index, step, global sample, (domain << 28) | (aux << 24) | (chain << 16) | idx16)
    for k in range(2048):
        dom = 1 + k % 5
        ctr[k] = (k * 7, k // 3, 1000 + k % 11, (dom << 28) | ((k % 3) << 24) | ((k & 1) << 16) | (k % 48))
    key = np.array([SEED & 0xFFFFFFFF, SEED >> 32], dtype=np.uint32)
    lib_words = B.pt_philox_selftest(key, ctr)
    cur_words = native.curand_philox(key, ctr)
    assert np.array_equal(lib_words, cur_words)
    for n in range(0, 4096, 131):
        assert np.array_equal(cur_words[n], ref.philox(key, ctr[n]))


# (L, d, S, T): fast path = L a power of two >= 8; the others run the general-L kernels
SHAPES = [(8, 2, 4, 8), (16, 2, 3, 5), (32, 2, 3, 6), (64, 2, 2, 3), (128, 2, 1, 3),
          (8, 3, 3, 4), (16, 3, 2, 3),
          (2, 2, 2, 3), (4, 2, 3, 4), (6, 2, 2, 5), (10, 2, 2, 3), (12, 2, 1, 2), (20, 2, 1, 2),
          (2, 3, 3, 3), (4, 3, 2, 4), (6, 3, 2, 3), (10, 3, 1, 2),
          # long ladders: several 32-temperature groups in the lane-per-pair Houdayer phase of the fused kernel
          (16, 2, 1, 70), (8, 2, 1, 130), (32, 2, 1, 48), (8, 3, 1, 33),
          # the largest lattices of the word-parallel path
          (256, 2, 1, 2), (32, 3, 1, 2)]


@pytest.mark.parametrize("L,d,S,T", SHAPES)
def test_init_state_matches_oracle(L, d, S, T):
    betas = wl.betas_geometric(0.3, 1.6, T)
    o = open_both(L, d, S, T, betas, offset=5)
    assert np.array_equal(o.get_couplings(), B.pt_get_couplings())
    tm_o, tx_o = o.get_thresholds(64)
    tm_g, tx_g = B.pt_get_thresholds(64)
    assert np.array_equal(tm_o, tm_g) and np.array_equal(tx_o, tx_g)
    assert_same_state(o, "init")
    assert B.pt_get_path() == int(L >= 8 and (L & (L - 1)) == 0 and ((d == 2 and L <= 256) or (d == 3 and L <= 32)))


@pytest.mark.parametrize("L,d,S,T", SHAPES)
def test_sweep_exchange_houdayer_match_oracle(L, d, S, T):
    betas = wl.betas_geometric(0.3, 1.6, T)
    o = open_both(L, d, S, T, betas, offset=1)
    for step in range(6):
        o.sweep(1); B.pt_sweep(1)
        assert_same_state(o, "sweep %d" % step)
        o.houdayer_step(); B.houdayer_step()
        assert_same_state(o, "houdayer %d" % step)
        o.exchange(); B.pt_exchange()
        assert_same_state(o, "exchange %d" % step)
    o.sweep(3); B.pt_sweep(3)               # several sweeps in one residency
    assert_same_state(o, "sweep(3)")
    o.mcs(5, 2, True, True); B.pt_mcs(5, 2, True, True)
    assert_same_state(o, "mcs")


@pytest.mark.parametrize("L,d", [(8, 2), (16, 2), (32, 2), (64, 2), (8, 3), (16, 3)])
def test_general_path_equals_fast_path_and_oracle(L, d):
    S, T = 2, 4
    betas = wl.betas_linear(0.2, 1.4, T)
    o = open_both(L, d, S, T, betas, general=True)
    assert B.pt_get_path() == 0
    o.mcs(4, 1, True, True); B.pt_mcs(4, 1, True, True)
    assert_same_state(o, "general")
    general = B.state()
    B.pt_open(L, d, S, T, betas, SEED, 0)
    assert B.pt_get_path() == 1
    B.pt_mcs(4, 1, True, True)
    fast = B.state()
    for k in fast:
        assert np.array_equal(fast[k], general[k]), k


def test_config_C1_full_run():
    w = wl.C1
    o = open_both(w.L, w.d, w.S, w.T, w.betas())
    done = 0
    for upto in (1, 2, 10, 100, 1000):
        o.mcs(upto - done, 1, False, True); B.pt_mcs(upto - done, 1, False, True)
        done = upto
        assert_same_state(o, "C1 after %d MCS" % upto)
    # the survey's worked example W1 (tests/golden/survey_worked_examples.json)
    assert H.crc(B.pt_get_spins()) == "15a1d815"
    assert B.pt_get_swap_counts()[1].sum(axis=(0, 1)).tolist() == [536, 1136, 2482, 3973, 5292, 6483, 7319]


def test_worked_example_W3_with_houdayer_3d():
    b3 = np.array([0.4 * pow(1.1 / 0.4, t / 3.0) for t in range(4)])
    o = open_both(4, 3, 2, 4, b3)
    o.mcs(100, 1, True, True); B.pt_mcs(100, 1, True, True)
    assert_same_state(o, "W3")
    assert H.crc(B.pt_get_spins()) == "b4e49247"
    assert B.pt_get_cluster_sizes()[1].sum() == 25733


@pytest.mark.parametrize("name,S,n_mcs", [("C2", 6, 40), ("C3", 6, 40), ("C4", 2, 12), ("C5", 1, 6)])
def test_config_shapes_subset(name, S, n_mcs):
    """BASELINE configs C2-C5 at full L, T and beta ladder on the first S samples (every sample is a pure
    function of (seed, global sample index), so a subset run equals the same samples of the full run)."""
    w = wl.CONFIGS[name]
    o = open_both(w.L, w.d, S, w.T, w.betas())
    rec_o, rec_g = [], []
    for m in range(1, n_mcs + 1):
        o.mcs(1, 1, w.houdayer, True); B.pt_mcs(1, 1, w.houdayer, True)
        if w.measure_every and m % w.measure_every == 0:
            rec_o.append(o.measure_overlap()); rec_g.append(B.pt_measure_overlap())
        if m in (1, 2, n_mcs // 2):
            assert_same_state(o, "%s MCS %d" % (name, m))
    assert_same_state(o, "%s end" % name)
    for a, b in zip(rec_o, rec_g):
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_sharding_invariance_and_offsets():
    w = wl.C3
    T = 6
    betas = wl.betas_geometric(0.4, 1.1, T)
    B.pt_open(w.L, w.d, 4, T, betas, SEED, 0)
    B.pt_mcs(10, 1, True, True)
    full = B.state()
    B.pt_open(w.L, w.d, 2, T, betas, SEED, 2)
    B.pt_mcs(10, 1, True, True)
    part = B.state()
    for k in full:
        if k != "counters":
            assert np.array_equal(full[k][2:], part[k]), k


def test_special_cases_and_set_hooks():
    L, d, S, T = 16, 2, 2, 3
    betas = np.array([0.0, 0.0, 0.0])
    o = open_both(L, d, S, T, betas)
    s0 = B.pt_get_spins()
    B.pt_sweep(1)
    assert np.array_equal(B.pt_get_spins(), -s0)              # beta = 0: every site flips
    B.pt_exchange()
    assert np.array_equal(B.pt_get_perm()[1][0, 0], [1, 2, 0])   # equal betas: cyclic shift
    # B = -A: whole lattice exchanged; B = A: nothing happens
    s = s0.copy(); s[:, 1] = -s[:, 0]
    B.pt_set_spins(s)
    E0 = B.pt_get_energy()
    B.houdayer_step()
    assert (B.pt_get_cluster_sizes()[0] == L * L).all()
    assert np.array_equal(B.pt_get_energy(), E0)
    Q, QL = B.pt_measure_overlap()
    assert (Q == -L * L).all() and (QL == d * L * L).all()
    s[:, 1] = s[:, 0]
    B.pt_set_spins(s)
    B.houdayer_step()
    assert (B.pt_get_cluster_sizes()[0] == 0).all() and np.array_equal(B.pt_get_spins(), s)
    # ferromagnet through pt_set_couplings
    B.pt_set_couplings(np.ones((S, d, L * L), dtype=np.int8))
    B.pt_set_spins(np.ones((S, 2, T, L * L), dtype=np.int8))
    assert (B.pt_recompute_energy()[0] == -d * L * L).all()
    with pytest.raises(B.PTError):
        B.pt_set_spins(np.zeros((S, 2, T, L * L), dtype=np.int8))


def test_single_temperature_and_counters():
    o = open_both(8, 3, 2, 1, np.array([0.7]))
    o.mcs(3, 1, True, True); B.pt_mcs(3, 1, True, True)
    assert_same_state(o, "T=1")
    assert B.pt_get_counters() == (3, 3, 3)
    with pytest.raises(B.PTError) as e:
        B.pt_sweep(-1)
    assert e.value.code == B.PT_ERR_ARG


@pytest.mark.parametrize("L,d,S,T,houd,general,n_mcs,every", [
    (8, 3, 5, 6, False, False, 30, 10),        # C3-like: one fused launch, records from the resident state
    (32, 2, 3, 8, True, False, 12, 1),         # a record after every MCS, with the cluster move
    (16, 2, 2, 40, True, False, 25, 10),       # n_mcs not a multiple: two records, five more MCS
    (16, 3, 2, 40, False, False, 20, 5),       # T*W >= 512 without cluster moves: chain-split CTAs -> the separate calls
    (6, 2, 2, 4, True, True, 9, 3),            # general-L path -> the separate calls
    (64, 2, 1, 3, True, False, 6, 2)])
def test_mcs_with_fused_overlap_records(L, d, S, T, houd, general, n_mcs, every):
    import torch

    betas = wl.betas_geometric(0.3, 1.6, T)
    o = open_both(L, d, S, T, betas, offset=3, general=general)
    n_rec = n_mcs // every
    Qr = torch.full((max(n_rec, 1), S, T), -12345, dtype=torch.int32, device="cuda")
    QLr = torch.full_like(Qr, -12345)
    B.pt_mcs_measure_device(n_mcs, 1, houd, True, every, Qr, QLr)
    Qh, QLh = Qr.cpu().numpy(), QLr.cpu().numpy()
    for r in range(n_rec):
        o.mcs(every, 1, houd, True)
        Qo, QLo = o.measure_overlap()
        assert np.array_equal(Qo, Qh[r]) and np.array_equal(QLo, QLh[r]), r
    o.mcs(n_mcs - n_rec * every, 1, houd, True)
    assert_same_state(o, "after the call")
    # Q only
    B.pt_mcs_measure_device(every, 1, houd, True, every, Qr, None)
    o.mcs(every, 1, houd, True)
    assert np.array_equal(o.measure_overlap()[0], Qr.cpu().numpy()[0])
    assert_same_state(o, "Q only")
    with pytest.raises(B.PTError):
        B.pt_mcs_measure_device(4, 1, houd, True, 0, Qr, QLr)


def test_very_long_ladder_walks_on_global_scratch():
    """T > 4096: the PT walk of k_exchange no longer fits its shared-memory scratch and runs on global memory
    (k_exchange<GLOBAL_SCRATCH>); a sample no longer fits the fused kernel either, so pt_mcs issues the separate kernels."""
    L, d, S, T = 8, 2, 2, 4200
    betas = wl.betas_linear(0.1, 2.0, T)
    o = ref.Oracle(L, d, S, T, betas, SEED, 7)
    B.pt_open(L, d, S, T, betas, SEED, 7, track_round_trips=True)
    assert B.pt_get_fused() == 0
    assert_same_state(o, "init")
    for step in range(3):
        o.sweep(1); B.pt_sweep(1)
        o.houdayer_step(); B.houdayer_step()
        o.exchange(); B.pt_exchange()
        assert_same_state(o, "step %d" % step)
    o.mcs(3, 1, True, True); B.pt_mcs(3, 1, True, True)
    assert_same_state(o, "mcs")
    for a, b in zip(o.get_round_trips(), B.pt_get_round_trips()):
        assert np.array_equal(a, b)
    att, acc = B.pt_get_swap_counts()
    assert (att == 6).all() and acc.sum() > 0


@pytest.mark.parametrize("L,d,S,T,general", [(32, 2, 3, 8, False), (8, 3, 2, 6, False), (128, 2, 1, 3, False), (6, 2, 2, 4, True)])
def test_checkpoint_and_resume_continue_bit_identically(L, d, S, T, general):
    """spins + slot_of_temp + the three counters (and the seed) are the complete state (counter-based RNG): a run that is
    re-initialised and restored from them continues exactly like the uninterrupted run and like the oracle."""
    betas = wl.betas_geometric(0.3, 1.6, T)
    o = open_both(L, d, S, T, betas, offset=9, general=general)
    o.mcs(7, 1, True, True); B.pt_mcs(7, 1, True, True)
    o.sweep(2); B.pt_sweep(2)                                   # counters no longer equal to one another
    spins, (tos, sot), counters = B.pt_get_spins(), B.pt_get_perm(), B.pt_get_counters()
    B.pt_open(L, d, S, T, betas, SEED, 9, general=general)      # a fresh context: same couplings from the seed
    B.pt_set_spins(spins)
    B.pt_set_perm(sot)
    B.pt_set_counters(*counters)
    assert np.array_equal(B.pt_get_perm()[0], tos)
    o.mcs(9, 1, True, True); B.pt_mcs(9, 1, True, True)
    a, b = o.state(), B.state()
    for k in ("spins", "energy", "temp_of_slot", "slot_of_temp", "last_size", "counters"):
        assert np.array_equal(a[k], b[k]), k
    assert B.pt_recompute_energy()[1] == 0
    # the observables that count since init restart at the re-init (ptglass.h): 9 passes, not the restored step counter
    assert (b["attempts"] == 9).all() and (b["accepts"] <= b["attempts"]).all()
    with pytest.raises(B.PTError) as e:                         # not a permutation
        bad = sot.copy(); bad[0, 0, 0] = bad[0, 0, 1]
        B.pt_set_perm(bad)
    assert e.value.code == B.PT_ERR_ARG


@pytest.mark.parametrize("L,d,general", [(64, 2, False), (8, 3, False), (6, 2, True)])
def test_sample_groups_on_side_streams_do_not_change_results(L, d, general):
    """The separate-kernel MCS loop cuts the samples into groups that run on their own streams (pt_set_sample_groups):
    samples never interact (P:7), so every grouping gives the oracle's state, bit for bit (pin P8 on the device)."""
    S, T = 11, 6
    betas = wl.betas_geometric(0.3, 1.8, T)
    try:
        B.pt_set_fused(0)                                       # the three separate kernels per MCS
        for groups in (1, 2, 5, 8, -1):
            o = open_both(L, d, S, T, betas, offset=3, general=general)
            B.pt_set_sample_groups(groups)
            o.mcs(6, 1, True, True); B.pt_mcs(6, 1, True, True)
            o.mcs(3, 2, 2, True); B.pt_mcs(3, 2, 2, True)       # multi-cluster variant, two sweeps per MCS
            assert_same_state(o, "groups %d" % groups)
            o.close()
    finally:
        B.pt_set_fused(-1)
    with pytest.raises(B.PTError) as e:
        B.pt_set_sample_groups(0)
    assert e.value.code == B.PT_ERR_ARG
    B.pt_set_sample_groups(-1)


@pytest.mark.parametrize("L,d,general,fused", [(32, 2, False, True), (32, 2, False, False), (8, 3, False, True),
                                                 (128, 2, False, True), (6, 2, True, True), (4, 3, True, True)])
def test_async_chunked_upload_then_mcs_matches_the_oracle(L, d, general, fused):
    """pt_set_spins_async queues sample-chunked copies + packing + energies on the group streams and returns; the MCS that
    follows runs group by group on the same streams.  Same state as the oracle given the same spins, for the fused launch
    (one per group), the separate kernels, the overlap records of a fused measurement, and the general-L path."""
    import torch
    S, T = 7, 5
    betas = wl.betas_geometric(0.3, 1.7, T)
    rng = np.random.default_rng(L * 10 + d)
    spins = (rng.integers(0, 2, size=(S, 2, T, L ** d), dtype=np.int8) * 2 - 1).astype(np.int8)
    hs = torch.from_numpy(spins.copy()).pin_memory()
    try:
        B.pt_set_fused(-1 if fused else 0)
        for groups in (3, 1, -1):
            o = open_both(L, d, S, T, betas, offset=2, general=general)
            B.pt_set_sample_groups(groups)
            o.set_spins(spins)
            B.pt_set_spins_async(hs.numpy())
            o.mcs(5, 1, True, True); B.pt_mcs(5, 1, True, True)
            B.pt_synchronize()
            assert_same_state(o, "async upload, groups %d" % groups)
            # a second upload followed by a fused measurement: the records of every group land in their own rows
            o.set_spins(spins)
            B.pt_set_spins_async(hs.numpy())
            Qr = torch.zeros((2, S, T), dtype=torch.int32, device="cuda"); QLr = torch.zeros_like(Qr)
            B.pt_mcs_measure_device(4, 1, False, True, 2, Qr, QLr)
            recs = []
            for _ in range(2):
                o.mcs(2, 1, False, True)
                recs.append(o.measure_overlap())
            B.pt_synchronize()
            for r in range(2):
                assert np.array_equal(Qr[r].cpu().numpy(), recs[r][0]) and np.array_equal(QLr[r].cpu().numpy(), recs[r][1])
            assert_same_state(o, "async upload + fused measurement, groups %d" % groups)
            o.close()
        # values other than +1/-1 are taken by their sign and reported by the next pt_synchronize
        bad = hs.numpy().copy(); bad[1, 0, 2, 5] = 3; bad[2, 1, 0, 0] = -7
        hb = torch.from_numpy(bad).pin_memory()
        B.pt_set_spins_async(hb.numpy())
        with pytest.raises(B.PTError) as e:
            B.pt_synchronize()
        assert e.value.code == B.PT_ERR_ARG
        B.pt_synchronize()                                      # reported once
        assert np.array_equal(B.pt_get_spins(), np.where(bad < 0, -1, 1).astype(np.int8))
    finally:
        B.pt_set_fused(-1)
        B.pt_set_sample_groups(-1)


@pytest.mark.parametrize("L,d,general", [(32, 2, False), (8, 2, False), (128, 2, False), (16, 3, False), (6, 2, True), (4, 3, True), (10, 2, True)])
def test_bit_packed_boundary_round_trip_and_dynamics(L, d, general):
    """pt_set_spins_packed / pt_get_spins_packed carry the state as natural-order bit maps (bit i = site i, 1 <=> -1): same
    state as the int8 calls, and the dynamics that follow match the oracle fed with the int8 array."""
    S, T, N = 5, 4, L ** d
    betas = wl.betas_geometric(0.3, 1.7, T)
    rng = np.random.default_rng(L + d)
    spins = (rng.integers(0, 2, size=(S, 2, T, N), dtype=np.int8) * 2 - 1).astype(np.int8)
    NWn = (N + 31) // 32
    padded = np.zeros((S, 2, T, NWn * 32), dtype=np.uint8)
    padded[..., :N] = spins < 0
    bits = np.ascontiguousarray(np.packbits(padded, axis=-1, bitorder="little")).view("<u4").reshape(S, 2, T, NWn)
    o = open_both(L, d, S, T, betas, offset=1, general=general)
    o.set_spins(spins)
    B.pt_set_spins_packed(bits)
    assert np.array_equal(B.pt_get_spins(), spins)
    assert np.array_equal(B.pt_get_spins_packed(), bits)
    assert_same_state(o, "packed upload")
    o.mcs(6, 1, True, True); B.pt_mcs(6, 1, True, True)
    assert_same_state(o, "packed upload + mcs")
    got = B.pt_get_spins_packed()
    back = np.unpackbits(got.view(np.uint8).reshape(S, 2, T, NWn * 4), axis=-1, bitorder="little")[..., :N]
    assert np.array_equal(np.where(back == 1, -1, 1).astype(np.int8), o.get_spins())
    o.close()


def test_counter_overflow_is_refused_and_leaves_the_state_alone():
    L, d, S, T = 8, 2, 2, 4
    betas = wl.betas_geometric(0.3, 1.6, T)
    o = open_both(L, d, S, T, betas)
    top = 2 ** 32 - 1
    B.pt_set_counters(top - 2, top - 1, top - 1)
    B.pt_mcs(1, 2, True, True)                                  # reaches (top, top, top) exactly: allowed
    assert tuple(B.pt_get_counters()) == (top, top, top)
    st0 = B.state()
    assert (st0["attempts"] == 1).all()                         # passes since init, whatever pt_set_counters placed (R20)
    import torch
    Qr = torch.empty((4, S, T), dtype=torch.int32, device="cuda")
    for fn in (lambda: B.pt_sweep(1), B.pt_exchange, B.houdayer_step, B.houdayer_multi_step,
               lambda: B.pt_mcs(1, 1, True, True), lambda: B.pt_mcs(1, 0, False, True), lambda: B.pt_mcs(1, 0, 2, False),
               lambda: B.pt_mcs_measure_device(4, 1, True, True, 1, Qr), lambda: B.pt_mcs_measure_device(3, 0, 2, True, 1, Qr),
               lambda: B.pt_mcs_measure_device(2, 1, False, False, 2, Qr)):
        with pytest.raises(B.PTError) as e:
            fn()
        assert e.value.code == B.PT_ERR_OVERFLOW
    st1 = B.state()
    for k in st0:
        assert np.array_equal(st0[k], st1[k]), k
    B.pt_mcs(0, 1, True, True)                                  # nothing to do: fine
    o.close()
