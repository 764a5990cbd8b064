"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (one pt_mcs call per step,
whole S on the device): C2-C5.  The oracle cannot run a whole config, so
  (i)  sampled samples g in {0, 1, S/2, S-1} are recomputed one by one by the oracle through `sample_offset`
       (every sample is a pure function of (seed, g), pin P8) and compared bit for bit, and
  (ii) size-independent invariants are checked on ALL samples: tracked E == recomputed E, the two maps are inverse
       permutations, attempts == number of passes, accepts <= attempts, Houdayer conserves E1+E2 and Q.
and (iii), SURVEY 8(d)'s parity subset part (i): ALL S samples for the first 16 MCS, full state, against the oracle run
as one process per host core over disjoint `sample_offset` ranges (oracle/pool.py).  Part (ii) of the subset (sampled
samples for the whole 10^4 MCS) is tests/test_gpu_zz_fulllength.py.
Run on the B200 box with `-m gpu`."""
import numpy as np
import pytest

from oracle import ref
from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod
import workloads as wl
from oracle import pool as OP

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()
    yield
    B.pt_free()


def run_like_bench(w, n_mcs):
    """The step of bench.py: pt_mcs in one call (or in chunks of measure_every with the measurement between)."""
    recs = []
    if w.measure_every:
        import torch
        n_rec = n_mcs // w.measure_every
        Qr = torch.empty((n_rec, w.S, w.T), dtype=torch.int32, device="cuda")
        QLr = torch.empty_like(Qr)
        B.pt_mcs_measure_device(n_mcs, 1, w.houdayer, True, w.measure_every, Qr, QLr)
        Qh, QLh = Qr.cpu().numpy(), QLr.cpu().numpy()
        recs = [(Qh[r], QLh[r]) for r in range(n_rec)]
    else:
        B.pt_mcs(n_mcs, 1, w.houdayer, True)
    return recs


def oracle_sample(w, g, n_mcs):
    o = ref.Oracle(w.L, w.d, 1, w.T, w.betas(), wl.SEED, g)
    recs = []
    for m in range(1, n_mcs + 1):
        o.mcs(1, 1, w.houdayer, True)
        if w.measure_every and m % w.measure_every == 0:
            recs.append(o.measure_overlap())
    return o, recs


@pytest.mark.parametrize("name,n_mcs,n_check", [("C2", 100, 4), ("C3", 100, 4), ("C4", 40, 4), ("C5", 20, 3)])
def test_full_size_sampled_parity_and_invariants(name, n_mcs, n_check):
    w = wl.CONFIGS[name]
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    recs = run_like_bench(w, n_mcs)
    st = B.state()
    Q, QL = B.pt_measure_overlap()

    # (ii) invariants on every sample
    assert B.pt_recompute_energy()[1] == 0
    tos, sot = st["temp_of_slot"], st["slot_of_temp"]
    ar = np.broadcast_to(np.arange(w.T), tos.shape)
    assert np.array_equal(np.take_along_axis(tos, sot, axis=2), ar)
    assert np.array_equal(np.take_along_axis(sot, tos, axis=2), ar)
    assert (st["attempts"] == n_mcs).all() and (st["accepts"] <= st["attempts"]).all()
    assert tuple(st["counters"]) == (n_mcs, n_mcs, n_mcs if w.houdayer else 0)
    assert ((Q - w.N) % 2 == 0).all() and (abs(Q) <= w.N).all()
    assert ((QL - w.d * w.N) % 2 == 0).all() and (abs(QL) <= w.d * w.N).all()
    if w.houdayer:
        assert (st["last_size"] <= w.N).all() and (st["cum_size"] >= st["last_size"]).all()

    # (i) sampled samples against the oracle
    for g in [0, 1, w.S // 2, w.S - 1][:n_check]:
        o, orecs = oracle_sample(w, g, n_mcs)
        a = o.state()
        for k in a:
            if k == "counters":
                continue
            assert np.array_equal(a[k][0], st[k][g]), "%s sample %d: %s differs" % (name, g, k)
        Qo, QLo = o.measure_overlap()
        assert np.array_equal(Qo[0], Q[g]) and np.array_equal(QLo[0], QL[g])
        for (qa, qla), (qb, qlb) in zip(orecs, recs):
            assert np.array_equal(qa[0], qb[g]) and np.array_equal(qla[0], qlb[g])
        o.close()


@pytest.mark.parametrize("name", ["C2", "C5"])
def test_full_size_houdayer_conserves_pair_energy_and_overlap(name):
    w = wl.CONFIGS[name]
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    B.pt_mcs(5, 1, True, True)
    E0 = B.pt_get_energy().astype(np.int64)
    Q0, QL0 = B.pt_measure_overlap()
    B.houdayer_step()
    E1 = B.pt_get_energy().astype(np.int64)
    Q1, QL1 = B.pt_measure_overlap()
    assert np.array_equal(E0.sum(axis=1), E1.sum(axis=1))          # E1 + E2 per (sample, temperature)
    assert np.array_equal(Q0, Q1) and np.array_equal(QL0, QL1)
    assert B.pt_recompute_energy()[1] == 0
    assert (B.pt_get_cluster_sizes()[0] > 0).any()


def test_fused_and_separate_launches_agree_at_full_size():
    """pt_mcs fused (one CTA per sample, state resident in shared memory) == the three separate kernels."""
    w = wl.C2
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
    assert B.pt_get_fused() == 1
    B.pt_mcs(12, 1, True, True)
    fused = B.state()
    try:
        B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
        B.pt_set_fused(0)
        assert B.pt_get_fused() == 0
        B.pt_mcs(12, 1, True, True)
        sep = B.state()
    finally:
        B.pt_set_fused(-1)
    for k in fused:
        assert np.array_equal(fused[k], sep[k]), k


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_all_samples_first_16_mcs_full_state(name):
    """SURVEY 8(d) parity subset (i): every one of the S samples of the config for its first 16 MCS in bench.py's launch
    configuration (one pt_mcs / pt_mcs_measure_device call), compared bit for bit on the full state: spins, energies, both
    maps, swap attempts / accepts, last and cumulative cluster sizes, Q, QL (and C3's overlap record after MCS 10).  A
    blockIdx-dependent slip (a wrong Philox counter or slot index for some range of samples) cannot pass this."""
    w = wl.CONFIGS[name]
    n_mcs = 16
    pool = OP.OraclePool()
    try:
        futs = pool.submit_all_samples(w, n_mcs)                # the oracle runs on all host cores while the GPU works
        B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED)
        recs = run_like_bench(w, n_mcs)
        st = B.state()
        st["Q"], st["QL"] = B.pt_measure_overlap()
        assert B.pt_recompute_energy()[1] == 0
        want, orecs = OP.gather(futs, n_mcs)
    finally:
        pool.close()
    for k in OP.STATE_KEYS + ("Q", "QL"):
        if not np.array_equal(want[k], st[k]):
            bad = np.argwhere(want[k] != st[k])
            raise AssertionError("%s after %d MCS: %s differs at %d places, first at %s (sample %d)" % (
                name, n_mcs, k, len(bad), bad[0], bad[0][0]))
    assert len(orecs) == len(recs) == (n_mcs // w.measure_every if w.measure_every else 0)
    for (qa, qla), (qb, qlb) in zip(orecs, recs):
        assert np.array_equal(qa, qb) and np.array_equal(qla, qlb)


@pytest.mark.parametrize("full_staging", [False, True])
def test_int8_state_round_trip_through_the_staging_area_at_full_size(full_staging):
    """C2's 64 MiB int8 state does not fit the bounded 16 MiB staging area: pt_get_spins, pt_set_spins (validated first,
    then packed, chunk by chunk) and pt_set_spins_async (sample groups on streams, chunks within a group) move it in pieces
    of whole samples.  With PT_WS_FULL_STAGING the same calls move it whole / one group per copy.  Same bits either way."""
    import torch
    w = wl.C2
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, full_staging=full_staging)
    # the flag delivers what the header promises: the whole int8 state, or the bounded 16 MiB
    # (without it: 16 MiB plus the few bytes pt_workspace_bytes reserved for a swap table of the largest possible stride)
    sb = B.pt_get_stage_bytes()
    assert sb == w.S * 2 * w.T * w.N if full_staging else (16 << 20) <= sb < (17 << 20)
    B.pt_mcs(3, 1, True, True)
    spins, E = B.pt_get_spins(), B.pt_get_energy()
    B.pt_open(w.L, w.d, w.S, w.T, w.betas(), wl.SEED, full_staging=full_staging)
    B.pt_set_spins(spins)
    assert np.array_equal(B.pt_get_spins(), spins) and B.pt_recompute_energy()[1] == 0
    hs = torch.from_numpy(-spins).pin_memory()
    B.pt_set_spins_async(hs.numpy())
    B.pt_mcs(0, 1, True, True)
    B.pt_synchronize()
    assert np.array_equal(B.pt_get_spins(), -spins) and B.pt_recompute_energy()[1] == 0
    bad = spins.copy(); bad[1000, 1, 31, 1023] = 0
    with pytest.raises(B.PTError) as e:
        B.pt_set_spins(bad)
    assert e.value.code == B.PT_ERR_ARG
    assert np.array_equal(B.pt_get_spins(), -spins)            # a rejected input leaves the state unchanged
