"""Multi-GPU host logic on CPU: world_size-2 `gloo` processes.  The path shards by contiguous
ranges of GLOBAL sample index with no data-path collective; what the ranks share is only (a) the offset rule
rank -> sample_offset = rank * S, (b) the final all-gather of integer observables and (c) the max-over-ranks
timing reduction of bench.py.  Each rank drives the CPU oracle on its shard (the CUDA library needs a GPU); rank 0
checks the gathered observables against one unsharded run, which is pin P8 across processes."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, S_per_rank, out_q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    from oracle import ref
    import workloads as wl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L, d, T, n_mcs = 8, 3, 6, 12
    betas = wl.betas_geometric(0.4, 1.1, T)
    o = ref.Oracle(L, d, S_per_rank, T, betas, wl.SEED, sample_offset=rank * S_per_rank)   # bench.py's offset rule
    o.mcs(n_mcs, 1, True, True)
    E = torch.from_numpy(o.get_energy().copy())
    Q = torch.from_numpy(o.measure_overlap()[0].copy())
    acc = torch.from_numpy(o.get_swap_counts()[1].astype(np.int64))
    gathered = {}
    for name, t in (("E", E), ("Q", Q), ("acc", acc)):
        parts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(parts, t)
        gathered[name] = torch.cat(parts, dim=0).numpy()
    # max-over-ranks timing, as bench.py reduces it
    t_ms = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)
    dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    dist.barrier()
    if rank == 0:
        full = ref.Oracle(L, d, S_per_rank * world, T, betas, wl.SEED, 0)
        full.mcs(n_mcs, 1, True, True)
        ok = (np.array_equal(gathered["E"], full.get_energy())
              and np.array_equal(gathered["Q"], full.measure_overlap()[0])
              and np.array_equal(gathered["acc"], full.get_swap_counts()[1].astype(np.int64))
              and float(t_ms.item()) == 10.0 + 5.0 * (world - 1))
        out_q.put(bool(ok))
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_sharding_matches_single_run():
    import torch.multiprocessing as mp

    from oracle import ref
    ref.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 3, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(240)
        assert p.exitcode == 0
    assert q.get(timeout=10) is True


def _worker_gpu(rank, world, port, S_per_rank, out_q):
    """The same split through the CUDA library: every rank is its own process with its own context on the one GPU of the
    box (the ranks never wait on one another's kernels: no data-path collective), offsets by bench.py's rule."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    from oracle import ref
    from paper_2003_04621_b200 import binding as B
    import workloads as wl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L, d, T, n_mcs = 32, 2, 8, 10
    betas = wl.betas_geometric(0.3, 2.0, T)
    B.pt_open(L, d, S_per_rank, T, betas, wl.SEED, sample_offset=rank * S_per_rank, device="cuda:0")
    B.pt_mcs(n_mcs, 1, True, True)
    mine = {"E": B.pt_get_energy(), "Q": B.pt_measure_overlap()[0], "acc": B.pt_get_swap_counts()[1].astype(np.int64),
            "sot": B.pt_get_perm()[1]}
    gathered = {}
    for name, a in mine.items():
        t = torch.from_numpy(np.ascontiguousarray(a))
        parts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(parts, t)
        gathered[name] = torch.cat(parts, dim=0).numpy()
    dist.barrier()
    if rank == 0:
        S = S_per_rank * world
        B.pt_open(L, d, S, T, betas, wl.SEED, device="cuda:0")          # one unsharded run on the GPU
        B.pt_mcs(n_mcs, 1, True, True)
        one = {"E": B.pt_get_energy(), "Q": B.pt_measure_overlap()[0], "acc": B.pt_get_swap_counts()[1].astype(np.int64),
               "sot": B.pt_get_perm()[1]}
        o = ref.Oracle(L, d, S, T, betas, wl.SEED, 0)                    # and the oracle
        o.mcs(n_mcs, 1, True, True)
        orc = {"E": o.get_energy(), "Q": o.measure_overlap()[0], "acc": o.get_swap_counts()[1].astype(np.int64),
               "sot": o.get_perm()[1]}
        out_q.put(all(np.array_equal(gathered[k], one[k]) and np.array_equal(gathered[k], orc[k]) for k in gathered))
    B.pt_free()
    dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.timeout(600)
def test_two_processes_on_one_gpu_shard_through_the_cuda_library():
    """SURVEY 8(e) across process boundaries: two processes x pt_init_shard(offset = rank * S) x pt_mcs on the GPU, the
    gathered observables equal one unsharded GPU run and the oracle."""
    import torch.multiprocessing as mp

    from oracle import ref
    from paper_2003_04621_b200 import build as build_mod
    ref.build()
    build_mod.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_gpu, args=(r, 2, port, 5, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(500)
        assert p.exitcode == 0
    assert q.get(timeout=10) is True
