"""pt_exchange_noalloc: the one entry point for callers that must not allocate device memory.

Who that is: a hook that runs inside another program's GPU job after that program's memory pool has taken the card (a
fresh cudaMalloc fails there, or is against the host program's rules), or a loop that cannot take the device-wide
synchronisation cudaMalloc / cudaFree bring while other streams are busy.  Such a caller has no workspace to give to
pt_bind, so this call runs one PT pass on arrays the caller already holds and keeps its scratch (threshold table, signs,
energies by temperature) in a fixed 4 MiB area inside libptglass.so.

What is checked: maps and accept counts equal, bit for bit (integer work: no tolerance), those of the existing path
pt_exchange() on the same state -- on two calls in a row on one problem, then on a second, smaller problem, so that the
second and later calls find the scratch area full of an earlier call's tables and energies; and the refusal of a problem
that does not fit the area.

This file is collected last (pytest --collect-only): with `-x` a failure here hides no other test.  It does not depend on
what ran before it: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod
import workloads as wl


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()
    yield
    B._ck(B.lib().pt_free())


def _pass_both_ways(L, d, betas, offset):
    """One PT pass of the bound problem through pt_exchange_noalloc (on copies of the state in torch tensors) and through
    pt_exchange (on the state itself); returns nothing, asserts equality of everything a pass changes."""
    import torch

    E_slot, bad = B.pt_recompute_energy()               # [S][2][T], slot order
    assert bad == 0
    _, sot0 = B.pt_get_perm()
    _, acc0 = B.pt_get_swap_counts()
    step = B.pt_get_counters()[1]
    E_dev = torch.from_numpy(E_slot).cuda()
    sot_dev = torch.from_numpy(sot0.copy()).cuda()
    tos_dev = torch.full_like(sot_dev, -1)              # must be overwritten entirely
    acc_dev = torch.from_numpy(acc0.view(np.int64).copy()).cuda()
    B.pt_exchange_noalloc(L, d, betas, wl.SEED, offset, step, E_dev, sot_dev, tos_dev, acc_dev)
    B.pt_exchange()                                     # the existing path, same stream
    tos1, sot1 = B.pt_get_perm()
    _, acc1 = B.pt_get_swap_counts()
    torch.cuda.synchronize()
    assert np.array_equal(sot_dev.cpu().numpy(), sot1), "slot_of_temp"
    assert np.array_equal(tos_dev.cpu().numpy(), tos1), "temp_of_slot"
    assert np.array_equal(acc_dev.cpu().numpy().view(np.uint64), acc1), "accepts"
    assert np.array_equal(E_dev.cpu().numpy(), E_slot), "E_dev is an input"
    return int((acc1 - acc0).sum())


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_pt_exchange():
    # problem A: 2D L=32, a hot geometric ladder (swaps accepted and refused), global sample offset 5
    L, d, S, T, off = 32, 2, 6, 20, 5
    betas = wl.betas_geometric(0.2, 3.0, T)
    B.pt_open(L, d, S, T, betas, wl.SEED, off)
    B.pt_mcs(12, 1, True, True)                         # non-trivial energies, permutations and counts
    n_acc = _pass_both_ways(L, d, betas, off)           # first call on this device: does the set-up
    B.pt_sweep(2)
    n_acc += _pass_both_ways(L, d, betas, off)          # second call in a row: the area holds the first call's contents
    assert 0 < n_acc < 2 * S * 2 * (T - 1)              # both outcomes occurred
    # problem B, smaller (its tables end inside what problem A wrote): 3D, unordered ladder with a repeated beta, more
    # than 32 rungs so that the draws come in two batches
    L, d, S, T, off = 8, 3, 3, 37, 0
    betas = np.concatenate([wl.betas_geometric(0.15, 1.2, T - 3), [0.4, 0.4, 0.1]])
    B.pt_open(L, d, S, T, betas, wl.SEED, off)
    B.pt_mcs(5, 1, False, True)
    _pass_both_ways(L, d, betas, off)
    B.pt_sweep(1)
    _pass_both_ways(L, d, betas, off)
    # without the optional counts, and a ladder of one temperature (nothing to swap; the maps are still written)
    import torch

    E1 = torch.zeros((2, 2, 1), dtype=torch.int32, device="cuda")
    sot = torch.zeros_like(E1)
    tos = torch.full_like(E1, 7)
    B.pt_exchange_noalloc(4, 2, np.array([1.0]), 1, 0, 0, E1, sot, tos, None)
    torch.cuda.synchronize()
    assert int(tos.abs().sum()) == 0 and int(sot.abs().sum()) == 0


def test_refuses_what_does_not_fit_the_fixed_area():
    """No GPU needed: sizes and arguments are checked before any CUDA call, and nothing is dereferenced."""
    lib = B.lib()
    S, T = 60000, 64                                    # energies by temperature alone: 60000 * 2 * 64 * 4 B = 29 MiB > 4 MiB
    betas = np.ascontiguousarray(wl.betas_geometric(0.2, 3.0, T))
    fake = np.zeros(4, dtype=np.int32).ctypes.data      # never read: the call fails first
    rc = lib.pt_exchange_noalloc(32, 2, S, T, betas.ctypes.data, 1, 0, 0, fake, fake, fake, None, None)
    assert rc == B.PT_ERR_ARG
    msg = B.pt_last_error()
    assert str(B.PT_NOALLOC_SCRATCH_BYTES) in msg and "pt_bind" in msg
    for args in [(31, 2, 1, 2), (8, 4, 1, 2), (8, 2, 0, 2), (8, 2, 1, 0)]:
        assert lib.pt_exchange_noalloc(*args, betas.ctypes.data, 1, 0, 0, fake, fake, fake, None, None) == B.PT_ERR_ARG
    assert lib.pt_exchange_noalloc(8, 2, 1, 2, betas.ctypes.data, 1, 0, 0, None, fake, fake, None, None) == B.PT_ERR_ARG
