"""Thin Python binding of the C ABI in include/ptglass.h (and the probes of include/ptglass_diag.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libptglass.so.  PyTorch is used for exactly two things: the
device workspace (one uint8 tensor) and the CUDA stream.  There is no CPU fallback: if the shared library is
missing this module raises at import of the first call, and on a box without a CUDA device every compute call
fails with PT_ERR_CUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libptglass.so")

PT_OK, PT_ERR_ARG, PT_ERR_STATE, PT_ERR_OVERFLOW, PT_ERR_CUDA = 0, -1, -2, -3, -4

# every symbol include/ptglass.h and include/ptglass_diag.h (probes) declare: name -> (restype, argtypes)
_vp, _i, _sz = C.c_void_p, C.c_int, C.c_size_t
SYMBOLS = {
    "pt_workspace_bytes": (_i, [_i, _i, _i, _i, C.POINTER(_sz)]),
    "pt_workspace_bytes_ex": (_i, [_i, _i, _i, _i, _i, C.POINTER(_sz)]),
    "pt_set_workspace_flags": (_i, [_i]),
    "pt_get_stage_bytes": (_i, [C.POINTER(_sz)]),
    "pt_is_dev_build": (_i, []),
    "pt_bind": (_i, [_vp, _sz, _vp]),
    "pt_init": (_i, [_i, _i, _i, _i, _vp, C.c_uint64]),
    "pt_init_shard": (_i, [_i, _i, _i, _i, _vp, C.c_uint64, C.c_uint32]),
    "pt_free": (_i, []),
    "pt_sweep": (_i, [_i]),
    "pt_exchange": (_i, []),
    "houdayer_step": (_i, []),
    "houdayer_multi_step": (_i, []),
    "pt_set_cluster_moves": (_i, [_vp]),
    "pt_mcs": (_i, [_i, _i, _i, _i]),
    "pt_set_perm": (_i, [_vp]),
    "pt_set_counters": (_i, [C.c_uint32, C.c_uint32, C.c_uint32]),
    "pt_mcs_measure_device": (_i, [_i, _i, _i, _i, _i, _vp, _vp]),
    "pt_set_fused": (_i, [_i]),
    "pt_get_fused": (_i, [_vp]),
    "pt_schedule_family": (_i, [C.c_double, C.c_double, _i, C.c_double, _vp, _vp]),
    "pt_set_round_trip_tracking": (_i, [_i]),
    "pt_set_coupling_probability": (_i, [C.c_double]),
    "pt_get_round_trips": (_i, [_vp, _vp, _vp]),
    "pt_get_energy": (_i, [_vp]),
    "pt_measure_overlap": (_i, [_vp, _vp]),
    "pt_measure_overlap_profile": (_i, [_vp]),
    "pt_measure_overlap_profile_device": (_i, [_vp]),
    "pt_get_swap_counts": (_i, [_vp, _vp]),
    "pt_get_cluster_sizes": (_i, [_vp, _vp]),
    "pt_get_perm": (_i, [_vp, _vp]),
    "pt_get_energy_device": (_i, [_vp]),
    "pt_measure_overlap_device": (_i, [_vp, _vp]),
    "pt_get_spins": (_i, [_vp]),
    "pt_get_couplings": (_i, [_vp]),
    "pt_get_thresholds": (_i, [_vp, _vp, _sz]),
    "pt_get_counters": (_i, [_vp, _vp, _vp]),
    "pt_set_spins": (_i, [_vp]),
    "pt_set_spins_async": (_i, [_vp]),
    "pt_set_spins_packed": (_i, [_vp]),
    "pt_get_spins_packed": (_i, [_vp]),
    "pt_set_couplings": (_i, [_vp]),
    "pt_recompute_energy": (_i, [_vp, _vp]),
    "pt_set_couplings_fixed": (_i, [_vp, _i]),
    "pt_get_couplings_fixed": (_i, [_vp, _vp]),
    "pt_synchronize": (_i, []),
    "pt_get_launch_count": (_i, [_vp]),
    "pt_set_profiling": (_i, [_i]),
    "pt_get_kernel_times": (_i, [_vp, _vp]),
    "pt_set_sample_groups": (_i, [_i]),
    "pt_set_phase_clocks": (_i, [_i]),
    "pt_get_phase_clocks": (_i, [_vp]),
    "pt_get_path": (_i, [_vp]),
    "pt_force_general_path": (_i, [_i]),
    "pt_exchange_noalloc": (_i, [_i, _i, _i, _i, _vp, C.c_uint64, C.c_uint32, C.c_uint32, _vp, _vp, _vp, _vp, _vp]),
    "pt_philox_selftest": (_i, [_vp, _vp, _vp, _i]),
    "pt_threshold_selftest": (_i, [_vp, _vp, _i]),
    "pt_microbench": (_i, [_i, _i, _i, _vp, _vp, _vp, _vp]),
    "pt_last_error": (C.c_char_p, []),
}

_lib = None


class PTError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("ptglass error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Load libptglass.so (built in-tree by paper_2003_04621_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: run `python -m paper_2003_04621_b200.build` (nvcc, sm_100a) first; "
                              "there is no CPU fallback" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _ck(rc):
    if rc != PT_OK:
        raise PTError(rc, lib().pt_last_error().decode())


def _p(a):
    return None if a is None else a.ctypes.data


# shape of the bound problem, kept only to size the numpy output buffers
_shape = dict(L=0, d=0, S=0, T=0, N=0)
_workspace = None     # keeps the torch tensor alive while bound


def pt_last_error() -> str:
    return lib().pt_last_error().decode()


def pt_workspace_bytes(L, d, n_samples, n_temps) -> int:
    out = _sz()
    _ck(lib().pt_workspace_bytes(L, d, n_samples, n_temps, C.byref(out)))
    return out.value


PT_WS_FIXED_COUPLINGS, PT_WS_FULL_STAGING = 1, 2


def pt_workspace_bytes_ex(L, d, n_samples, n_temps, flags) -> int:
    n = _sz(0)
    _ck(lib().pt_workspace_bytes_ex(L, d, n_samples, n_temps, int(flags), C.byref(n)))
    return n.value


def pt_set_workspace_flags(flags):
    """Which optional parts (PT_WS_*) the bound workspace was sized for; after pt_bind, before pt_init."""
    _ck(lib().pt_set_workspace_flags(int(flags)))


def pt_get_stage_bytes() -> int:
    n = _sz(0)
    _ck(lib().pt_get_stage_bytes(C.byref(n)))
    return n.value


def pt_is_dev_build() -> int:
    return int(lib().pt_is_dev_build())


def pt_bind(workspace, stream=None):
    """workspace: a CUDA uint8 torch tensor; stream: torch.cuda.Stream or None (current stream)."""
    global _workspace
    import torch

    assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()
    s = torch.cuda.current_stream(workspace.device) if stream is None else stream
    _ck(lib().pt_bind(workspace.data_ptr(), workspace.numel(), s.cuda_stream))
    _workspace = (workspace, s)


def pt_init(L, d, n_samples, n_temps, betas, seed, sample_offset=None):
    b = np.ascontiguousarray(betas, dtype=np.float64)
    if b.shape != (n_temps,):
        raise PTError(PT_ERR_ARG, "betas must have shape (n_temps,)")
    if sample_offset is None:
        _ck(lib().pt_init(L, d, n_samples, n_temps, _p(b), seed))
    else:
        _ck(lib().pt_init_shard(L, d, n_samples, n_temps, _p(b), seed, sample_offset))
    _shape.update(L=L, d=d, S=n_samples, T=n_temps, N=L ** d)


def pt_init_shard(L, d, n_samples, n_temps, betas, seed, sample_offset):
    pt_init(L, d, n_samples, n_temps, betas, seed, sample_offset)


def pt_free():
    global _workspace
    _ck(lib().pt_free())
    _workspace = None


def pt_open(L, d, n_samples, n_temps, betas, seed, sample_offset=0, device="cuda:0", stream=None, general=False,
            track_round_trips=False, p_ferro=None, fixed_couplings=False, full_staging=False):
    """Convenience: allocate the workspace with torch, bind it and initialise.  Returns the workspace tensor.
    fixed_couplings: size the workspace for pt_set_couplings_fixed (the int32 coupling arrays, NEXT-3);
    full_staging: a staging area of the whole int8 state (whole-group copies in pt_set_spins_async)."""
    import torch

    flags = (PT_WS_FIXED_COUPLINGS if fixed_couplings else 0) | (PT_WS_FULL_STAGING if full_staging else 0)
    nbytes = pt_workspace_bytes_ex(L, d, n_samples, n_temps, flags)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
    with torch.cuda.device(ws.device):
        pt_bind(ws, stream)
        pt_set_workspace_flags(flags)
        if general:
            pt_force_general_path(0)
        if track_round_trips:
            pt_set_round_trip_tracking(1)
        if p_ferro is not None:
            pt_set_coupling_probability(p_ferro)
        pt_init(L, d, n_samples, n_temps, betas, seed, sample_offset)
    return ws


def pt_schedule_family(T_min, T_max, n_temps, phi):
    """(temps, betas) of Eq. (6)-(7); host only."""
    t = np.zeros(max(n_temps, 0), dtype=np.float64)
    b = np.zeros(max(n_temps, 0), dtype=np.float64)
    _ck(lib().pt_schedule_family(float(T_min), float(T_max), int(n_temps), float(phi), _p(t), _p(b)))
    return t, b


def pt_set_coupling_probability(p_ferro):
    _ck(lib().pt_set_coupling_probability(float(p_ferro)))


def pt_set_round_trip_tracking(on):
    _ck(lib().pt_set_round_trip_tracking(int(on)))


def pt_get_round_trips():
    trips = np.zeros((_shape["S"], 2, _shape["T"]), dtype=np.uint32)
    tau_sum = np.zeros((_shape["S"], 2, 32), dtype=np.uint64)
    tau_cnt = np.zeros((_shape["S"], 2, 32), dtype=np.uint64)
    _ck(lib().pt_get_round_trips(_p(trips), _p(tau_sum), _p(tau_cnt)))
    return trips, tau_sum, tau_cnt


def pt_sweep(n=1):
    _ck(lib().pt_sweep(n))


def pt_exchange():
    _ck(lib().pt_exchange())


def houdayer_step():
    _ck(lib().houdayer_step())


def houdayer_multi_step():
    _ck(lib().houdayer_multi_step())


def pt_set_cluster_moves(n_clu):
    """n_clu: [T] int32 host array of single-cluster moves per temperature, or None for one move everywhere."""
    if n_clu is None:
        _ck(lib().pt_set_cluster_moves(None))
        return
    a = np.ascontiguousarray(n_clu, dtype=np.int32)
    _ck(lib().pt_set_cluster_moves(a.ctypes.data))


def pt_mcs(n_mcs, n_metro=1, do_houdayer=False, do_exchange=True):
    _ck(lib().pt_mcs(n_mcs, n_metro, int(do_houdayer), int(do_exchange)))


def pt_mcs_measure_device(n_mcs, n_metro, do_houdayer, do_exchange, measure_every, Q_rec_dev, QL_rec_dev=None):
    """Q_rec_dev / QL_rec_dev: torch int32 CUDA tensors [n_mcs // measure_every][S][T] (QL optional)."""
    _ck(lib().pt_mcs_measure_device(n_mcs, n_metro, int(do_houdayer), int(do_exchange), int(measure_every),
                                    Q_rec_dev.data_ptr(), None if QL_rec_dev is None else QL_rec_dev.data_ptr()))


def pt_set_perm(slot_of_temp):
    a = np.ascontiguousarray(slot_of_temp, dtype=np.int32)
    if a.shape != (_shape["S"], 2, _shape["T"]):
        raise PTError(PT_ERR_ARG, "slot_of_temp must have shape [S][2][T]")
    _ck(lib().pt_set_perm(_p(a)))


def pt_set_counters(n_sweep, n_exchange, n_houdayer):
    _ck(lib().pt_set_counters(int(n_sweep), int(n_exchange), int(n_houdayer)))


def pt_set_fused(mode):
    _ck(lib().pt_set_fused(mode))


def pt_get_fused() -> int:
    f = C.c_int()
    _ck(lib().pt_get_fused(C.byref(f)))
    return f.value


def pt_get_energy(out=None):
    E = np.empty((_shape["S"], 2, _shape["T"]), dtype=np.int32) if out is None else out
    _ck(lib().pt_get_energy(_p(E)))
    return E


def pt_measure_overlap(link=True):
    Q = np.empty((_shape["S"], _shape["T"]), dtype=np.int32)
    QL = np.empty((_shape["S"], _shape["T"]), dtype=np.int32) if link else None
    _ck(lib().pt_measure_overlap(_p(Q), _p(QL)))
    return Q, QL


def pt_get_energy_device(E_dev):
    _ck(lib().pt_get_energy_device(E_dev.data_ptr()))


def pt_measure_overlap_device(Q_dev, QL_dev=None):
    _ck(lib().pt_measure_overlap_device(Q_dev.data_ptr(), None if QL_dev is None else QL_dev.data_ptr()))


def pt_measure_overlap_profile():
    prof = np.empty((_shape["S"], _shape["T"], _shape["d"], _shape["L"]), dtype=np.int32)
    _ck(lib().pt_measure_overlap_profile(_p(prof)))
    return prof


def pt_measure_overlap_profile_device(prof_dev):
    _ck(lib().pt_measure_overlap_profile_device(prof_dev.data_ptr()))


def pt_get_swap_counts():
    a = np.zeros((_shape["S"], 2, max(_shape["T"] - 1, 0)), dtype=np.uint64)
    b = np.zeros_like(a)
    _ck(lib().pt_get_swap_counts(_p(a), _p(b)))
    return a, b


def pt_get_cluster_sizes():
    last = np.empty((_shape["S"], _shape["T"]), dtype=np.uint32)
    cum = np.empty((_shape["S"], _shape["T"]), dtype=np.uint64)
    _ck(lib().pt_get_cluster_sizes(_p(last), _p(cum)))
    return last, cum


def pt_get_perm():
    tos = np.empty((_shape["S"], 2, _shape["T"]), dtype=np.int32)
    sot = np.empty((_shape["S"], 2, _shape["T"]), dtype=np.int32)
    _ck(lib().pt_get_perm(_p(tos), _p(sot)))
    return tos, sot


def pt_get_spins(out=None):
    s = np.empty((_shape["S"], 2, _shape["T"], _shape["N"]), dtype=np.int8) if out is None else out
    _ck(lib().pt_get_spins(_p(s)))
    return s


def pt_get_couplings():
    J = np.empty((_shape["S"], _shape["d"], _shape["N"]), dtype=np.int8)
    _ck(lib().pt_get_couplings(_p(J)))
    return J


def pt_get_thresholds(thrX_stride):
    thrM = np.zeros((_shape["T"], _shape["d"]), dtype=np.uint32)
    thrX = np.zeros((max(_shape["T"] - 1, 0), thrX_stride), dtype=np.uint32)
    _ck(lib().pt_get_thresholds(_p(thrM), _p(thrX), thrX_stride))
    return thrM, thrX


def pt_get_counters():
    a, b, c = C.c_uint32(), C.c_uint32(), C.c_uint32()
    _ck(lib().pt_get_counters(C.byref(a), C.byref(b), C.byref(c)))
    return a.value, b.value, c.value


def pt_set_spins(spins):
    s = np.ascontiguousarray(spins, dtype=np.int8)
    if s.shape != (_shape["S"], 2, _shape["T"], _shape["N"]):
        raise PTError(PT_ERR_ARG, "spins must have shape [S][2][T][N]")
    _ck(lib().pt_set_spins(_p(s)))


def pt_set_spins_async(spins):
    """spins: a C-contiguous int8 numpy array [S][2][T][N] (pinned for a truly asynchronous copy); must stay alive and
    unchanged until the next synchronising call."""
    assert spins.dtype == np.int8 and spins.flags["C_CONTIGUOUS"]
    _ck(lib().pt_set_spins_async(spins.ctypes.data))


def pt_set_spins_packed(bits):
    """bits: C-contiguous uint32 [S][2][T][ceil(N/32)] (pinned for an asynchronous copy; keep alive until the next sync)."""
    assert bits.dtype == np.uint32 and bits.flags["C_CONTIGUOUS"]
    assert bits.shape == (_shape["S"], 2, _shape["T"], (_shape["N"] + 31) // 32)
    _ck(lib().pt_set_spins_packed(bits.ctypes.data))


def pt_get_spins_packed(out=None):
    shape = (_shape["S"], 2, _shape["T"], (_shape["N"] + 31) // 32)
    b = np.zeros(shape, dtype=np.uint32) if out is None else out
    assert b.dtype == np.uint32 and b.shape == shape and b.flags["C_CONTIGUOUS"]
    _ck(lib().pt_get_spins_packed(b.ctypes.data))
    return b


def pt_set_couplings(J):
    j = np.ascontiguousarray(J, dtype=np.int8)
    if j.shape != (_shape["S"], _shape["d"], _shape["N"]):
        raise PTError(PT_ERR_ARG, "J must have shape [S][d][N]")
    _ck(lib().pt_set_couplings(_p(j)))


def pt_set_couplings_fixed(Jq, frac_bits):
    j = np.ascontiguousarray(Jq, dtype=np.int32)
    if j.shape != (_shape["S"], _shape["d"], _shape["N"]):
        raise PTError(PT_ERR_ARG, "Jq must have shape [S][d][N]")
    _ck(lib().pt_set_couplings_fixed(_p(j), int(frac_bits)))


def pt_get_couplings_fixed():
    j = np.empty((_shape["S"], _shape["d"], _shape["N"]), dtype=np.int32)
    f = C.c_int()
    _ck(lib().pt_get_couplings_fixed(_p(j), C.byref(f)))
    return j, f.value


def pt_recompute_energy():
    E = np.empty((_shape["S"], 2, _shape["T"]), dtype=np.int32)
    bad = C.c_int()
    _ck(lib().pt_recompute_energy(_p(E), C.byref(bad)))
    return E, bad.value


def pt_synchronize():
    _ck(lib().pt_synchronize())


def pt_get_launch_count() -> int:
    n = C.c_uint64()
    _ck(lib().pt_get_launch_count(C.byref(n)))
    return n.value


def pt_set_profiling(on):
    _ck(lib().pt_set_profiling(int(on)))


def pt_get_kernel_times():
    """(ms[5], launches[5]) for the sweep, Houdayer, exchange, measurement and fused-MCS kernels since
    pt_set_profiling."""
    ms = np.zeros(5, dtype=np.float64)
    n = np.zeros(5, dtype=np.uint64)
    _ck(lib().pt_get_kernel_times(_p(ms), _p(n)))
    return ms, n


def pt_set_sample_groups(n):
    _ck(lib().pt_set_sample_groups(int(n)))


def pt_set_phase_clocks(on):
    _ck(lib().pt_set_phase_clocks(int(on)))


def pt_get_phase_clocks():
    """SM clocks summed over the CTAs of the fused launches since pt_set_phase_clocks: sweeps, Houdayer, PT pass, rest."""
    c = np.zeros(4, dtype=np.uint64)
    _ck(lib().pt_get_phase_clocks(_p(c)))
    return c


def pt_get_path() -> int:
    f = C.c_int()
    _ck(lib().pt_get_path(C.byref(f)))
    return f.value


def pt_force_general_path(force):
    _ck(lib().pt_force_general_path(force))


PT_NOALLOC_SCRATCH_BYTES = 4 << 20


def pt_exchange_noalloc(L, d, betas, seed, sample_offset, step, E_dev, slot_of_temp_dev, temp_of_slot_dev,
                        accepts_dev=None, stream=None):
    """One PT pass on the caller's own device arrays, for callers that must not allocate device memory (a hook inside a
    job whose memory pool already owns the card, a loop that cannot take cudaMalloc's device-wide synchronisation): needs
    no workspace, no pt_bind, no pt_init; its scratch is a fixed 4 MiB area inside the library (see include/ptglass.h).
    E_dev [S][2][T] int32 (slot order, read only), slot_of_temp_dev (updated in place) and temp_of_slot_dev (overwritten)
    are torch CUDA int32 tensors of one shape; accepts_dev an int64 / uint64 CUDA tensor [S][2][T-1] or None.  S and T are
    taken from E_dev's shape.  Queued on `stream` (default: torch's current stream of E_dev's device); does not
    synchronise.  Calls whose GPU work may overlap race on the shared scratch: keep them on one stream."""
    import torch

    b = np.ascontiguousarray(betas, dtype=np.float64)
    S, two, T = E_dev.shape
    if two != 2 or b.shape != (T,):
        raise PTError(PT_ERR_ARG, "E_dev must have shape [S][2][T] and betas shape (T,)")
    for a in (E_dev, slot_of_temp_dev, temp_of_slot_dev):
        assert a.is_cuda and a.dtype == torch.int32 and a.is_contiguous() and a.shape == E_dev.shape
    if accepts_dev is not None:
        assert accepts_dev.is_cuda and accepts_dev.element_size() == 8 and accepts_dev.is_contiguous()
        assert tuple(accepts_dev.shape) == (S, 2, max(T - 1, 0))
    with torch.cuda.device(E_dev.device):
        st = torch.cuda.current_stream() if stream is None else stream
        _ck(lib().pt_exchange_noalloc(int(L), int(d), int(S), int(T), _p(b), int(seed), int(sample_offset), int(step),
                                      E_dev.data_ptr(), slot_of_temp_dev.data_ptr(), temp_of_slot_dev.data_ptr(),
                                      None if accepts_dev is None else accepts_dev.data_ptr(), st.cuda_stream))


def pt_philox_selftest(key, ctr):
    k = np.ascontiguousarray(key, dtype=np.uint32)
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    out = np.empty_like(c)
    _ck(lib().pt_philox_selftest(_p(k), _p(c), _p(out), c.shape[0]))
    return out


def pt_threshold_selftest(x):
    """THR(x) from the device double exp for a float64 array x (<= 0)."""
    a = np.ascontiguousarray(x, dtype=np.float64).ravel()
    out = np.zeros(a.size, dtype=np.uint32)
    for i in range(0, a.size, 20000):                       # the staging area is the device scratch
        ai, oi = a[i:i + 20000].copy(), out[i:i + 20000]
        _ck(lib().pt_threshold_selftest(_p(ai), _p(oi), int(ai.size)))
    return out


def pt_microbench(kind, ctas_per_sm=8, iters=2000, device="cuda:0"):
    """Returns (thread-ops per ns, kernel ms) of INT32 microbenchmark `kind` (see ptglass.h)."""
    import torch

    scratch = torch.zeros(64, dtype=torch.uint8, device=device)
    ops, ms = C.c_double(), C.c_double()
    with torch.cuda.device(scratch.device):
        st = torch.cuda.current_stream().cuda_stream
        rc = lib().pt_microbench(kind, ctas_per_sm, iters, scratch.data_ptr(), st, C.byref(ops), C.byref(ms))
    if rc != PT_OK:
        raise PTError(rc, "pt_microbench failed")
    return ops.value, ms.value


def state():
    """Everything the parity tests compare (same keys as oracle.ref.Oracle.state)."""
    tos, sot = pt_get_perm()
    att, acc = pt_get_swap_counts()
    last, cum = pt_get_cluster_sizes()
    return dict(spins=pt_get_spins(), energy=pt_get_energy(), temp_of_slot=tos, slot_of_temp=sot,
                attempts=att, accepts=acc, last_size=last, cum_size=cum,
                counters=np.array(pt_get_counters(), dtype=np.uint32))
