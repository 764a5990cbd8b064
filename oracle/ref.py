"""ctypes front end of the CPU oracle (oracle/ref_ptglass.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from the product package (oracle/pool.py takes shapes and beta ladders from the neutral top-level
`workloads` module); the product never imports it.  Argument marshalling only --
all arithmetic of the method is in ref_ptglass.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ref_ptglass.c")
_HDR = os.path.join(_HERE, "ref_ptglass.h")
_LIB = os.path.join(_HERE, "libref_ptglass.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math).  Returns the path of the shared object."""
    stale = (not os.path.exists(_LIB)) or any(os.path.getmtime(p) > os.path.getmtime(_LIB) for p in (_SRC, _HDR))
    if force or stale:
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.ref_create.restype = C.c_void_p
        L.ref_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_uint64, C.c_uint32]
        L.ref_create_p.restype = C.c_void_p
        L.ref_create_p.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_uint64, C.c_uint32, C.c_double]
        L.ref_destroy.argtypes = [C.c_void_p]
        L.ref_destroy.restype = None
        L.ref_threshold.restype = C.c_uint32
        L.ref_threshold.argtypes = [C.c_double]
        L.ref_philox4x32_10.restype = None
        L.ref_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        for name, args in {
            "ref_sweep": [C.c_void_p, C.c_int],
            "ref_exchange": [C.c_void_p],
            "ref_houdayer": [C.c_void_p],
            "ref_houdayer_multi": [C.c_void_p],
            "ref_set_cluster_moves": [C.c_void_p, C.c_void_p],
            "ref_mcs": [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int],
            "ref_get_energy": [C.c_void_p, C.c_void_p],
            "ref_measure_overlap": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_get_swap_counts": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_measure_overlap_profile": [C.c_void_p, C.c_void_p],
            "ref_get_cluster_sizes": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_get_perm": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_get_spins": [C.c_void_p, C.c_void_p],
            "ref_get_couplings": [C.c_void_p, C.c_void_p],
            "ref_get_thresholds": [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t],
            "ref_get_counters": [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_set_spins": [C.c_void_p, C.c_void_p],
            "ref_set_couplings": [C.c_void_p, C.c_void_p],
            "ref_recompute_energy": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_set_couplings_fixed": [C.c_void_p, C.c_void_p, C.c_int],
            "ref_get_couplings_fixed": [C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_get_round_trips": [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p],
            "ref_schedule_family": [C.c_double, C.c_double, C.c_int, C.c_double, C.c_void_p, C.c_void_p],
        }.items():
            fn = getattr(L, name)
            fn.restype = C.c_int
            fn.argtypes = args
        _lib = L
    return _lib


def philox(key, ctr) -> np.ndarray:
    k = np.asarray(key, dtype=np.uint32).copy()
    c = np.asarray(ctr, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().ref_philox4x32_10(k.ctypes.data, c.ctypes.data, out.ctypes.data)
    return out


def schedule_family(T_min, T_max, n_temps, phi):
    """(temps, betas) of Eq. (6)-(7)."""
    t = np.zeros(n_temps, dtype=np.float64)
    b = np.zeros(n_temps, dtype=np.float64)
    if lib().ref_schedule_family(float(T_min), float(T_max), int(n_temps), float(phi), t.ctypes.data, b.ctypes.data) != 0:
        raise ValueError("ref_schedule_family rejected the arguments")
    return t, b


def threshold(x: float) -> int:
    return int(lib().ref_threshold(float(x)))


def _p(a):
    return None if a is None else a.ctypes.data


class Oracle:
    """One oracle simulation.  Mirrors the product's call names (pt_* -> methods) so one harness drives both."""

    def __init__(self, L, d, n_samples, n_temps, betas, seed, sample_offset=0, p_ferro=None):
        b = np.ascontiguousarray(betas, dtype=np.float64)
        assert b.shape == (n_temps,)
        self.L, self.d, self.S, self.T = L, d, n_samples, n_temps
        self.N = L ** d
        if p_ferro is None:
            self._h = lib().ref_create(L, d, n_samples, n_temps, b.ctypes.data, seed, sample_offset)
        else:
            self._h = lib().ref_create_p(L, d, n_samples, n_temps, b.ctypes.data, seed, sample_offset, float(p_ferro))
        if not self._h:
            raise ValueError("ref_create rejected the arguments")

    def close(self):
        if self._h:
            lib().ref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != 0:
            raise RuntimeError("oracle call failed: %d" % rc)

    def sweep(self, n=1):
        self._ck(lib().ref_sweep(self._h, n))

    def exchange(self):
        self._ck(lib().ref_exchange(self._h))

    def houdayer_step(self):
        self._ck(lib().ref_houdayer(self._h))

    def houdayer_multi_step(self):
        self._ck(lib().ref_houdayer_multi(self._h))

    def set_cluster_moves(self, n_clu):
        if n_clu is None:
            self._ck(lib().ref_set_cluster_moves(self._h, None))
            return
        a = np.ascontiguousarray(n_clu, dtype=np.int32)
        assert a.shape == (self.T,)
        self._ck(lib().ref_set_cluster_moves(self._h, _p(a)))

    def mcs(self, n_mcs, n_metro=1, do_houdayer=False, do_exchange=True):
        self._ck(lib().ref_mcs(self._h, n_mcs, n_metro, int(do_houdayer), int(do_exchange)))

    def get_energy(self):
        E = np.zeros((self.S, 2, self.T), dtype=np.int32)
        self._ck(lib().ref_get_energy(self._h, _p(E)))
        return E

    def measure_overlap(self):
        Q = np.zeros((self.S, self.T), dtype=np.int32)
        QL = np.zeros((self.S, self.T), dtype=np.int32)
        self._ck(lib().ref_measure_overlap(self._h, _p(Q), _p(QL)))
        return Q, QL

    def measure_overlap_profile(self):
        prof = np.zeros((self.S, self.T, self.d, self.L), dtype=np.int32)
        self._ck(lib().ref_measure_overlap_profile(self._h, _p(prof)))
        return prof

    def get_swap_counts(self):
        a = np.zeros((self.S, 2, max(self.T - 1, 0)), dtype=np.uint64)
        b = np.zeros_like(a)
        self._ck(lib().ref_get_swap_counts(self._h, _p(a), _p(b)))
        return a, b

    def get_cluster_sizes(self):
        last = np.zeros((self.S, self.T), dtype=np.uint32)
        cum = np.zeros((self.S, self.T), dtype=np.uint64)
        self._ck(lib().ref_get_cluster_sizes(self._h, _p(last), _p(cum)))
        return last, cum

    def get_perm(self):
        tos = np.zeros((self.S, 2, self.T), dtype=np.int32)
        sot = np.zeros((self.S, 2, self.T), dtype=np.int32)
        self._ck(lib().ref_get_perm(self._h, _p(tos), _p(sot)))
        return tos, sot

    def get_spins(self):
        s = np.zeros((self.S, 2, self.T, self.N), dtype=np.int8)
        self._ck(lib().ref_get_spins(self._h, _p(s)))
        return s

    def get_couplings(self):
        J = np.zeros((self.S, self.d, self.N), dtype=np.int8)
        self._ck(lib().ref_get_couplings(self._h, _p(J)))
        return J

    def get_thresholds(self, thrX_stride):
        thrM = np.zeros((self.T, self.d), dtype=np.uint32)
        thrX = np.zeros((max(self.T - 1, 0), thrX_stride), dtype=np.uint32)
        self._ck(lib().ref_get_thresholds(self._h, _p(thrM), _p(thrX), thrX_stride))
        return thrM, thrX

    def get_counters(self):
        a, b, c = C.c_uint32(), C.c_uint32(), C.c_uint32()
        self._ck(lib().ref_get_counters(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.int8)
        assert s.shape == (self.S, 2, self.T, self.N)
        self._ck(lib().ref_set_spins(self._h, _p(s)))

    def set_couplings(self, J):
        j = np.ascontiguousarray(J, dtype=np.int8)
        assert j.shape == (self.S, self.d, self.N)
        self._ck(lib().ref_set_couplings(self._h, _p(j)))

    def get_round_trips(self):
        trips = np.zeros((self.S, 2, self.T), dtype=np.uint32)
        tau_sum = np.zeros((self.S, 2, 32), dtype=np.uint64)
        tau_cnt = np.zeros((self.S, 2, 32), dtype=np.uint64)
        self._ck(lib().ref_get_round_trips(self._h, _p(trips), _p(tau_sum), _p(tau_cnt)))
        return trips, tau_sum, tau_cnt

    def set_couplings_fixed(self, Jq, fbits):
        j = np.ascontiguousarray(Jq, dtype=np.int32)
        assert j.shape == (self.S, self.d, self.N)
        self._ck(lib().ref_set_couplings_fixed(self._h, _p(j), int(fbits)))

    def get_couplings_fixed(self):
        j = np.zeros((self.S, self.d, self.N), dtype=np.int32)
        f = C.c_int()
        self._ck(lib().ref_get_couplings_fixed(self._h, _p(j), C.byref(f)))
        return j, f.value

    def recompute_energy(self):
        E = np.zeros((self.S, 2, self.T), dtype=np.int32)
        bad = C.c_int()
        self._ck(lib().ref_recompute_energy(self._h, _p(E), C.byref(bad)))
        return E, bad.value

    def state(self):
        """Everything the parity tests compare, as a dict of arrays (same keys as the product binding)."""
        tos, sot = self.get_perm()
        att, acc = self.get_swap_counts()
        last, cum = self.get_cluster_sizes()
        E_slot, _ = self.recompute_energy()
        return dict(spins=self.get_spins(), energy=self.get_energy(), temp_of_slot=tos, slot_of_temp=sot,
                    attempts=att, accepts=acc, last_size=last, cum_size=cum,
                    counters=np.array(self.get_counters(), dtype=np.uint32))
