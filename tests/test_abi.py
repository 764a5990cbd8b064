"""The C-ABI shared library loads and exports every symbol include/ptglass.h and include/ptglass_diag.h declare; argument and state errors
are reported without a GPU.  No compute calls here."""
import os
import re

import numpy as np
import pytest

from paper_2003_04621_b200 import binding as B
from paper_2003_04621_b200 import build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build()
    return B.lib()


def test_header_symbols_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "ptglass.h")).read()
    diag = open(os.path.join(ROOT, "include", "ptglass_diag.h")).read()
    # the probes live in their own header: the method's header declares none of them
    for probe in ("pt_microbench", "pt_philox_selftest", "pt_threshold_selftest", "pt_force_general_path", "pt_is_dev_build"):
        assert re.search(r"\b%s\s*\(" % probe, re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)) is None, probe
        assert re.search(r"\b%s\s*\(" % probe, diag), probe
    hdr = hdr + diag
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(pt_[a-z_]+|houdayer_step|houdayer_multi_step)\s*\(", hdr))
    assert names == set(B.SYMBOLS), names ^ set(B.SYMBOLS)
    for n in names:
        assert hasattr(lib, n)
    assert B.pt_is_dev_build() == 0, "tests must run on the full library, not a PTG_DEV_LATTICE build"


def test_workspace_bytes_and_shape_errors(lib):
    n = B.pt_workspace_bytes(32, 2, 1024, 32)
    # packed spins 8 MiB + the bounded int8 staging area 16 MiB dominate; the int32 couplings of the fixed-point model
    # (8 + 16 MiB) only on request
    assert 24 * 2 ** 20 < n < 32 * 2 ** 20
    assert 48 * 2 ** 20 < B.pt_workspace_bytes_ex(32, 2, 1024, 32, B.PT_WS_FIXED_COUPLINGS) < 56 * 2 ** 20
    assert 72 * 2 ** 20 < B.pt_workspace_bytes_ex(32, 2, 1024, 32, B.PT_WS_FULL_STAGING) < 80 * 2 ** 20
    for args in [(31, 2, 1, 2), (8, 4, 1, 2), (8, 2, 0, 2), (8, 2, 1, 0), (8, 2, 1, 70000), (0, 2, 1, 1), (2048, 3, 1, 1)]:
        with pytest.raises(B.PTError) as e:
            B.pt_workspace_bytes(*args)
        assert e.value.code == B.PT_ERR_ARG
        assert B.pt_last_error()


def test_calls_before_init_are_state_errors(lib):
    B._ck(lib.pt_free())
    for fn in (lambda: B.pt_sweep(1), B.pt_exchange, B.houdayer_step, lambda: B.pt_mcs(1), B.pt_get_counters):
        with pytest.raises(B.PTError) as e:
            fn()
        assert e.value.code == B.PT_ERR_STATE
    b = np.array([0.5, 1.0])
    with pytest.raises(B.PTError) as e:
        lib.pt_bind(None, 0, None) and None
        B._ck(lib.pt_bind(None, 0, None))
    assert e.value.code == B.PT_ERR_ARG
    with pytest.raises(B.PTError) as e:
        B._ck(lib.pt_init(8, 2, 1, 2, b.ctypes.data, 1))
    assert e.value.code == B.PT_ERR_STATE      # nothing bound


def test_schedule_family_host_call_matches_oracle_and_closed_forms(lib):
    """pt_schedule_family is a pure host function (Eq. (6)-(7)): no device needed.  Floating point:
    both sides evaluate the same two pow() calls in double, so the tolerance is 1 ulp (derived: one rounding each in
    pow, the product, the sum and the reciprocal; identical operation order on the same libm gives equality)."""
    from oracle import ref

    for (tmin, tmax, nt, phi) in [(0.2, 1.5, 32, 1.0), (0.2, 1.5, 32, 0.6), (0.2, 1.5, 32, 2.5), (0.1, 3.0, 7, 1.7), (0.5, 0.5, 1, 1.0)]:
        t, b = B.pt_schedule_family(tmin, tmax, nt, phi)
        to, bo = ref.schedule_family(tmin, tmax, nt, phi)
        assert np.all(np.abs(t - to) <= np.spacing(to)) and np.all(np.abs(b - bo) <= np.spacing(bo))
        assert t[0] == tmin and abs(t[-1] - tmax) <= 2 * np.spacing(tmax)
    t, _ = B.pt_schedule_family(0.2, 1.5, 32, 1.0)
    assert np.allclose(t, 0.2 + 1.3 * np.arange(32) / 31, rtol=4e-16, atol=0)        # phi = 1: linear
    for bad in [(0.0, 1.0, 4, 1.0), (1.0, 0.5, 4, 1.0), (0.2, 1.5, 0, 1.0), (0.2, 1.5, 4, 0.0), (0.2, float("inf"), 4, 1.0)]:
        with pytest.raises(B.PTError) as e:
            B.pt_schedule_family(*bad)
        assert e.value.code == B.PT_ERR_ARG
