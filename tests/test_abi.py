"""The C-ABI shared library loads and exports every symbol include/ptglass.h declares; argument and state errors
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
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(pt_[a-z_]+|houdayer_step)\s*\(", hdr))
    assert names == set(B.SYMBOLS), names ^ set(B.SYMBOLS)
    for n in names:
        assert hasattr(lib, n)


def test_workspace_bytes_and_shape_errors(lib):
    n = B.pt_workspace_bytes(32, 2, 1024, 32)
    # packed spins 8 MiB + int8 staging 64 MiB dominate
    assert 72 * 2 ** 20 < n < 80 * 2 ** 20
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
