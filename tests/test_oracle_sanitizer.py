"""SURVEY section 5, sanitizer row: the host oracle built with -fsanitize=address,undefined replays the worked examples
W1-W3 (and a short run of every move on a 3D lattice) in a subprocess; any out-of-bounds access, use after free, signed
overflow or misaligned access in oracle/ref_ptglass.c aborts that process.  CPU only."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import sys
sys.path.insert(0, %(root)r)
from oracle import ref
ref._LIB = %(lib)r
ref.build = lambda force=False: %(lib)r          # the sanitised build instead of oracle/libref_ptglass.so
from tests import test_oracle_pins as pins
pins.test_survey_worked_examples()
import numpy as np
import workloads as wl
o = ref.Oracle(4, 3, 2, 5, wl.betas_geometric(0.3, 1.5, 5), wl.SEED, 1)
o.mcs(6, 1, True, True)
o.houdayer_multi_step()
o.measure_overlap()
assert o.recompute_energy()[1] == 0
print("sanitised oracle ok")
"""


def test_oracle_under_address_and_undefined_sanitizers(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("gcc has no libasan on this box")
    lib = str(tmp_path / "libref_ptglass_san.so")
    src = os.path.join(ROOT, "oracle", "ref_ptglass.c")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=c99", "-fPIC", "-shared", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", lib, src, "-lm"])
    env = dict(os.environ, LD_PRELOAD=os.path.realpath(asan), ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    out = subprocess.run([sys.executable, "-c", CHILD % dict(root=ROOT, lib=lib)], env=env, capture_output=True, text=True,
                         timeout=600)
    assert out.returncode == 0 and "sanitised oracle ok" in out.stdout, (out.stdout[-2000:], out.stderr[-4000:])
