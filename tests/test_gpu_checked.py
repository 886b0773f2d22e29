"""-m gpu: memory checking with the library's own bounds-checked build.  compute-sanitizer is closed on
the GPU pool (profiles/r2_sanitizers.md), so the kernels are compiled a second time with -DMT_CHECKED
(libmuon_transport_checked.so): every index into a global array — inputs, outputs, permutation, parked records, sort
keys, alias tables, field grid, spatial hash — is compared with the array's size before use and counted instead of
dereferenced when it is out of range.  tests/sanitize_target.py runs every schedule, placement and geometry through it
(each case also bit-exact against the oracle) and then proves the checks can fire."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_checked_build_runs_clean_and_can_fire():
    from paper_2512_10520_b200 import build
    lib = build.build(checked=True)
    env = dict(os.environ, MUON_TRANSPORT_LIB=lib)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitize_target.py"), "--checked"], env=env,
                       capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "checked build: 0 violations in every case; self-test fired" in r.stdout
