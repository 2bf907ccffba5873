"""The checked build of the library (transport kernel compiled -DAEPID_CHECKED: every voxel, tally and queue index and the
invariants of the queue protocol are tested inside the kernel and raise error bit 16) runs the small workloads that exercise
every kernel and the parking / head-room paths of the scheduler, in a process of its own (the binding holds one library)."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_checked_build_runs_the_workloads_without_raising_a_check():
    from paper_2510_24154_b200 import build as b
    lib = b.build_checked()
    env = dict(os.environ, AEPID_LIBRARY=lib)
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_workload.py"), "200000"], env=env, capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-2000:]
    assert "sanitizer workload done" in p.stdout
    # the library that ran is the checked one
    q = subprocess.run([sys.executable, "-c", "import paper_2510_24154_b200.binding as b; print(b.LIB_PATH)"], env=env, capture_output=True, text=True, cwd=ROOT)
    assert q.stdout.strip() == lib
