"""-m gpu: the edge-case, multi-tile and fuzz parity tests once more against libpeek_checked.so
(-DPEEK_CHECKED: every index computed from device data is range-checked against the extents the arrays
were passed with, every workspace piece is followed by a canary verified after the call's last kernel).
compute-sanitizer is closed on this pool; this build stands in for it: a
violation prints its source line and traps, which fails the parity run below."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_parity_suite_on_checked_build():
    from paper_2607_02525_b200 import build
    lib = build.build_libpeek(checked=True)
    env = dict(os.environ, PEEK_LIB=lib)
    sel = ("edge_cases or empty_cache or single_and or wide_root or multi_tile or local_stage or "
           "random_forests or update_matches or small_configs or work_counters or ragged")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_parity.py"),
                        "-x", "-q", "-m", "gpu", "-k", sel, "-p", "no:cacheprovider"],
                       capture_output=True, text=True, env=env, cwd=ROOT, timeout=3000)
    tail = (r.stdout + r.stderr)[-3000:]
    assert "PEEK_CHECKED" not in r.stdout + r.stderr, tail
    assert r.returncode == 0, tail
    assert " passed" in r.stdout, tail
