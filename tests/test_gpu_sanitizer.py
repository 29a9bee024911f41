"""Sanitizer tier (SURVEY.md section 4 tier 4, section 5): the smallest one-pass case
under compute-sanitizer's racecheck.  The one-pass kernel hands planes between its three roles through
shared memory under nine named barriers and recycles slots by hand; a missing or misplaced barrier
shows up here as a shared-memory hazard long before it shows up as a wrong number.  The full sweep
(memcheck, racecheck, initcheck, synccheck over every path) is recorded in profiles/r3_sanitizer.md."""
import os
import shutil
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def _sanitizer():
    exe = shutil.which("compute-sanitizer")
    if exe is None and os.path.exists("/usr/local/cuda/bin/compute-sanitizer"):
        exe = "/usr/local/cuda/bin/compute-sanitizer"
    return exe


@pytest.mark.skipif(_sanitizer() is None, reason="compute-sanitizer is not installed")
def test_racecheck_on_the_smallest_onepass_case():
    cmd = [_sanitizer(), "--tool", "racecheck", "--racecheck-report", "all", "--error-exitcode", "3",
           sys.executable, os.path.join(HERE, "sanitizer_cases.py"), "onepass_small"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
    out = r.stdout + r.stderr
    if "compute-sanitizer is closed" in out:                         # some GPU pools replace the tool by a stub
        pytest.skip(out.strip().splitlines()[0][:200])
    assert "ran onepass_small" in out, out[-3000:]                   # the run did the work ...
    assert r.returncode == 0, out[-3000:]                            # ... and racecheck had nothing to report
    assert "RACECHECK SUMMARY: 0 hazards displayed (0 errors, 0 warnings)" in out, out[-3000:]
