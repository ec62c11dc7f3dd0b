"""tests/sanitizer_cases.py (the input for compute-sanitizer, which is closed on this GPU pool: profiles/r2_sanitizer.md)
must at least keep running, and checking its own results, without the tool."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_sanitizer_cases_run_plainly():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_cases.py")], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "sanitizer_cases: all cases ran" in r.stdout
