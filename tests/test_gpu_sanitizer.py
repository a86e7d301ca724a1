"""compute-sanitizer over tests/sanitizer_cases.py (memcheck / racecheck on the shared-memory and TMA
kernels; synccheck and initcheck as well).

B200_PROFILING.md: the four tools in ONE call have left a B200 unusable, so a plain `pytest -m gpu` runs none of them; a tool runs
only when SANITIZER_TOOL names it, one tool per gpurun call:

    SANITIZER_TOOL=racecheck python -m pytest tests/test_gpu_sanitizer.py -m gpu -q

The records of those four calls are in profiles/r2_sanitizer.md.
"""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOOLS = ("memcheck", "racecheck", "synccheck", "initcheck")


@pytest.mark.gpu
@pytest.mark.parametrize("tool", TOOLS)
def test_compute_sanitizer_clean(tool):
    if os.environ.get("SANITIZER_TOOL", "") != tool:
        pytest.skip("set SANITIZER_TOOL=%s to run this tool (one tool per call)" % tool)
    exe = shutil.which("compute-sanitizer") or "/usr/local/cuda/bin/compute-sanitizer"
    if not os.path.exists(exe):
        pytest.skip("compute-sanitizer not installed")
    r = subprocess.run([exe, "--tool", tool, "--print-limit", "20", sys.executable, os.path.join(ROOT, "tests", "sanitizer_cases.py")],
                       capture_output=True, text=True, cwd=ROOT, timeout=3000)
    tail = (r.stdout + r.stderr)[-3000:]
    if "closed on this pool" in tail:
        pytest.skip("compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md); tests/test_gpu_memory_safety.py stands in")
    log = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(log):
        with open(os.path.join(log, "sanitizer_%s.log" % tool), "w") as fh:
            fh.write(r.stdout + r.stderr)
    assert r.returncode == 0, tail
    assert "sanitizer cases ok" in r.stdout, tail
    assert "ERROR SUMMARY: 0 errors" in r.stdout + r.stderr, tail
