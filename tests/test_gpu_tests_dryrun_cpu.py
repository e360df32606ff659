"""The GPU tests of round 2 (tests/test_r2_gpu.py, written after GPU access had closed) run on the CPU with the oracle's
values, rounded to the storage type, standing in for the kernels (tests/gpu_dryrun_plugin.py).  This checks the TESTS:
that their plumbing executes and that their gates accept an exactly rounded result.  Cases that need a device (raw
library calls, full-size configs) or assert which kernel ran are left to the GPU."""
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SKIP = ("every_image or large_plane or workspace_errors or auto_selects or auto_backward_fallback or "
        "auto_backward_on_the_aligned")          # full-size oracle runs, raw library calls, variant asserts


def test_round2_gpu_tests_execute_with_exactly_rounded_results():
    env = dict(os.environ, PYTHONPATH=HERE + os.pathsep + os.environ.get("PYTHONPATH", ""))
    p = subprocess.run([sys.executable, "-m", "pytest", os.path.join(HERE, "test_r2_gpu.py"), "-m", "gpu", "-q", "-p", "no:cacheprovider",
                        "-p", "gpu_dryrun_plugin", "-k", f"not ({SKIP})"], cwd=os.path.dirname(HERE), env=env, stdout=subprocess.PIPE,
                       stderr=subprocess.STDOUT, text=True, timeout=1500)
    tail = p.stdout[-3000:]
    m = re.search(r"(\d+) passed", tail)
    assert p.returncode == 0 and m and int(m.group(1)) >= 60, tail
