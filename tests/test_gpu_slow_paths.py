"""The rare exact paths of the kernels (in-bucket ranking with pid tie-break, oracle-order Eq. 3
decision, exact direction of the fused histogram) are taken by a tiny fraction of the elements in
a normal run.  `libcuba_slowpaths.so` is the same source compiled with CUBA_FORCE_SLOW_PATHS=1,
where EVERY element takes them; the one-step, many-round, fused-schedule and edge-case parity
tests must pass bit for bit against it too.  Runs in a subprocess because the binding loads one
library per process (CUBA_LIB_PATH selects it)."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_parity_with_every_element_on_the_exact_fallback_paths():
    if os.environ.get("CUBA_SLOWPATHS_CHILD"):
        pytest.skip("already inside the slow-paths run")
    from paper_1208_0961_b200 import build as cuda_build
    lib = cuda_build.build_slowpaths()
    env = dict(os.environ, CUBA_LIB_PATH=lib, CUBA_SLOWPATHS_CHILD="1")
    cmd = [sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_parity.py"), "-m", "gpu", "-x", "-q",
           "-k", "one_step or fused or edge_cases or k_steps"]
    res = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=1500)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-2000:]
    assert " passed" in res.stdout and "failed" not in res.stdout
