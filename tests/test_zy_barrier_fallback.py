"""-m gpu: the counts kernel's barrier TIME-OUT fallback, executed by the test suite instead of by hand.

Above 128 ranks counts_kernel's CTAs exchange block sums through a grid barrier with a bounded wait; a CTA whose wait
runs out rebuilds its row prefixes from the count matrix itself (deadlock-free by construction).
In a normal run nobody times out, so that branch would never execute.  This test compiles the library once more with
-DXDEV_TEST_FORCE_BARRIER_TIMEOUT (odd CTAs take the fallback although everyone arrived) into a temporary file and
runs the R > 128 parity cases -- AllToAllv through plan slots and graph replays, top-k and AllToAllvDynamic -- against
it in a subprocess (NCCLX_B200_LIB selects the library).  Results must be bit-identical to the oracle either way.
Named test_zy_* so that it is collected near the end (it compiles for ~45 s and `pytest -x` stops at the first failure)."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_forced_barrier_timeout_build_passes_the_large_R_parity_cases(tmp_path):
    from paper_2510_20171_b200 import build as B
    try:
        B.nvcc()
    except RuntimeError:
        pytest.skip("nvcc not available on this box: the variant library cannot be built")
    lib = B.build_variant(["-DXDEV_TEST_FORCE_BARRIER_TIMEOUT"], str(tmp_path / "libncclx_b200_forced_timeout.so"))
    env = dict(os.environ, NCCLX_B200_LIB=lib)
    cmd = [sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-p", "no:cacheprovider",
           "tests/test_gpu_alltoallv.py", "tests/test_gpu_parity_reach.py",
           "-k", "large_R or above_128 or randomised"]
    r = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-4000:]
    assert r.returncode == 0, tail
    assert " passed" in r.stdout and "no tests ran" not in r.stdout, tail
    # the subprocess must really have used the variant library
    probe = subprocess.run([sys.executable, "-c", "from paper_2510_20171_b200 import binding; print(binding.LIB_PATH)"],
                           env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert probe.stdout.strip() == lib
