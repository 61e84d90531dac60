"""The pool's compute-sanitizer is closed (profiles/README.md), so the memory checking the survey asks for
(PAPER.md :185-187: the paper's own gridding bug was an unchecked race) is done by the library
itself: libgridder_checked.so is the same source compiled with -DGRIDDER_CHECKED, in which every index a kernel
computes -- shared-memory slots, workspace arrays, the caller's buffers -- is compared with its bound and failures
are counted (gridder_check_violations).  The parity tests of the pre-summed, per-visibility, w-plane and
channel-grid paths run once more on that build, in a process of their own; no check may fail."""
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

CODE = r"""
import sys
sys.path.insert(0, {root!r})
sys.path.insert(0, {root!r} + "/tests")
from paper_1003_5575_b200 import build, gridder
gridder.select_library(build.build(checked=True))
import pytest
rc = pytest.main(["-x", "-q", "-m", "gpu", "-p", "no:cacheprovider",
                  "-k", "not checked_build and not config_2 and not large_grid and not run_host",
                  {root!r} + "/tests/test_gpu_presum.py", {root!r} + "/tests/test_gpu_channels.py",
                  {root!r} + "/tests/test_gpu_wplanes.py", {root!r} + "/tests/test_gpu_parity.py"])
v = gridder.check_violations()
print("CHECKED_BUILD_VIOLATIONS", v, "PYTEST_RC", int(rc))
sys.exit(0 if (rc == 0 and v == 0) else 1)
"""


def test_parity_suites_on_the_index_checking_build(repo_root):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    res = subprocess.run([sys.executable, "-c", CODE.format(root=str(repo_root))], capture_output=True, text=True, timeout=1500)
    tail = (res.stdout + res.stderr)[-3000:]
    assert "CHECKED_BUILD_VIOLATIONS 0 PYTEST_RC 0" in res.stdout, tail
    assert res.returncode == 0, tail
