"""The exact search with its sampled bound switched off, and with a bound that fails for most queries
(FS_FLAT_SAMPLE=off / fail, DESIGN 5.2): the parity cases of test_gpu_flat.py must hold either way -- the
second setting sends nearly every query through the re-run path.  The library reads the variable once per
process, so each variant runs in a fresh interpreter."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("mode", ["off", "fail"])
def test_flat_sample_variant(mode):
    env = dict(os.environ, FS_FLAT_SAMPLE=mode, FS_IVFPQ_C1="fused")
    cmd = [sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider",
           os.path.join(ROOT, "tests", "test_gpu_flat.py"), "-k", "sampled_bound or cfg3_shaped",
           os.path.join(ROOT, "tests", "test_gpu_ivfpq.py") + "::test_c1_large_nlist"]
    res = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-2000:]
