"""Every IVFPQ scan kernel behind FS_IVFPQ_SCAN (DESIGN 5.3) against the oracle.

The library reads the variable once per process, so each variant runs the d = 96 / M = 16 parity
cases (the only shapes the fixed-point kernels take) in a fresh interpreter."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("variant", ["pair", "rot", "grp", "persistent"])
def test_scan_variant(variant):
    env = dict(os.environ, FS_IVFPQ_SCAN=variant)
    cmd = [sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider",
           os.path.join(ROOT, "tests", "test_gpu_ivfpq.py"),
           "-k", "many_lists_per_item or tiny_config_trained_quantizers"]
    res = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-2000:]
