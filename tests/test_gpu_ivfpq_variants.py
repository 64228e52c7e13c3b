"""Both C1 paths behind FS_IVFPQ_C1 (DESIGN 5.3) against the oracle.

The library reads the variable once per process, so each variant runs the parity cases in a fresh
interpreter."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("variant", ["c1-fused", "c1-matrix-multipass", "c1-matrix-long-rows"])
def test_scan_variant(variant):
    if variant == "c1-fused":          # C1 on the fused engine whatever the shape
        env = dict(os.environ, FS_IVFPQ_C1="fused")
    elif variant == "c1-matrix-multipass":  # C1 through the distance matrix, in passes of 128 queries
        env = dict(os.environ, FS_IVFPQ_C1="matrix", FS_IVFPQ_C1_BYTES="32768")
    else:
        env = dict(os.environ)
    cmd = [sys.executable, "-m", "pytest", "-x", "-q", "-m", "gpu", "-p", "no:cacheprovider",
           os.path.join(ROOT, "tests", "test_gpu_ivfpq.py"),
           "-k", "many_lists_per_item or tiny_config_trained_quantizers"]
    if variant == "c1-matrix-long-rows":
        env = dict(os.environ, FS_IVFPQ_C1="matrix", FS_IVFPQ_C1_BYTES=str(512 * 32768 * 4))
        cmd[-1] = "c1_large_nlist"
    res = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-2000:]
