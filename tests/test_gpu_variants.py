"""The opt-in / fallback edge kernels stay parity-green: the same full-size force parity case (cfg4, bf16, width 128, against the
oracle) is run in a child process per environment switch (the switches are read once per process).
DESIGN.md section 4.1: LSD_EDGE_TMA=1 gathers the backward's rows with TMA gather4 into 128-byte swizzled regions;
LSD_EDGE_FWD4=0 runs the forward instantiation of k_edge_rows (two tiles in flight) instead of k_edge_fwd4.  These are the only
two kernel switches the library still reads (the round-1 / opt-in kernel families behind the others were removed in round 3)."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
@pytest.mark.parametrize("env", [{"LSD_EDGE_TMA": "1"}, {"LSD_EDGE_FWD4": "0"}])
def test_edge_kernel_variant_matches_oracle(env):
    e = dict(os.environ)
    e.update(env)
    cmd = [sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_fullsize.py"), "-q", "-x", "-m", "gpu", "-k",
           "test_full_size_forces_match_oracle and cfg4 and bf16"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=e)
    assert r.returncode == 0, (env, r.stdout[-2000:], r.stderr[-2000:])
    assert " passed" in r.stdout and "no tests ran" not in r.stdout, r.stdout[-500:]
