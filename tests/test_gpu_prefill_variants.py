"""The earlier prefill structures stay selectable (FP8ATTN_PREFILL_V = 1: tile-owning softmax warpgroups,
3: boustrophedon quarters with correction warpgroups; DESIGN.md section 5.2a / 5.2c) as cross-checks of the
default kernel: same Alg. 1 values, different schedule.  The variable is read once per
process, so each variant runs a slice of tests/test_gpu_prefill.py in a process of its own."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("variant", ["1", "3"])
def test_variant_passes_the_prefill_parity_slice(variant):
    env = dict(os.environ, FP8ATTN_PREFILL_V=variant)
    sel = "128 and (shape0 or shape3 or shape4 or shape7 or shape8)"
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_prefill.py"), "-x", "-q",
                        "-k", sel], env=env, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert " passed" in r.stdout
