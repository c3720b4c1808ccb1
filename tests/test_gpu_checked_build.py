"""`compute-sanitizer` is closed on the GPU pool this was developed on, so the memcheck half of SURVEY section 5's "race
detection / sanitizers" row is done by the kernel itself: the -DDUALIP_CHECKED build of the library asserts, inside the
streaming kernel, every staged-row position against the stage capacity, every item index against J before it becomes a
shared-memory or accumulator offset, every x position against nnz, every candidate-list slot, and every row's padded extent
against the stage (csrc/dualip_grad_tma.cuh, DUALIP_CHECK*).  This test re-runs GPU parity tests against that build in a
child pytest (tests/conftest.py swaps the library when DUALIP_TEST_CHECKED=1) and fails on any violation bit: configs 1-2
through dualip_grad with x and dualip_solve, both reductions; ragged rows of every projection kind; near-tied clusters (the
candidate compaction list); rows of 20,000 nonzeros; J*m beyond shared memory.  (The racecheck half has no hand-made
stand-in; what guards it is that every result is bit-reproducible run to run and across pipeline geometries --
test_run_to_run_and_geometry_bit_reproducible, test_pipeline_geometry_does_not_change_a_bit.)"""
import os
import subprocess
import sys

import pytest
import torch

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(os.environ.get("DUALIP_TEST_CHECKED") == "1", reason="this IS the child run")
def test_gpu_parity_tests_pass_on_the_checked_build_without_a_violation():
    assert torch.cuda.is_available()
    env = dict(os.environ, DUALIP_TEST_CHECKED="1")
    sel = ("not direct and (grad_parity_small or clustered_near_ties or very_long_rows or many_items or group_width "
           "or grad_with_x_and_short_solve or count_row_gradient)")
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu and not slow", "-k", sel, "-p", "no:cacheprovider",
                        os.path.join(ROOT, "tests", "test_gpu_parity.py"), os.path.join(ROOT, "tests", "test_gpu_sanitizer_cases.py"),
                        os.path.join(ROOT, "tests", "test_gpu_extensions.py")],
                       cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=1500)
    tail = r.stdout[-3000:]
    assert r.returncode == 0, tail
    assert " passed" in tail and "no tests ran" not in tail, tail
