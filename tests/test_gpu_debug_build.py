"""The range-checked build (-DAVM_DEBUG, libavm_debug.so): every table, map, slot, ticket and exchange-area index of the
device code is checked and the kernel traps on a violation.  compute-sanitizer is not available on the GPU pool, so the
tests that stress the slot / ticket / append machinery (edge cases incl. capacity overflow, the relaunch guard with queued
electrons, launch shapes, grid maps, banded runs, a stack of two tetrahedral slabs) are run once more against that build, in a subprocess."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SELECT = ("test_edge_cases or test_relaunch_guard_gives_same_run or test_launch_shape_does_not_change_the_run or "
          "test_run_grid_map_same_seed or test_config2_reduced_same_seed or test_banded_config1_same_seed or "
          "test_overflow_tally_in_every_form or test_two_stacked_tetrahedral_slabs_of_different_size")


def test_stress_tests_pass_under_the_range_checked_build(avm):
    from paper_2509_15377_b200 import build
    so = build.build(defines=["-DAVM_DEBUG"])
    assert os.path.exists(so)
    env = dict(os.environ, AVM_LIBRARY=so)
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-k", SELECT, "-p", "no:cacheprovider",
                        os.path.join(ROOT, "tests", "test_gpu_parity.py"), os.path.join(ROOT, "tests", "test_gpu_banded.py"),
                        os.path.join(ROOT, "tests", "test_gpu_step_forms.py"), os.path.join(ROOT, "tests", "test_gpu_next2.py")],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = r.stdout[-3000:] + r.stderr[-2000:]
    assert r.returncode == 0, tail
    assert "AVM_CHECK failed" not in r.stdout and " passed" in r.stdout, tail
