"""A quick subset of tests/test_gpu_parity.py, run on the CPU against the emulated library (tests/gpu_dryrun): it
checks the GPU tests' own code (signatures, expectations, option handling) and, once more, the kernels' logic."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

QUICK = ("(test_select_parity_small or test_select_uniform or test_select_mask or test_match_parity_small or kernel_families "
         "or zero_blocks or exact_ties or host_forms or moving_stats or (register and tiny) or (warp and dims0) "
         "or (pruned and dims0-6) or staging_timeout or (fem_solve and dims0)) and not 11-11")


def test_gpu_test_file_runs_on_the_emulated_library():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "gpu_dryrun", "run.py"), "-k", QUICK],
                       capture_output=True, text=True, timeout=900, cwd=ROOT)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert " passed" in r.stdout and "failed" not in r.stdout, tail
