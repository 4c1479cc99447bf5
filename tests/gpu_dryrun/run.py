"""python tests/gpu_dryrun/run.py [pytest args]: tests/test_gpu_parity.py on the emulated library (see adapter.py)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import adapter  # noqa: E402,F401  (patches torch, installs the stand-in binding)
import pytest  # noqa: E402

sys.exit(pytest.main(["-x", "-q", "-m", "gpu", "-p", "no:cacheprovider",
                      os.path.join(adapter.ROOT, "tests", "test_gpu_parity.py")] + sys.argv[1:]))
