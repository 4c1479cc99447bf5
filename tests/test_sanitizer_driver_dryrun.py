"""tests/sanitizer_driver.py is the FIRST command meant for a GPU box (every kernel once on tiny inputs under
compute-sanitizer, before the -m gpu suite).  Here the script itself runs unchanged, in a subprocess, against the CPU
emulation of the kernels (NRR_DRIVER_LIB): its own code -- argument marshalling, expectations, option handling --
must not be what fails on the box."""
import importlib.util
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _emulated_library():
    spec = importlib.util.spec_from_file_location("build_emul", os.path.join(ROOT, "tests", "cuda_emul", "build_emul.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.build()


def test_sanitizer_driver_runs_on_the_emulated_library():
    env = dict(os.environ, NRR_DRIVER_LIB=_emulated_library())
    for args in ([], ["--quick"]):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_driver.py")] + args, env=env,
                           capture_output=True, text=True, timeout=900, cwd=ROOT)
        tail = (r.stdout + r.stderr)[-2000:]
        assert r.returncode == 0, tail
        assert "ALL OK" in r.stdout and "FAIL" not in r.stdout, tail
