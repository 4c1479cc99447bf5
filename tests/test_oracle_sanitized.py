"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: oracle/nrr_oracle.c is
compiled with -fsanitize=address,undefined -fno-sanitize-recover and its entry points are exercised on small inputs
(ragged shapes, masks, volume borders, every connectivity pattern, the warp's clamping) in a subprocess with the
sanitizer runtimes preloaded.  Any out-of-bounds access, signed overflow or misaligned access aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import numpy as np, oracle
from oracle import fem
rng = np.random.default_rng(0)
vol = rng.uniform(0, 1000, (13, 17, 19)).astype(np.float32)
mov = (vol + rng.normal(0, 5, vol.shape)).astype(np.float32)
mask = (rng.uniform(size=vol.shape) < 0.6).astype(np.uint8)
for block, stride in (((3, 3, 3), (1, 1, 1)), ((5, 3, 7), (2, 3, 1)), ((19, 17, 13), (1, 1, 1))):
    for m in (None, mask):
        sel = oracle.select(vol, block, stride, 0.4, m)
        for conn in (6, 18, 26):
            oracle.select_pruned(vol, block, stride, 0.4, m, conn)
        if len(sel["centres"]):
            r = oracle.match(vol, mov, sel["centres"][:40], block, (3, 2, 4))
            assert np.all(np.isfinite(r["ncc"]))
            oracle.ncc_at(vol, mov, sel["centres"][0], block, r["disp"][0])
field = rng.uniform(-30, 30, (3,) + vol.shape).astype(np.float32)
oracle.warp(vol, field)
oracle.variance(rng.uniform(size=7)); oracle.ncc(rng.uniform(size=7), rng.uniform(size=7)); oracle.count(10, 0.3)
print("sanitized oracle ok")
"""


def _runtime(name):
    p = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_runs_clean_under_asan_and_ubsan():
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("sanitizer runtimes not installed")
    env = dict(os.environ, NRR_ORACLE_SANITIZE="1", LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               PYTHONPATH=ROOT, OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", CHILD], capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout + r.stderr)[-3000:]
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
