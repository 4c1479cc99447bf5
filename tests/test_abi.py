"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol declared in
include/nrr_bm.h, validates its arguments before touching CUDA, and fails loudly (no CPU fallback) when no
device is present.  No compute call needs a GPU here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def nrr():
    import __graft_entry__ as ge
    ge.build()
    import paper_2308_10868_b200 as p
    return p


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nrr_bm.h")).read()
    return sorted(set(re.findall(r"NRR_BM_API[^;(]*?\b(nrr_bm_\w+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = _declared_symbols()
    assert "nrr_bm_select_blocks" in syms and "nrr_bm_match" in syms
    assert len(syms) >= 10


def test_library_exports_every_declared_symbol(nrr):
    L = nrr.lib()
    for s in _declared_symbols():
        assert hasattr(L, s), "libnrr_bm.so does not export %s" % s
    assert sorted(nrr.EXPORTS) == _declared_symbols()
    assert nrr.nrr_bm_version() == 200


def test_library_is_built_for_sm_100a(nrr):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", nrr.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_argument_validation_happens_before_cuda(nrr):
    L = nrr.lib()
    i3 = lambda a, b, c: (ctypes.c_int * 3)(a, b, c)
    n = ctypes.c_int(0)
    buf = (ctypes.c_float * 8)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    # (dims, block, stride, frac) -> status
    cases = [
        (i3(8, 8, 8), i3(4, 3, 3), i3(1, 1, 1), 0.5, -3),     # even block edge
        (i3(8, 8, 8), i3(3, 0, 3), i3(1, 1, 1), 0.5, -3),
        (i3(8, 0, 8), i3(3, 3, 3), i3(1, 1, 1), 0.5, -2),
        (i3(8, 8, 2), i3(3, 3, 3), i3(1, 1, 1), 0.5, -2),     # block larger than the volume
        (i3(8, 8, 8), i3(3, 3, 3), i3(1, 0, 1), 0.5, -4),
        (i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.0, -6),
        (i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 1.5, -6),
        (i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), float("nan"), -6),
    ]
    for dims, block, stride, frac, want in cases:
        rc = L.nrr_bm_select_blocks(p, dims, block, stride, frac, None, p, 4, ctypes.byref(n), None, None, None)
        assert rc == want, (list(dims), list(block), list(stride), frac, rc)
        assert nrr.lib().nrr_bm_last_error()
    assert L.nrr_bm_select_blocks(None, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.5, None, p, 4, ctypes.byref(n), None, None, None) == -1
    assert L.nrr_bm_select_blocks(p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.5, None, p, -1, ctypes.byref(n), None, None, None) == -11
    assert L.nrr_bm_match(p, p, i3(8, 8, 8), p, 1, i3(3, 3, 3), i3(1, -1, 1), p, p, None) == -5
    assert L.nrr_bm_match(p, p, i3(8, 8, 8), p, -1, i3(3, 3, 3), i3(1, 1, 1), p, p, None) == -11
    assert L.nrr_bm_match(p, None, i3(8, 8, 8), p, 1, i3(3, 3, 3), i3(1, 1, 1), p, p, None) == -1
    assert L.nrr_bm_match(p, p, i3(8, 8, 8), None, 1, i3(3, 3, 3), i3(1, 1, 1), p, p, None) == -1
    # the entry points added in r1c validate the same way
    assert L.nrr_bm_select_blocks_pruned(p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.5, None, 7, p, 4, ctypes.byref(n), None, None, None) == -11
    assert L.nrr_bm_select_blocks_pruned(p, i3(8, 8, 8), i3(3, 2, 3), i3(1, 1, 1), 0.5, None, 6, p, 4, ctypes.byref(n), None, None, None) == -3
    assert L.nrr_bm_register(p, p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, -1, 1), 0.5, None, p, 4, None, p, p, None) == -5
    assert L.nrr_bm_register(p, None, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, 1, 1), 0.5, None, p, 4, None, p, p, None) == -1
    assert L.nrr_bm_register(p, p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, 1, 1), 2.0, None, p, 4, None, p, p, None) == -6
    assert L.nrr_bm_moving_stats(p, i3(8, 8, 8), i3(3, 4, 3), p, None) == -3
    assert L.nrr_bm_moving_stats(None, i3(8, 8, 8), i3(3, 3, 3), p, None) == -1
    assert L.nrr_bm_warp(p, i3(8, 8, 0), p, p, None) == -2
    assert L.nrr_bm_warp(p, i3(8, 8, 8), p, None, None) == -1
    q = ctypes.cast((ctypes.c_float * 8)(), ctypes.c_void_p)
    assert L.nrr_bm_warp(p, i3(2, 2, 2), q, p, None) == -11           # in place
    info = (ctypes.c_int * 6)()
    assert L.nrr_bm_pair_task_table(i3(7, 5, 7), i3(5, 5, 5), None, 0, info) == -11      # not square in-plane: no plan
    assert L.nrr_bm_pair_task_table(i3(7, 7, 7), i3(5, 5, 5), None, 0, info) == -7 and info[0] == 256
    assert nrr.lib().nrr_bm_status_string(-7) == b"NRR_E_CAPACITY"
    assert nrr.lib().nrr_bm_status_string(-12) == b"NRR_E_DEVICE"
    assert L.nrr_bm_set_option(b"no_such_option", 1.0) == -11
    # r2: plans, the parameter sweep, the capacity bound
    g, bnd = ctypes.c_int(0), ctypes.c_int(0)
    assert L.nrr_bm_capacity_bound(i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 0), 0.5, ctypes.byref(g), ctypes.byref(bnd)) == -4
    assert L.nrr_bm_capacity_bound(i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.0, ctypes.byref(g), ctypes.byref(bnd)) == -6
    assert L.nrr_bm_capacity_bound(i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), 0.5, ctypes.byref(g), ctypes.byref(bnd)) == 0
    assert g.value == 216 and 108 <= bnd.value <= 109
    h = ctypes.c_void_p()
    assert L.nrr_bm_plan_create(p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, 1, 1), 0.5, None, 0, None, None) == -1
    assert L.nrr_bm_plan_create(p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, 1, 1), 0.5, None, 5, None, ctypes.byref(h)) == -11
    assert L.nrr_bm_plan_create(p, i3(8, 8, 8), i3(3, 3, 3), i3(1, 1, 1), i3(1, -1, 1), 0.5, None, 0, None, ctypes.byref(h)) == -5
    assert L.nrr_bm_plan_create_host(p, i3(8, 8, 8), i3(2, 3, 3), i3(1, 1, 1), i3(1, 1, 1), 0.5, None, 0, ctypes.byref(h)) == -3
    assert not h.value
    assert L.nrr_bm_plan_match(None, p, p, p, None) == -11 and L.nrr_bm_plan_match_host(None, p, p, p) == -11
    assert L.nrr_bm_plan_info(None, None, None) == -11 and L.nrr_bm_plan_destroy(None) == 0
    assert L.nrr_bm_register_batch(p, p, i3(8, 8, 8), None, None, 0, None, None, None, None, None, None) == 0       # nothing to do
    assert L.nrr_bm_register_batch(p, p, i3(8, 8, 8), None, None, 2, None, None, None, None, None, None) == -1
    fh = ctypes.c_void_p()
    assert L.nrr_bm_fem_create(i3(8, 8, 8), i3(2, 0, 2), 1.0, 0.3, ctypes.byref(fh)) == -4
    assert L.nrr_bm_fem_create(i3(8, 8, 8), i3(2, 2, 2), -1.0, 0.3, ctypes.byref(fh)) == -11
    assert L.nrr_bm_fem_create(i3(8, 8, 8), i3(2, 2, 2), 1.0, 0.5, ctypes.byref(fh)) == -11      # incompressible: lambda is infinite
    assert L.nrr_bm_fem_create(i3(8, 8, 8), i3(2, 2, 2), 1.0, 0.3, None) == -1
    assert not fh.value and L.nrr_bm_fem_destroy(None) == 0
    assert L.nrr_bm_fem_solve(None, p, p, p, 1, 1.0, 1, 1e-10, 10, p, None, None) == -11
    assert L.nrr_bm_fem_dense_field(None, p, p, None) == -11
    assert nrr.lib().nrr_bm_status_string(-13) == b"NRR_E_NOCONV"
    st = (nrr.nrr_bm_setting * 1)()
    st[0].block[:] = [3, 3, 3]; st[0].stride[:] = [1, 1, 1]; st[0].window[:] = [1, 1, 1]; st[0].frac = 7.0
    one = (ctypes.c_void_p * 1)(p.value)
    cap = (ctypes.c_int * 1)(4)
    assert L.nrr_bm_register_batch(p, p, i3(8, 8, 8), None, st, 1, one, cap, None, one, one, None) == -6


def test_match_info_dispatch_table(nrr):
    for b in (5, 7, 9, 11):
        for r in (3, 5, 7, 9):
            info = nrr.nrr_bm_match_info((256, 256, 124), (b, b, b), (r, r, r))
            assert info["fast"] and info["candidates"] == (2 * r + 1) ** 3
            assert info["threads"] % 32 == 0 and 32 <= info["threads"] <= 512
            assert info["smem_bytes"] <= 227 * 1024
    assert nrr.nrr_bm_match_info((256, 256, 60), (7, 7, 7), (5, 5, 3))["fast"]
    assert not nrr.nrr_bm_match_info((256, 256, 60), (7, 5, 7), (5, 5, 3))["fast"]       # not square in-plane
    assert nrr.nrr_bm_match_info((256, 256, 60), (7, 7, 3), (5, 5, 2))["kernel"] == 2     # thick-slice block
    assert nrr.nrr_bm_match_info((254, 256, 60), (7, 7, 7), (5, 5, 3)) == dict(
        nrr.nrr_bm_match_info((256, 256, 60), (7, 7, 7), (5, 5, 3)), tma=False)            # plain-load staging
    assert not nrr.nrr_bm_match_info((256, 256, 60), (7, 7, 7), (4, 4, 4))["fast"]
    with pytest.raises(nrr.NrrError):
        nrr.nrr_bm_match_info((256, 256, 60), (7, 7, 7), (5, 5, 300))       # window beyond every kernel's limits


def test_no_cpu_fallback_without_a_device(nrr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    vol = np.zeros((8, 8, 8), np.float32)
    with pytest.raises(nrr.NrrError) as ei:
        nrr.nrr_bm_match_host(vol, vol, np.zeros((1, 3), np.int32) + 4, (3, 3, 3), (1, 1, 1))
    assert ei.value.status == -10                                           # NRR_E_CUDA, loudly
    with pytest.raises(nrr.NrrError):
        nrr.nrr_bm_select_blocks_host(vol, (3, 3, 3), (1, 1, 1), 0.5)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2308_10868_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "nrr_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "nrr_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2308_10868_b200" not in otext.replace("paper_2308_10868_b200/ (the CUDA path)", "").replace(
        "shares nothing with paper_2308_10868_b200/", "")
