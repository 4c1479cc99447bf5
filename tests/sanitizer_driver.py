#!/usr/bin/env python
"""TEST INFRASTRUCTURE: one small invocation of every kernel of libnrr_bm.so through the C ABI's host-buffer entry
points (ctypes only -- no torch, so that compute-sanitizer instruments nothing but this library), each checked
against the oracle.  Meant to run under

    compute-sanitizer --tool memcheck  --error-exitcode 1 python tests/sanitizer_driver.py
    compute-sanitizer --tool racecheck --error-exitcode 1 python tests/sanitizer_driver.py --quick
    compute-sanitizer --tool synccheck --error-exitcode 1 python tests/sanitizer_driver.py --quick

on the GPU box BEFORE the -m gpu suite: smallest inputs first, the process exits non-zero at the first mismatch or
non-zero status.  (memcheck / racecheck of the shared-memory staging.)"""
import ctypes
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import oracle                                            # noqa: E402
from nrr_inputs import spherical_mask                    # noqa: E402
from _parity import assert_match_parity, assert_select_parity      # noqa: E402

# NRR_DRIVER_LIB: dry run of this script on the CPU emulation of the kernels (tests/cuda_emul), no GPU needed
L = ctypes.CDLL(os.environ.get("NRR_DRIVER_LIB") or os.path.join(ROOT, "paper_2308_10868_b200", "libnrr_bm.so"))
L.nrr_bm_last_error.restype = ctypes.c_char_p
L.nrr_bm_set_option.argtypes = [ctypes.c_char_p, ctypes.c_double]
vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
i3p = ctypes.POINTER(ctypes.c_int)
L.nrr_bm_select_blocks_host.argtypes = [vp, i3p, i3p, i3p, cd, vp, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci)]
L.nrr_bm_select_blocks_pruned_host.argtypes = [vp, i3p, i3p, i3p, cd, vp, ci, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci)]
L.nrr_bm_match_host.argtypes = [vp, vp, i3p, vp, ci, i3p, i3p, vp, vp]
L.nrr_bm_moving_stats_host.argtypes = [vp, i3p, i3p, vp]
L.nrr_bm_register_host.argtypes = [vp, vp, i3p, i3p, i3p, i3p, cd, vp, vp, ci, ctypes.POINTER(ci), vp, vp]
L.nrr_bm_warp_host.argtypes = [vp, i3p, vp, vp]
L.nrr_bm_match_info.argtypes = [i3p, i3p, i3p, i3p]


def i3(t):
    return (ctypes.c_int * 3)(int(t[0]), int(t[1]), int(t[2]))


def check(rc, what):
    if rc != 0:
        print("FAIL %s: status %d: %s" % (what, rc, L.nrr_bm_last_error().decode()), flush=True)
        sys.exit(2)


def opt(name, v):
    check(L.nrr_bm_set_option(name.encode(), float(v)), "set_option " + name)


def smooth(dims, seed, sigma=1.5):
    from scipy import ndimage
    nx, ny, nz = dims
    v = ndimage.gaussian_filter(np.random.default_rng(seed).standard_normal((nz, ny, nx)), sigma, mode="reflect")
    return ((v - v.min()) / (v.max() - v.min()) * 1000.0).astype(np.float32)


def shift_noise(vol, s, noise, seed):
    nz, ny, nx = vol.shape
    iz = np.clip(np.arange(nz) - s[2], 0, nz - 1)
    iy = np.clip(np.arange(ny) - s[1], 0, ny - 1)
    ix = np.clip(np.arange(nx) - s[0], 0, nx - 1)
    m = vol[np.ix_(iz, iy, ix)].astype(np.float64) + np.random.default_rng(seed).normal(0, noise, size=vol.shape)
    return np.ascontiguousarray(m, dtype=np.float32)


def dims_of(v):
    nz, ny, nx = v.shape
    return (nx, ny, nz)


def cap_of(dims, block, stride):
    return max(1, int(np.prod([max(0, (dims[a] - block[a]) // stride[a] + 1) for a in range(3)])))


def select(vol, block, stride, frac, mask=None, conn=None):
    dims = dims_of(vol)
    cap = cap_of(dims, block, stride)
    blocks = np.empty((cap, 3), np.int32)
    var = np.empty((cap,), np.float64)
    n, nc = ci(0), ci(0)
    mp = None if mask is None else mask.ctypes.data
    if conn is None:
        rc = L.nrr_bm_select_blocks_host(vol.ctypes.data, i3(dims), i3(block), i3(stride), float(frac), mp,
                                         blocks.ctypes.data, cap, ctypes.byref(n), var.ctypes.data, ctypes.byref(nc))
    else:
        rc = L.nrr_bm_select_blocks_pruned_host(vol.ctypes.data, i3(dims), i3(block), i3(stride), float(frac), mp, conn,
                                                blocks.ctypes.data, cap, ctypes.byref(n), var.ctypes.data, ctypes.byref(nc))
    check(rc, "select %s %s" % (dims, block))
    return blocks[:n.value], n.value, nc.value, var[:n.value]


def match(vol, mov, centres, block, window):
    dims = dims_of(vol)
    centres = np.ascontiguousarray(centres, np.int32)
    n = len(centres)
    disp = np.empty((n, 3), np.int32)
    ncc = np.empty((n,), np.float32)
    check(L.nrr_bm_match_host(vol.ctypes.data, mov.ctypes.data, i3(dims), centres.ctypes.data, n, i3(block), i3(window),
                              disp.ctypes.data, ncc.ctypes.data), "match %s %s %s" % (dims, block, window))
    return disp, ncc


def info(dims, block, window):
    out = (ctypes.c_int * 6)()
    check(L.nrr_bm_match_info(i3(dims), i3(block), i3(window), out), "match_info")
    return list(out)


def case_select(dims, block, stride, frac, mask_r, generic=0, conn=None):
    vol = smooth(dims, 100 + dims[0])
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    opt("select_generic", generic)
    got = select(vol, block, stride, frac, mask, conn)
    opt("select_generic", 0)
    ora = oracle.select(vol, block, stride, frac, mask) if conn is None else oracle.select_pruned(vol, block, stride, frac, mask, conn)
    assert_select_parity(got[0], got[1], got[2], ora, got[3])
    print("ok select dims=%s block=%s stride=%s generic=%d conn=%s: N=%d K=%d" % (dims, block, stride, generic, conn, got[2], got[1]), flush=True)


def case_stats(dims, block, generic):
    vol = smooth(dims, 21)
    vol[:6, :8, :9] = 321.0
    out = np.full(vol.shape, -7.0, np.float32)
    opt("boxstat_generic", generic)
    check(L.nrr_bm_moving_stats_host(vol.ctypes.data, i3(dims), i3(block), out.ctypes.data), "moving_stats")
    opt("boxstat_generic", 0)
    win = np.lib.stride_tricks.sliding_window_view(vol.astype(np.float64), block[::-1])
    ss = ((win - win.mean(axis=(3, 4, 5), keepdims=True)) ** 2).sum(axis=(3, 4, 5))
    want = np.where(ss > 1e-9, 1.0 / np.sqrt(np.maximum(ss, 1e-300)), 0.0)
    valid = out[: ss.shape[0], : ss.shape[1], : ss.shape[2]]
    assert np.all(valid[ss <= 1e-9] == 0.0)
    rel = np.abs(valid - want)[ss > 1e-9] * np.sqrt(ss[ss > 1e-9])
    assert rel.max() < 2e-6, rel.max()
    untouched = np.ones(vol.shape, bool)
    untouched[: ss.shape[0], : ss.shape[1], : ss.shape[2]] = False
    assert np.all(out[untouched] == -7.0)
    print("ok moving_stats dims=%s block=%s generic=%d: max rel err %.2e" % (dims, block, generic, rel.max()), flush=True)


def case_match(dims, block, window, opts=None, stride=None, frac=1.0, expect_kernel=None, label=""):
    vol = smooth(dims, 200 + dims[0])
    mov = shift_noise(vol, (1, -1, 1), 20.0, 201 + dims[0])
    sel = oracle.select(vol, block, stride or block, frac)
    for k, v in (opts or {}).items():
        opt(k, v)
    inf = info(dims, block, window)
    d, s = match(vol, mov, sel["centres"], block, window)
    for k in (opts or {}):
        opt(k, 0)
    if expect_kernel is not None:
        assert inf[0] == expect_kernel, inf
    ora = oracle.match(vol, mov, sel["centres"], block, window)
    ex = assert_match_parity(d, s, ora, label=label)
    print("ok match dims=%s block=%s window=%s opts=%s kernel=%d tma=%d G=%d: %d blocks, %d exempt, max|dNCC| %.2e" % (
        dims, block, window, opts, inf[0], inf[3], inf[5], len(d), ex, np.max(np.abs(s.astype(np.float64) - ora["ncc"]))), flush=True)


def case_register():
    from nrr_inputs import CONFIGS, make_pair
    cfg = CONFIGS["tiny"]
    fixed, moving, mask = make_pair(cfg)
    cap = cap_of(cfg.dims, cfg.block, cfg.stride)
    blocks = np.full((cap, 3), -99, np.int32)
    disp = np.full((cap, 3), -99, np.int32)
    ncc = np.full((cap,), -99.0, np.float32)
    n = ci(0)
    check(L.nrr_bm_register_host(fixed.ctypes.data, moving.ctypes.data, i3(cfg.dims), i3(cfg.block), i3(cfg.stride),
                                 i3(cfg.window), float(cfg.frac), None, blocks.ctypes.data, cap, ctypes.byref(n),
                                 disp.ctypes.data, ncc.ctypes.data), "register_host tiny")
    sel = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    assert n.value == len(sel["centres"]) and np.array_equal(blocks[:n.value], sel["centres"])
    ora = oracle.match(fixed, moving, sel["centres"], cfg.block, cfg.window)
    assert_match_parity(disp[:n.value], ncc[:n.value], ora, label="tiny register")
    print("ok register_host tiny: %d blocks" % n.value, flush=True)


def case_warp():
    rng = np.random.default_rng(90)
    dims = (37, 21, 9)
    nx, ny, nz = dims
    img = rng.uniform(0, 1000, (nz, ny, nx)).astype(np.float32)
    field = rng.uniform(-2.5, 2.5, (3, nz, ny, nx)).astype(np.float32)
    out = np.empty_like(img)
    check(L.nrr_bm_warp_host(img.ctypes.data, i3(dims), field.ctypes.data, out.ctypes.data), "warp")
    want = oracle.warp(img, field)
    assert np.max(np.abs(out.astype(np.float64) - want)) <= 8 * 2.0 ** -24 * 1000.0
    print("ok warp", flush=True)


def case_plan():
    """Plans (pre-operative select + records, intra-operative match; slab-pipelined host form; block ranges)."""
    vp = ctypes.c_void_p
    L.nrr_bm_plan_create_host.argtypes = [vp, i3p, i3p, i3p, i3p, cd, vp, ci, ctypes.POINTER(vp)]
    L.nrr_bm_plan_info.argtypes = [vp, i3p, i3p]
    L.nrr_bm_plan_blocks_host.argtypes = [vp, vp, vp]
    L.nrr_bm_plan_match_host.argtypes = [vp, vp, vp, vp]
    L.nrr_bm_plan_destroy.argtypes = [vp]
    dims, block, stride, window, frac = (48, 40, 30), (7, 7, 7), (5, 5, 5), (5, 5, 3), 0.5
    vol = smooth(dims, 500)
    mov = shift_noise(vol, (1, -1, 1), 12.0, 501)
    mask = spherical_mask(dims, 18.0)
    h = vp()
    check(L.nrr_bm_plan_create_host(vol.ctypes.data, i3(dims), i3(block), i3(stride), i3(window), frac, mask.ctypes.data, 0,
                                    ctypes.byref(h)), "plan_create_host")
    n, nc = ci(0), ci(0)
    check(L.nrr_bm_plan_info(h, ctypes.byref(n), ctypes.byref(nc)), "plan_info")
    blocks = np.empty((n.value, 3), np.int32)
    check(L.nrr_bm_plan_blocks_host(h, blocks.ctypes.data, None), "plan_blocks_host")
    sel = oracle.select(vol, block, stride, frac, mask)
    assert n.value == len(sel["centres"]) and np.array_equal(blocks, sel["centres"])
    ora = oracle.match(vol, mov, sel["centres"], block, window)
    for slabs in (4, 1, 7):
        opt("plan_slabs", slabs)
        disp = np.full((n.value, 3), -99, np.int32)
        ncc = np.full((n.value,), -99.0, np.float32)
        check(L.nrr_bm_plan_match_host(h, mov.ctypes.data, disp.ctypes.data, ncc.ctypes.data), "plan_match_host")
        assert_match_parity(disp, ncc, ora, label="plan, %d slabs" % slabs)
    opt("plan_slabs", 4)
    check(L.nrr_bm_plan_destroy(h), "plan_destroy")
    print("ok plan (host form, slabs 4/1/7): %d blocks" % n.value, flush=True)


def case_fem():
    """FEM regularisation: cell table, FP64 scatter, PCG, dense field -- against the oracle's direct solve."""
    from oracle import fem as ofem
    vp = ctypes.c_void_p
    L.nrr_bm_fem_create.argtypes = [i3p, i3p, cd, cd, ctypes.POINTER(vp)]
    L.nrr_bm_fem_solve_host.argtypes = [vp, vp, vp, vp, ci, cd, ci, cd, ci, vp, i3p]
    L.nrr_bm_fem_dense_field_host.argtypes = [vp, vp, vp]
    L.nrr_bm_fem_destroy.argtypes = [vp]
    dims, spacing = (13, 9, 11), (4, 2, 5)
    rng = np.random.default_rng(11)
    msh = ofem.mesh(dims, spacing)
    blocks = np.vstack([msh["xyz"][np.all(msh["xyz"] < np.asarray(dims), axis=1)],
                        np.floor(rng.uniform(0, np.asarray(dims) - 1e-9, (150, 3)))]).astype(np.int32)
    disp = rng.integers(-3, 4, blocks.shape).astype(np.int32)
    ncc = rng.uniform(-0.2, 1.0, len(blocks)).astype(np.float32)
    h = vp()
    check(L.nrr_bm_fem_create(i3(dims), i3(spacing), 3.0, 0.45, ctypes.byref(h)), "fem_create")
    u = np.empty((len(msh["xyz"]), 3))
    it = ci(0)
    check(L.nrr_bm_fem_solve_host(h, blocks.ctypes.data, disp.ctypes.data, ncc.ctypes.data, len(blocks), 0.5, 3, 1e-12, 5000,
                                  u.ctypes.data, ctypes.byref(it)), "fem_solve_host")
    want = ofem.solve(msh, 3.0, 0.45, blocks, disp, ncc, 0.5, 3)["U"]
    assert np.max(np.abs(u - want)) <= 1e-6 * max(1.0, np.max(np.abs(want)))
    field = np.empty((3, dims[2], dims[1], dims[0]), np.float32)
    check(L.nrr_bm_fem_dense_field_host(h, u.ctypes.data, field.ctypes.data), "fem_dense_field_host")
    assert np.max(np.abs(field - ofem.dense_field(msh, u, dims))) <= 2e-6 * max(1.0, np.max(np.abs(u)))
    check(L.nrr_bm_fem_destroy(h), "fem_destroy")
    print("ok fem: %d nodes, %d CG iterations" % (len(u), it.value), flush=True)


def main():
    quick = "--quick" in sys.argv
    # ---- selection: unrolled cubic statistics + single-CTA tail, runtime-shaped statistics, multi-launch select
    case_select((41, 37, 29), (5, 5, 5), (5, 5, 5), 0.30, None)
    case_select((41, 37, 29), (7, 7, 7), (5, 5, 5), 0.25, 15.0)
    if not quick:
        case_select((41, 37, 29), (3, 5, 7), (4, 3, 2), 0.50, 15.0)
        case_select((41, 37, 29), (9, 9, 9), (6, 6, 6), 1.00, None)
        case_select((40, 40, 40), (11, 11, 11), (3, 3, 3), 0.5, None)
        case_select((41, 37, 29), (5, 5, 5), (5, 5, 5), 0.30, None, generic=1)
        case_select((64, 50, 33), (5, 5, 5), (1, 1, 1), 0.05, 20.0, generic=1)
        case_select((48, 44, 40), (3, 3, 3), (1, 1, 1), 0.05, None, conn=26)
    # ---- moving statistics: sliding kernel (each B), generic kernel
    for b in ((5, 7) if quick else (5, 7, 9, 11)):
        case_stats((70, 45, 33), (b, b, b), 0)
    if not quick:
        case_stats((70, 45, 33), (7, 7, 3), 0)
        case_stats((70, 45, 33), (7, 7, 7), 1)
        case_stats((40, 36, 24), (3, 5, 3), 0)
    # ---- matching: pair kernel (TMA / plain staging), rows kernel, generic kernel
    case_match((40, 36, 24), (5, 5, 5), (3, 3, 3), expect_kernel=2, label="pair tma")
    case_match((41, 37, 29), (5, 5, 5), (3, 3, 3), expect_kernel=2, label="pair plain")
    case_match((48, 40, 30), (7, 7, 7), (5, 5, 3), expect_kernel=2)
    if not quick:
        case_match((48, 44, 40), (7, 7, 7), (5, 5, 5), expect_kernel=2, stride=(5, 5, 5), frac=0.5)
        case_match((44, 40, 36), (9, 9, 9), (3, 3, 2), expect_kernel=2)
        case_match((44, 40, 40), (9, 9, 9), (7, 7, 7), expect_kernel=2, frac=0.5)
        case_match((40, 40, 40), (11, 11, 11), (3, 3, 3), expect_kernel=2)
        case_match((36, 32, 28), (5, 5, 5), (7, 7, 1), expect_kernel=2)
        case_match((48, 44, 24), (7, 7, 3), (5, 5, 2), expect_kernel=2)
        case_match((40, 36, 24), (5, 5, 5), (3, 3, 3), {"pair_blocks_per_cta": 3}, expect_kernel=2)
        case_match((40, 36, 24), (5, 5, 5), (3, 3, 3), {"disable_tma": 1}, expect_kernel=2)
    case_match((40, 36, 24), (5, 5, 5), (3, 3, 3), {"force_rows": 1}, expect_kernel=1)
    if not quick:
        case_match((41, 37, 29), (5, 5, 5), (3, 3, 3), {"force_rows": 1}, expect_kernel=1)
        case_match((40, 36, 24), (3, 5, 3), (2, 1, 3), expect_kernel=0)
        case_match((33, 31, 29), (7, 7, 7), (4, 4, 4), expect_kernel=0)
    case_register()
    case_plan()
    if not quick:
        case_warp()
        case_fem()
    print("ALL OK", flush=True)


if __name__ == "__main__":
    main()
