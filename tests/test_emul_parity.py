"""CPU tests (-m "not gpu") of the CUDA kernels' LOGIC: the product's .cu sources compiled as plain C++ against
the fiber-per-thread emulation under tests/cuda_emul, called through the C-ABI host entry points and compared
with the oracle under the same acceptance rules as the GPU parity tests (tests/_parity.py).  This catches index,
layout, barrier and tie-rule mistakes without a GPU; it says nothing about hardware behaviour or speed, which the
-m gpu tests and bench.py cover."""
import ctypes

import numpy as np
import pytest

import oracle
import _emul
from nrr_inputs import CONFIGS, make_pair, spherical_mask
from _parity import assert_match_parity, assert_select_parity


def _smooth(dims, seed, sigma=1.5):
    from scipy import ndimage
    nx, ny, nz = dims
    v = ndimage.gaussian_filter(np.random.default_rng(seed).standard_normal((nz, ny, nx)), sigma, mode="reflect")
    return ((v - v.min()) / (v.max() - v.min()) * 1000.0).astype(np.float32)


def _shift_noise(vol, s, noise, seed):
    nz, ny, nx = vol.shape
    iz = np.clip(np.arange(nz) - s[2], 0, nz - 1)
    iy = np.clip(np.arange(ny) - s[1], 0, ny - 1)
    ix = np.clip(np.arange(nx) - s[0], 0, nx - 1)
    m = vol[np.ix_(iz, iy, ix)].astype(np.float64) + np.random.default_rng(seed).normal(0, noise, size=vol.shape)
    return np.ascontiguousarray(m, dtype=np.float32)


@pytest.fixture(autouse=True)
def _default_options():
    for name, v in (("force_rows", 0), ("force_generic", 0), ("disable_tma", 0), ("pair_blocks_per_cta", 0), ("tie_band", 1e-4),
                    ("select_generic", 0), ("boxstat_generic", 0), ("debug_expect_tx_extra", 0)):
        _emul.set_option(name, v)
    yield


@pytest.mark.parametrize("dims,block,stride,frac,mask_r", [
    ((41, 37, 29), (5, 5, 5), (5, 5, 5), 0.30, None),
    ((41, 37, 29), (7, 7, 7), (5, 5, 5), 0.25, 15.0),
    ((41, 37, 29), (3, 5, 7), (4, 3, 2), 0.50, 15.0),
    ((130, 3, 3), (3, 3, 3), (1, 1, 1), 0.10, None),
    ((9, 9, 9), (9, 9, 9), (1, 1, 1), 1.00, None),
])
def test_emulated_selection_matches_the_oracle(dims, block, stride, frac, mask_r):
    vol = _smooth(dims, 100 + dims[0])
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    ora = oracle.select(vol, block, stride, frac, mask)
    for generic in (0, 1):       # single-CTA tail + unrolled statistics / multi-launch radix select + runtime shapes
        _emul.set_option("select_generic", generic)
        blocks, n, ncand, var = _emul.select(vol, block, stride, frac, mask)
        assert_select_parity(blocks, n, ncand, ora, var)
    _emul.set_option("select_generic", 0)


def test_emulated_selection_ties_go_to_the_lower_index():
    vol = np.full((12, 15, 20), 42.0, dtype=np.float32)            # uniform image: first K grid positions
    ora = oracle.select(vol, (3, 3, 3), (3, 3, 3), 0.25)
    blocks, n, ncand, var = _emul.select(vol, (3, 3, 3), (3, 3, 3), 0.25)
    assert_select_parity(blocks, n, ncand, ora, var)
    vol2 = np.zeros((10, 10, 30), dtype=np.float32)                # the same pattern three times: exact variance ties
    pat = np.arange(125, dtype=np.float32).reshape(5, 5, 5)
    for x in (0, 10, 25):
        vol2[0:5, 5:10, x:x + 5] = pat
    for frac in (0.1, 0.17, 0.34):                                  # K cuts through the tied group
        ora = oracle.select(vol2, (5, 5, 5), (5, 5, 5), frac)
        for generic in (0, 1):
            _emul.set_option("select_generic", generic)
            blocks, n, ncand, var = _emul.select(vol2, (5, 5, 5), (5, 5, 5), frac)
            assert_select_parity(blocks, n, ncand, ora, var)
    _emul.set_option("select_generic", 0)


def test_emulated_tiny_config_all_three_matching_kernels():
    cfg = CONFIGS["tiny"]
    fixed, moving, mask = make_pair(cfg)
    ora = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    blocks, n, ncand, var = _emul.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    assert_select_parity(blocks, n, ncand, ora, var)
    om = oracle.match(fixed, moving, ora["centres"], cfg.block, cfg.window)
    dims = fixed.shape[::-1]
    for opts, kernel in ((dict(), 2), (dict(force_rows=1), 1), (dict(force_generic=1), 0)):
        for k, v in opts.items():
            _emul.set_option(k, v)
        assert _emul.match_info(dims, cfg.block, cfg.window)["kernel"] == kernel
        disp, ncc = _emul.match(fixed, moving, blocks, cfg.block, cfg.window)
        assert_match_parity(disp, ncc, om, "tiny kernel %d" % kernel)
        for k in opts:
            _emul.set_option(k, 0)


def _grid_blocks(dims, block, stride):
    """Every stride-grid block, borders included (their windows leave the volume: skip rule)."""
    axes = [np.arange(0, dims[a] - block[a] + 1, stride[a]) + (block[a] - 1) // 2 for a in range(3)]
    zz, yy, xx = np.meshgrid(axes[2], axes[1], axes[0], indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1).astype(np.int32)


@pytest.mark.parametrize("dims,b,r,rz,stride,g", [
    ((28, 26, 22), 5, 3, 3, (7, 7, 8), 0),        # W = 7: 3 pairs + the odd plane
    ((32, 30, 26), 7, 5, 5, (9, 11, 9), 0),       # the config-3 shape (block 7, window 5); planner's G
    ((32, 30, 26), 7, 5, 5, (9, 11, 9), 3),       # a group size that leaves a partial last CTA
    ((32, 30, 24), 7, 5, 3, (12, 11, 8), 0),      # the config-2 shape: anisotropic window (5,5,3)
    ((36, 34, 30), 9, 7, 7, (13, 12, 10), 0),     # the config-4 shape
    ((28, 28, 24), 5, 5, 0, (11, 11, 9), 0),      # rz = 0: only the y-pair warps of the last (only) candidate plane work
    ((32, 30, 30), 11, 3, 3, (10, 9, 9), 0),
    ((29, 27, 25), 5, 3, 3, (6, 7, 8), 0),        # nx not a multiple of 4: TMA cannot address it, plain staging
    ((32, 30, 20), (7, 3), 5, 2, (9, 11, 5), 0),  # thick-slice block 7 x 7 x 3
    ((28, 28, 24), (5, 9), 3, 3, (8, 8, 5), 0),   # block 5 x 5 x 9
    ((28, 28, 12), (5, 1), 3, 1, (8, 8, 3), 0),   # a single plane: no pair-table planes at all
])
def test_emulated_pair_kernel_matches_the_oracle(dims, b, r, rz, stride, g):
    b, bz = b if isinstance(b, tuple) else (b, b)
    fixed = _smooth(dims, 7 + b + r)
    moving = _shift_noise(fixed, (1, -2, 1), 8.0, 11)
    block, window = (b, b, bz), (r, r, rz)
    blocks = _grid_blocks(dims, block, stride)
    _emul.set_option("pair_blocks_per_cta", g)
    assert _emul.match_info(dims, block, window)["kernel"] == 2
    om = oracle.match(fixed, moving, blocks, block, window)
    disp, ncc = _emul.match(fixed, moving, blocks, block, window)
    assert_match_parity(disp, ncc, om, "pair %s" % (dims,))
    _emul.set_option("disable_tma", 1)                     # plain-load staging must not change a bit
    assert _emul.match_info(dims, block, window)["kernel"] == 2
    disp2, ncc2 = _emul.match(fixed, moving, blocks, block, window)
    _emul.set_option("disable_tma", 0)
    assert np.array_equal(disp, disp2) and np.array_equal(ncc, ncc2)
    _emul.set_option("force_rows", 1)                      # the one-row-per-thread kernel on the same input
    disp, ncc = _emul.match(fixed, moving, blocks, block, window)
    assert_match_parity(disp, ncc, om, "rows %s" % (dims,))


def test_emulated_degenerate_inputs():
    """Constant regions (zero variance: NCC := 0, lowest index wins), exact ties, blocks that leave the volume."""
    dims = (24, 24, 20)
    fixed = _smooth(dims, 3)
    fixed[:, :, :12] = 500.0                               # constant half: zero-variance fixed blocks and candidates
    moving = fixed.copy()
    moving[10:, :, :] = _shift_noise(fixed, (1, 0, 0), 5.0, 5)[10:, :, :]
    block, window = (5, 5, 5), (3, 3, 3)
    blocks = _grid_blocks(dims, block, (6, 6, 5))
    om = oracle.match(fixed, moving, blocks, block, window)
    for opts in (dict(), dict(force_rows=1), dict(force_generic=1)):
        for k, v in opts.items():
            _emul.set_option(k, v)
        disp, ncc = _emul.match(fixed, moving, blocks, block, window)
        assert_match_parity(disp, ncc, om, "degenerate %s" % (opts,))
        for k in opts:
            _emul.set_option(k, 0)
    bad = blocks.copy()
    bad[1] = (1, 2, 2)                                     # origin (-1, 0, 0): leaves the volume
    with pytest.raises(RuntimeError, match="leaves the volume"):
        _emul.match(fixed, moving, bad, block, window)


@pytest.mark.parametrize("dims,block,generic", [
    ((70, 45, 33), (7, 7, 7), 0),        # sliding kernel: two x tiles, ragged y and z, several z chunks
    ((70, 45, 33), (7, 7, 7), 1),        # generic kernel on the same input
    ((33, 29, 40), (5, 5, 5), 0),
    ((40, 38, 30), (9, 9, 9), 0),
    ((36, 30, 28), (11, 11, 11), 0),
    ((30, 22, 21), (3, 5, 7), 0),        # not square in-plane: generic kernel
    ((33, 29, 40), (7, 7, 3), 0),        # square in-plane, thin along z: sliding kernel with bz = 3
])
def test_emulated_moving_stats(dims, block, generic):
    """inv_sd[p] = 1/sqrt(SS of the moving block with origin p) against a plain numpy fp64 evaluation."""
    vol = _smooth(dims, 21)
    vol[:6, :8, :9] = 321.0                                 # a constant corner: SS = 0 -> inv_sd = 0
    _emul.set_option("boxstat_generic", generic)
    got = _emul.moving_stats(vol, block)
    _emul.set_option("boxstat_generic", 0)
    nz, ny, nx = vol.shape
    bx, by, bz = block
    v = vol.astype(np.float64)
    win = np.lib.stride_tricks.sliding_window_view(v, (bz, by, bx))
    ss = ((win - win.mean(axis=(3, 4, 5), keepdims=True)) ** 2).sum(axis=(3, 4, 5))
    want = np.where(ss > 1e-9, 1.0 / np.sqrt(np.maximum(ss, 1e-300)), 0.0)
    valid = got[: nz - bz + 1, : ny - by + 1, : nx - bx + 1]
    assert np.all(valid[ss <= 1e-9] == 0.0)
    rel = np.abs(valid - want)[ss > 1e-9] * np.sqrt(ss[ss > 1e-9])
    assert rel.max() < 1e-6, rel.max()
    untouched = np.ones(vol.shape, bool)
    untouched[: nz - bz + 1, : ny - by + 1, : nx - bx + 1] = False
    assert np.all(got[untouched] == -7.0)                   # origins whose block leaves the volume are not written


def test_emulated_register_needs_no_host_side_count():
    """nrr_bm_register: the matching kernels are launched for an upper bound on K and read K on the device
    (masked case: N < grid positions, so whole CTAs find nothing to do)."""
    dims, block, stride, window = (36, 32, 28), (5, 5, 5), (4, 4, 4), (3, 3, 3)
    fixed = _smooth(dims, 77)
    moving = _shift_noise(fixed, (-1, 2, 1), 6.0, 78)
    mask = spherical_mask(dims, 11.0)
    ora_sel = oracle.select(fixed, block, stride, 0.5, mask)
    ora = oracle.match(fixed, moving, ora_sel["centres"], block, window)
    assert 0 < len(ora_sel["centres"]) < 0.2 * 8 * 7 * 6             # far fewer than the host-side bound
    for opts in (dict(), dict(force_rows=1), dict(force_generic=1)):
        for k, v in opts.items():
            _emul.set_option(k, v)
        blocks, disp, ncc = _emul.register(fixed, moving, block, stride, window, 0.5, mask)
        assert np.array_equal(blocks, ora_sel["centres"])
        assert_match_parity(disp, ncc, ora, "register %s" % (opts,))
        for k in opts:
            _emul.set_option(k, 0)


@pytest.mark.parametrize("b,r,rz", [(7, 5, 5), (5, 3, 3), (7, 5, 3)])
def test_emulated_pair_kernel_every_candidate_row_can_win(b, r, rz):
    """Plants, for block i, an exact copy of the fixed block at displacement d_i in a noise volume, with the d_i
    running over EVERY (dy, dz) candidate row and every dx: a candidate row missing from the lane -> task table,
    or a wrong index in the epilogue, loses its block."""
    from nrr_inputs.planted import planted_pair
    fixed, moving, centres, want = planted_pair(b, r, rz)
    block, window = (b, b, b), (r, r, rz)
    assert _emul.match_info(fixed.shape[::-1], block, window)["kernel"] == 2
    disp, ncc = _emul.match(fixed, moving, centres, block, window)
    assert np.array_equal(disp, want)
    assert np.all(np.abs(ncc - 1.0) < 1e-5)
    om = oracle.match(fixed, moving, centres, block, window)
    assert_match_parity(disp, ncc, om, "planted displacements")


@pytest.mark.parametrize("conn", [6, 18, 26])
@pytest.mark.parametrize("dims,block,stride,frac,mask_r,generic", [
    ((24, 22, 20), (3, 3, 3), (1, 1, 1), 0.10, None, 0),        # the paper's setting: every voxel a candidate
    ((24, 22, 20), (3, 3, 3), (1, 1, 1), 0.90, 8.0, 0),         # K above what the pattern leaves: the whole set
    ((30, 28, 26), (5, 5, 5), (2, 1, 3), 0.30, 11.0, 1),        # anisotropic grid, multi-launch radix select
])
def test_emulated_pruned_selection_matches_the_oracle(conn, dims, block, stride, frac, mask_r, generic):
    """PAPER.md:376 connectivity patterns (reading Q20): the parallel fixed-point rounds against the oracle's
    sequential greedy walk, bit-exact set, order and variances."""
    vol = _smooth(dims, 300 + conn)
    vol[:5] = np.round(vol[:5] / 100.0) * 100.0                  # exact variance ties: the index rule decides
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    ora = oracle.select_pruned(vol, block, stride, frac, mask, conn)
    _emul.set_option("select_generic", generic)
    blocks, n, ncand, var = _emul.select_pruned(vol, block, stride, frac, mask, conn)
    _emul.set_option("select_generic", 0)
    assert_select_parity(blocks, n, ncand, ora, var)


def test_emulated_pruned_selection_uniform_image_closed_form():
    vol = np.full((9, 9, 9), 5.0, np.float32)
    blocks, n, ncand, var = _emul.select_pruned(vol, (3, 3, 3), (1, 1, 1), 1.0, None, 6)
    want = [[i + 1, j + 1, k + 1] for k in range(7) for j in range(7) for i in range(7) if (i + j + k) % 2 == 0]
    assert ncand == 343 and blocks.tolist() == want
    blocks, n, ncand, var = _emul.select_pruned(vol, (3, 3, 3), (1, 1, 1), 1.0, None, 0)
    assert n == 343                                              # no pattern: plain selection


def _warp_case(dims, amp, seed):
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    img = rng.uniform(0, 1000, (nz, ny, nx)).astype(np.float32)
    field = rng.uniform(-amp, amp, (3, nz, ny, nx)).astype(np.float32)
    field[:, 0, 0, :4] = [[-1e9, 1e9, 0.0, 2.0]] * 3             # far outside, integers: clamping / exact copies
    return img, field


@pytest.mark.parametrize("dims,amp", [((37, 21, 9), 2.5), ((16, 16, 16), 40.0), ((300, 3, 2), 1.0)])
def test_emulated_warp_matches_the_oracle(dims, amp):
    """|gpu - oracle| <= 8 * 2^-24 * max|image| (three fp32 interpolations, tolerances)."""
    img, field = _warp_case(dims, amp, 90 + dims[0])
    got, want = _emul.warp(img, field), oracle.warp(img, field)
    assert np.max(np.abs(got.astype(np.float64) - want)) <= 8 * 2.0 ** -24 * 1000.0
    zero = np.zeros_like(field)
    assert np.array_equal(_emul.warp(img, zero), img)              # identity is exact


def test_emulated_staging_timeout_is_an_error_code_not_a_fault():
    """A mis-programmed staging barrier (here: 16 bytes more expected than the copies deliver) must end as
    NRR_E_DEVICE with NaN results -- the kernels' bounded wait gives up, every thread of the CTA leaves in an
    orderly way, nothing traps (a device trap is an Xid on a shared GPU box)."""
    dims, block, window = (40, 36, 24), (5, 5, 5), (3, 3, 3)
    vol = _smooth(dims, 77)
    mov = _shift_noise(vol, (1, 0, -1), 10.0, 78)
    sel = oracle.select(vol, block, block, 0.5)
    assert _emul.match_info(dims, block, window)["kernel"] == 2 and _emul.match_info(dims, block, window)["tma"] == 1
    good_d, good_n = _emul.match(vol, mov, sel["centres"], block, window)
    _emul.set_option("debug_expect_tx_extra", 16)
    with pytest.raises(RuntimeError, match="status -12"):
        _emul.match(vol, mov, sel["centres"], block, window)
    _emul.set_option("debug_expect_tx_extra", 0)
    d, n = _emul.match(vol, mov, sel["centres"], block, window)      # the flag was cleared; the library still works
    assert np.array_equal(d, good_d) and np.array_equal(n, good_n)


# ------------------------------------------------------------------------------------------- plans, batch
@pytest.mark.parametrize("dims,block,stride,window,frac,mask_r", [
    ((48, 40, 30), (7, 7, 7), (5, 5, 5), (5, 5, 3), 0.5, 18.0),      # pair kernel, TMA staging, records kept by the plan
    ((41, 37, 29), (5, 5, 5), (4, 4, 4), (3, 3, 3), 0.3, None),      # nx % 4 != 0: plain staging
    ((24, 20, 16), (3, 5, 3), (4, 4, 4), (1, 1, 2), 0.5, None),      # generic kernel: no records
])
def test_emulated_plan_equals_select_then_match(dims, block, stride, window, frac, mask_r):
    """pre-operative plan (selection + fixed-block records), intra-operative match.  Bit-equal to
    nrr_bm_select_blocks + nrr_bm_match; the host form's slab pipeline and block ranges must not change a bit."""
    fixed = _smooth(dims, 500 + dims[0])
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    blocks, n, ncand, var = _emul.select(fixed, block, stride, frac, mask)
    assert n > 8
    for host in (True, False):
        plan = _emul.Plan(fixed, block, stride, window, frac, mask, host=host)
        pb, pv = plan.blocks()
        assert plan.n == n and plan.ncand == ncand and np.array_equal(pb, blocks) and np.array_equal(pv, var)
        for k, shift in enumerate(((1, -1, 1), (-2, 0, 1))):          # one plan, several intra-operative volumes
            moving = _shift_noise(fixed, shift, 12.0, 600 + k)
            want_d, want_n = _emul.match(fixed, moving, blocks, block, window)
            d, s = plan.match(moving)
            assert np.array_equal(d, want_d) and np.array_equal(s, want_n)
            for slabs in (1, 3, 1000):
                _emul.set_option("plan_slabs", slabs)
                d, s = plan.match_host(moving)
                assert np.array_equal(d, want_d) and np.array_equal(s, want_n), slabs
            _emul.set_option("plan_slabs", 4)
            # the natural shard: ranks match slices of the block list; stitched = whole
            out = (np.full((n, 3), -99, np.int32), np.full((n,), -99.0, np.float32))
            cuts = [0, n // 3, n // 3, n - 1, n]
            for a, b in zip(cuts[:-1], cuts[1:]):
                plan.match(moving, a, b - a, out=out)
            assert np.array_equal(out[0], want_d) and np.array_equal(out[1], want_n)
            part = plan.match(moving, 2, 3)
            assert np.all(part[0][:2] == -99) and np.all(part[0][5:] == -99) and np.array_equal(part[0][2:5], want_d[2:5])
        with pytest.raises(RuntimeError, match="status -11"):
            plan.match(moving, n - 1, 2)
        plan.destroy()


def test_emulated_plan_with_connectivity_pattern_and_oracle():
    dims, block, stride, window = (40, 36, 24), (5, 5, 5), (2, 2, 2), (3, 3, 3)
    fixed = _smooth(dims, 91)
    moving = _shift_noise(fixed, (1, 1, -1), 8.0, 92)
    ora_sel = oracle.select_pruned(fixed, block, stride, 0.2, None, 18)
    plan = _emul.Plan(fixed, block, stride, window, 0.2, None, connectivity=18)
    pb, pv = plan.blocks()
    assert_select_parity(pb, plan.n, plan.ncand, ora_sel, pv)
    d, s = plan.match_host(moving)
    assert_match_parity(d, s, oracle.match(fixed, moving, ora_sel["centres"], block, window), "plan, 18-connectivity")
    plan.destroy()


def test_emulated_batch_equals_separate_register_calls():
    """PAPER.md:527-540 / BASELINE.json configs[4]: many settings on one pair in one launch sequence; shared
    normalisers, shared variance keys (two fractions from one statistics pass), shared records."""
    dims = (44, 40, 36)
    fixed = _smooth(dims, 71)
    moving = _shift_noise(fixed, (1, -2, 1), 9.0, 72)
    mask = spherical_mask(dims, 17.0)
    settings = []
    for b in (5, 7):
        for r in (3, 5):
            for frac in (0.1, 0.3):
                settings.append(((b, b, b), (5, 5, 5), (r, r, r), frac))
    settings.append(((3, 5, 3), (4, 4, 4), (1, 2, 1), 0.5))          # a shape only the generic kernel takes
    settings.append(((7, 7, 7), (5, 5, 5), (4, 4, 4), 0.3))          # no fast instantiation: no records, shared selection
    L = _emul.lib()
    L.nrr_bm_launch_count.restype = ctypes.c_longlong
    L.nrr_bm_launch_count(1)
    got, out_n = _emul.register_batch(fixed, moving, settings, mask)
    batch_launches = L.nrr_bm_launch_count(1)
    assert len(got) == len(settings)
    for (block, stride, window, frac), (gb, gd, gs), k in zip(settings, got, out_n):
        wb, wd, ws = _emul.register(fixed, moving, block, stride, window, frac, mask)
        assert k == len(wb) and np.array_equal(gb, wb), (block, window, frac)
        assert np.array_equal(gd, wd) and np.array_equal(gs, ws), (block, window, frac)
    separate_launches = L.nrr_bm_launch_count(1)
    # 10 settings: 3 moving-statistics passes instead of 10, 3 variance passes instead of 10, 5 record sets instead of 8
    assert batch_launches <= separate_launches - 7 - 7 - 3, (batch_launches, separate_launches)
    ora_sel = oracle.select(fixed, (7, 7, 7), (5, 5, 5), 0.3, mask)
    assert np.array_equal(got[7][0], ora_sel["centres"])
    assert_match_parity(got[7][1], got[7][2], oracle.match(fixed, moving, ora_sel["centres"], (7, 7, 7), (5, 5, 5)), "batch")


def test_capacity_bound_is_the_count_rule():
    for dims, block, stride, frac in (((64, 64, 32), (5, 5, 5), (5, 5, 5), 0.3), ((256, 256, 124), (7, 7, 7), (5, 5, 5), 0.25),
                                      ((9, 9, 9), (9, 9, 9), (1, 1, 1), 1.0), ((30, 20, 10), (3, 5, 7), (2, 3, 1), 0.05)):
        ngrid, bound = _emul.capacity_bound(dims, block, stride, frac)
        assert ngrid == int(np.prod(oracle.grid(dims, block, stride)))
        for n in (ngrid, ngrid // 2, 1, 0):
            assert bound >= oracle.count(n, frac)
        assert bound <= min(ngrid, oracle.count(ngrid, frac) + 1)
