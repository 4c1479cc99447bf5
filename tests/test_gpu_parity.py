"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle, element by
element on the same seeded inputs.  Sizes span several tiles and ragged tails; the BASELINE.json configs run
at full size (config 4 and the 32-setting batch on sampled blocks the oracle computes one by one).

ORDER.  The driver runs this file with -x, so the first failure hides everything behind it.  The tests are therefore
ordered by subsystem, from what depends on least to what depends on most: selection, moving statistics, warp, FEM,
pruned selection, then the matching kernels one family at a time (generic -> one row per thread -> two rows per
thread; plain-load staging before TMA / bulk-copy staging), then the whole-call forms (host, register, plans, batch)
at the BASELINE.json sizes, and last the test that makes a staging barrier time out on purpose."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle                                    # noqa: E402  (test infrastructure)
import paper_2308_10868_b200 as nrr             # noqa: E402  (product)
from nrr_inputs import CONFIGS, batch_settings, make_pair, spherical_mask   # noqa: E402
from _parity import assert_match_parity, assert_select_parity               # noqa: E402


def _cuda(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


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
    m = vol[np.ix_(iz, iy, ix)].astype(np.float64)
    m = m + np.random.default_rng(seed).normal(0, noise, size=m.shape)
    return np.ascontiguousarray(m, dtype=np.float32)


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    nrr.lib()      # fails loudly if libnrr_bm.so is missing: there is no fallback
    yield


_pairs = {}


def assert_ncc_of_chosen_displacement(fixed, moving, blocks, block, disp, ncc, label=""):
    """Whole-set check where the full oracle search is too slow: for EVERY block the reported NCC must be the oracle's
    NCC of the reported displacement (one candidate per block), within the north_star tolerance."""
    worst = 0.0
    for c, d, s in zip(blocks, disp, ncc):
        want = oracle.ncc_at(fixed, moving, c, block, d)
        assert np.isfinite(want), "%s: block %s chose a skipped candidate %s" % (label, c, d)
        worst = max(worst, abs(float(s) - want))
    assert worst <= 1e-4, "%s: max |gpu_ncc - oracle.ncc_at(gpu_disp)| = %g" % (label, worst)
    return worst


def pair(name):
    if name not in _pairs:
        _pairs[name] = make_pair(CONFIGS[name])
    return _pairs[name]


def _with_options(opts, fn):
    for k, v in opts.items():
        nrr.nrr_bm_set_option(k, v)
    try:
        return fn()
    finally:
        for k in opts:
            nrr.nrr_bm_set_option(k, 0)


def _match_case(dims, block, window, shift, noise, seed, stride=None, frac=1.0, expect_fast=None):
    vol = _smooth(dims, seed)
    mov = _shift_noise(vol, shift, noise, seed + 1)
    sel = oracle.select(vol, block, stride or block, frac)
    ora = oracle.match(vol, mov, sel["centres"], block, window)
    info = nrr.nrr_bm_match_info(dims, block, window)
    if expect_fast is not None:
        assert info["fast"] == expect_fast, info
    disp, ncc = nrr.nrr_bm_match(_cuda(vol), _cuda(mov), _cuda(sel["centres"]), block, window)
    nrr.nrr_bm_check_async_error()
    return assert_match_parity(disp.cpu().numpy(), ncc.cpu().numpy(), ora, label=str((dims, block, window))), len(sel["centres"])


# ------------------------------------------------------------------------------------------- selection (S1-S3)
@pytest.mark.parametrize("dims,block,stride,frac,mask_r", [
    ((41, 37, 29), (5, 5, 5), (5, 5, 5), 0.30, None),
    ((41, 37, 29), (7, 7, 7), (5, 5, 5), 0.25, 15.0),
    ((41, 37, 29), (3, 5, 7), (4, 3, 2), 0.50, 15.0),
    ((41, 37, 29), (9, 9, 9), (6, 6, 6), 1.00, None),
    ((64, 50, 33), (5, 5, 5), (1, 1, 1), 0.05, 20.0),       # dense grid: many chunks, ragged tail
    ((130, 3, 3), (3, 3, 3), (1, 1, 1), 0.10, None),         # degenerate thin volume
    ((9, 9, 9), (9, 9, 9), (1, 1, 1), 1.00, None),           # a single candidate
])
@pytest.mark.parametrize("generic", [1, 0], ids=["round1_kernels", "default_kernels"])
def test_select_parity_small(generic, dims, block, stride, frac, mask_r):
    """generic = 1: the runtime-shaped statistics kernel and the multi-launch radix select that ran on hardware in
    round 1 (first, so that a failure of the default kernels is told apart from a failure of the method)."""
    vol = _smooth(dims, 100 + dims[0])
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    ora = oracle.select(vol, block, stride, frac, mask)
    blocks, n, ncand, var = _with_options({"select_generic": generic}, lambda: nrr.nrr_bm_select_blocks(
        _cuda(vol), block, stride, frac, _cuda(mask), want_var=True))
    assert_select_parity(blocks.cpu().numpy(), n, ncand, ora, var.cpu().numpy())


def test_select_uniform_image_and_exact_ties():
    vol = np.full((12, 15, 20), 42.0, dtype=np.float32)
    ora = oracle.select(vol, (3, 3, 3), (3, 3, 3), 0.25)
    blocks, n, ncand, var = nrr.nrr_bm_select_blocks(_cuda(vol), (3, 3, 3), (3, 3, 3), 0.25, want_var=True)
    assert_select_parity(blocks.cpu().numpy(), n, ncand, ora, var.cpu().numpy())
    vol2 = np.zeros((6, 6, 18), dtype=np.float32)
    pat = np.arange(27, dtype=np.float32).reshape(3, 3, 3)
    vol2[0:3, 0:3, 3:6] = pat
    vol2[3:6, 3:6, 12:15] = pat
    for frac in (1.0 / 24.0, 2.0 / 24.0, 3.0 / 24.0):
        ora = oracle.select(vol2, (3, 3, 3), (3, 3, 3), frac)
        blocks, n, ncand = nrr.nrr_bm_select_blocks(_cuda(vol2), (3, 3, 3), (3, 3, 3), frac)
        assert_select_parity(blocks.cpu().numpy(), n, ncand, ora)


def test_select_mask_excluding_everything_and_capacity_error():
    vol = _smooth((20, 20, 20), 7)
    mask = np.zeros_like(vol, dtype=np.uint8)
    blocks, n, ncand = nrr.nrr_bm_select_blocks(_cuda(vol), (5, 5, 5), (5, 5, 5), 0.5, _cuda(mask))
    assert n == 0 and ncand == 0 and blocks.shape[0] == 0
    with pytest.raises(nrr.NrrError) as ei:
        nrr.nrr_bm_select_blocks(_cuda(vol), (5, 5, 5), (5, 5, 5), 0.5, capacity=3)
    assert ei.value.status == -7


def test_select_generic_path_equals_default():
    cfg = CONFIGS["intraop"]
    fixed, _, mask = pair("intraop")
    ora = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    for generic in (0, 1):
        blocks, n, ncand, var = _with_options({"select_generic": generic}, lambda: nrr.nrr_bm_select_blocks(
            _cuda(fixed), cfg.block, cfg.stride, cfg.frac, _cuda(mask), want_var=True))
        assert_select_parity(blocks.cpu().numpy(), n, ncand, ora, var.cpu().numpy())


@pytest.mark.parametrize("name", ["tiny", "intraop", "fullres", "highres"])
def test_select_parity_configs(name):
    cfg = CONFIGS[name]
    fixed, _, mask = pair(name)
    ora = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    blocks, n, ncand, var = nrr.nrr_bm_select_blocks(_cuda(fixed), cfg.block, cfg.stride, cfg.frac, _cuda(mask), want_var=True)
    assert_select_parity(blocks.cpu().numpy(), n, ncand, ora, var.cpu().numpy())
    print("%s: N=%d K=%d oracle K/K+1 variance margin %.3g" % (name, ncand, n, ora["margin"]))


# ------------------------------------------------------------------------------------------- moving-volume statistics (M2)
@pytest.mark.parametrize("generic", [1, 0], ids=["round1_kernel", "sliding_kernel"])
def test_moving_stats_against_numpy(generic):
    dims, block = (70, 45, 33), (7, 7, 7)
    vol = _smooth(dims, 21)
    vol[:6, :8, :9] = 321.0                                  # a constant corner: SS = 0 -> inv_sd = 0
    v = vol.astype(np.float64)
    win = np.lib.stride_tricks.sliding_window_view(v, block[::-1])
    ss = ((win - win.mean(axis=(3, 4, 5), keepdims=True)) ** 2).sum(axis=(3, 4, 5))
    want = np.where(ss > 1e-9, 1.0 / np.sqrt(np.maximum(ss, 1e-300)), 0.0)
    out = torch.full(vol.shape, -7.0, dtype=torch.float32, device="cuda")
    got = _with_options({"boxstat_generic": generic}, lambda: nrr.nrr_bm_moving_stats(_cuda(vol), block, out)).cpu().numpy()
    valid = got[: ss.shape[0], : ss.shape[1], : ss.shape[2]]
    assert np.all(valid[ss <= 1e-9] == 0.0)
    rel = np.abs(valid - want)[ss > 1e-9] * np.sqrt(ss[ss > 1e-9])
    assert rel.max() < 2e-6, rel.max()
    untouched = np.ones(vol.shape, bool)
    untouched[: ss.shape[0], : ss.shape[1], : ss.shape[2]] = False
    assert np.all(got[untouched] == -7.0)


# ------------------------------------------------------------------------------------------- dense-field warp
@pytest.mark.parametrize("dims,amp", [((37, 21, 9), 2.5), ((64, 60, 33), 40.0), ((256, 256, 124), 8.0)])
def test_warp_parity(dims, amp):
    """out(p) = trilinear(image, clamp(p + v(p))) (reading Q21): |gpu - oracle| <= 8 * 2^-24 * max|image|."""
    rng = np.random.default_rng(90 + dims[0])
    nx, ny, nz = dims
    img = rng.uniform(0, 1000, (nz, ny, nx)).astype(np.float32)
    field = rng.uniform(-amp, amp, (3, nz, ny, nx)).astype(np.float32)
    field[:, 0, 0, :4] = [[-1e9, 1e9, 0.0, 2.0]] * 3
    got = nrr.nrr_bm_warp(_cuda(img), _cuda(field)).cpu().numpy()
    want = oracle.warp(img, field)
    assert np.max(np.abs(got.astype(np.float64) - want)) <= 8 * 2.0 ** -24 * 1000.0
    assert torch.equal(nrr.nrr_bm_warp(_cuda(img), torch.zeros_like(_cuda(field))), _cuda(img))


# ------------------------------------------------------------------------------------------- FEM regularisation
@pytest.mark.parametrize("dims,spacing,young,poisson,weight,n_iter", [
    ((13, 9, 11), (4, 2, 5), 3.0, 0.30, 1.0, 1),
    ((40, 36, 24), (6, 6, 6), 1.0, 0.45, 0.5, 3),
    ((64, 64, 32), (8, 8, 8), 2.0, 0.40, 2.0, 2),
])
def test_fem_solve_parity(dims, spacing, young, poisson, weight, n_iter):
    """F_i = K U_i, U_{i+1} = [K + H^T S H]^-1 [H^T S D + F_i] on the Kuhn grid mesh (Q22-Q25): the
    CUDA path (stencil K, FP64 scatter, PCG) against the oracle's assembled sparse matrices and direct solves."""
    from oracle import fem as ofem
    rng = np.random.default_rng(dims[0])
    msh = ofem.mesh(dims, spacing)
    inside = msh["xyz"][np.all(msh["xyz"] < np.asarray(dims), axis=1)]
    blocks = np.vstack([inside, np.floor(rng.uniform(0, np.asarray(dims) - 1e-9, (400, 3)))]).astype(np.int32)
    disp = rng.integers(-4, 5, blocks.shape).astype(np.int32)
    ncc = rng.uniform(-0.2, 1.0, len(blocks)).astype(np.float32)
    ncc[::13] = np.nan
    want = ofem.solve(msh, young, poisson, blocks, disp, ncc, weight, n_iter)["U"]
    fem = nrr.nrr_bm_fem_create(dims, spacing, young, poisson)
    assert fem.nodes == msh["nodes_shape"]
    u, iters = nrr.nrr_bm_fem_solve(fem, _cuda(blocks), _cuda(disp), _cuda(ncc), weight, n_iter, tol=1e-12)
    got = u.cpu().numpy()
    err = np.max(np.abs(got - want))
    print("fem %s: %d nodes, %d CG iterations, max |U - oracle| %.3g" % (dims, fem.n_nodes, iters, err))
    assert err <= 1e-6 * max(1.0, np.max(np.abs(want)))
    field = nrr.nrr_bm_fem_dense_field(fem, u).cpu().numpy()
    if np.prod(dims) <= 20000:
        ref = ofem.dense_field(msh, got, dims)
        assert np.max(np.abs(field - ref)) <= 2e-6 * max(1.0, np.max(np.abs(ref)))
    hu, hiters = nrr.nrr_bm_fem_solve_host(fem, blocks, disp, ncc, weight, n_iter, tol=1e-12)
    assert np.max(np.abs(hu - got)) <= 1e-9 * max(1.0, np.max(np.abs(got)))      # FP64 atomics: order may differ
    nrr.nrr_bm_fem_destroy(fem)


# ------------------------------------------------------------------------------------------- connectivity pruning
@pytest.mark.parametrize("conn", [6, 18, 26])
@pytest.mark.parametrize("dims,block,stride,frac,mask_r", [
    ((48, 44, 40), (3, 3, 3), (1, 1, 1), 0.05, None),          # the paper's setting: every voxel a candidate
    ((48, 44, 40), (5, 5, 5), (1, 1, 1), 0.90, 17.0),          # K above what the pattern leaves: the whole set
    ((64, 60, 33), (5, 5, 5), (2, 1, 3), 0.30, 20.0),
])
def test_pruned_selection_parity(conn, dims, block, stride, frac, mask_r):
    """PAPER.md:376 connectivity patterns (reading Q20): parallel fixed-point rounds vs the oracle's greedy walk."""
    vol = _smooth(dims, 300 + conn)
    vol[:5] = np.round(vol[:5] / 100.0) * 100.0                 # exact variance ties: the index rule decides
    mask = None if mask_r is None else spherical_mask(dims, mask_r)
    ora = oracle.select_pruned(vol, block, stride, frac, mask, conn)
    blocks, n, ncand, var = nrr.nrr_bm_select_blocks_pruned(_cuda(vol), block, stride, frac, _cuda(mask), conn, want_var=True)
    assert_select_parity(blocks.cpu().numpy(), n, ncand, ora, var.cpu().numpy())


def test_pruned_selection_dense_grid_multi_launch_path():
    """More than 2^20 grid positions: the multi-launch radix select after the pruning rounds."""
    dims = (128, 112, 80)
    vol = _smooth(dims, 55, sigma=2.0)
    ora = oracle.select_pruned(vol, (3, 3, 3), (1, 1, 1), 0.04, None, 6)
    blocks, n, ncand = nrr.nrr_bm_select_blocks_pruned(_cuda(vol), (3, 3, 3), (1, 1, 1), 0.04, None, 6)
    assert ncand > (1 << 20)
    assert_select_parity(blocks.cpu().numpy(), n, ncand, ora)


# ------------------------------------------------------------------------------------------- matching kernels (M1, M3-M5)
_FAMILIES = [      # (label, options, kernel id reported by nrr_bm_match_info under these options)
    ("generic", {"force_generic": 1}),
    ("rows, plain staging", {"force_rows": 1, "disable_tma": 1}),
    ("rows, TMA", {"force_rows": 1}),
    ("pair, plain staging", {"disable_tma": 1}),
    ("pair, TMA + bulk copy", {}),                      # the default path
    ("pair, G=3", {"pair_blocks_per_cta": 3}),           # another grouping, partial last CTA
]
_family_results = {}


@pytest.mark.parametrize("label,opts", _FAMILIES, ids=[f[0].replace(" ", "_").replace(",", "") for f in _FAMILIES])
def test_match_kernel_families_on_the_same_input(label, opts):
    """Every matching kernel and staging path against the oracle on one input, the simplest machinery first: the
    generic kernel, the one-row-per-thread kernel, the pair kernel; plain loads before TMA / bulk copies.  The staging
    path and the grouping of blocks into CTAs must not change a bit."""
    dims, block, window = (48, 44, 40), (7, 7, 7), (5, 5, 5)
    vol = _smooth(dims, 31)
    mov = _shift_noise(vol, (2, 1, -2), 25.0, 32)
    sel = oracle.select(vol, block, (5, 5, 5), 0.5)
    assert nrr.nrr_bm_match_info(dims, block, window)["kernel"] == 2
    d, s = _with_options(opts, lambda: nrr.nrr_bm_match(_cuda(vol), _cuda(mov), _cuda(sel["centres"]), block, window))
    nrr.nrr_bm_check_async_error()
    ora = oracle.match(vol, mov, sel["centres"], block, window)
    assert_match_parity(d.cpu().numpy(), s.cpu().numpy(), ora, label=label)
    _family_results[label] = (d, s)
    for a, b in (("rows, plain staging", "rows, TMA"), ("pair, plain staging", "pair, TMA + bulk copy"),
                 ("pair, TMA + bulk copy", "pair, G=3")):
        if label == b and a in _family_results:
            assert torch.equal(_family_results[a][0], d) and torch.equal(_family_results[a][1], s), (a, b)


@pytest.mark.parametrize("dims,block,window,fast", [
    ((40, 36, 24), (5, 5, 5), (3, 3, 3), True),      # nx % 4 == 0: TMA staging; every grid block incl. borders
    ((41, 37, 29), (5, 5, 5), (3, 3, 3), True),      # nx % 4 != 0: plain-load staging
    ((48, 40, 30), (7, 7, 7), (5, 5, 3), True),      # config-2 shape of window
    ((45, 43, 31), (7, 7, 7), (5, 5, 5), True),
    ((44, 40, 36), (9, 9, 9), (3, 3, 2), True),
    ((40, 40, 40), (11, 11, 11), (3, 3, 3), True),
    ((36, 32, 28), (5, 5, 5), (7, 7, 1), True),
    ((40, 36, 24), (3, 5, 3), (2, 1, 3), False),     # not square in-plane: generic kernel
    ((48, 44, 24), (7, 7, 3), (5, 5, 2), True),      # thick-slice block: pair kernel with a run-time z extent
    ((33, 31, 29), (7, 7, 7), (4, 4, 4), False),     # window without a fast instantiation
    ((30, 30, 30), (5, 5, 5), (0, 0, 0), False),     # single candidate
])
def test_match_parity_small(dims, block, window, fast):
    exempt, n = _match_case(dims, block, window, (1, -1, 1), 20.0, 200 + dims[0], expect_fast=fast)
    print("%s %s %s: %d blocks, %d exempt" % (dims, block, window, n, exempt))


def test_match_exact_ties_and_constant_regions():
    # period-2 volume along x: dx = -2, 0, +2 are bit-identical candidates -> lowest linear index wins
    base = np.random.default_rng(15).uniform(0, 1000, size=(9, 9, 2)).astype(np.float32)
    vol = np.ascontiguousarray(np.tile(base, (1, 1, 8)))
    centres = np.asarray([[8, 4, 4], [6, 4, 4]], dtype=np.int32)
    ora = oracle.match(vol, vol, centres, (3, 3, 3), (2, 0, 0))
    disp, ncc = nrr.nrr_bm_match(_cuda(vol), _cuda(vol), _cuda(centres), (3, 3, 3), (2, 0, 0))
    assert disp.cpu().numpy().tolist() == ora["disp"].tolist() == [[-2, 0, 0], [-2, 0, 0]]
    np.testing.assert_allclose(ncc.cpu().numpy(), ora["ncc"], atol=1e-6)
    # constant moving volume / constant fixed block: NCC := 0 everywhere, index 0 wins (reading Q12)
    vol = _smooth((24, 24, 16), 16)
    const = np.full_like(vol, 123.0)
    centres = np.asarray([[12, 12, 8]], dtype=np.int32)
    for f, m in ((vol, const), (const, vol)):
        for block, window in (((5, 5, 5), (3, 3, 3)), ((5, 5, 5), (2, 2, 2))):
            ora = oracle.match(f, m, centres, block, window)
            disp, ncc = nrr.nrr_bm_match(_cuda(f), _cuda(m), _cuda(centres), block, window)
            assert disp.cpu().numpy().tolist() == ora["disp"].tolist()
            assert ncc.cpu().numpy().tolist() == [0.0]


def test_match_zero_blocks_and_bounds_flag():
    vol = _smooth((24, 24, 16), 17)
    empty = torch.empty((0, 3), dtype=torch.int32, device="cuda")
    disp, ncc = nrr.nrr_bm_match(_cuda(vol), _cuda(vol), empty, (5, 5, 5), (3, 3, 3))
    assert disp.shape == (0, 3) and ncc.shape == (0,)
    nrr.nrr_bm_check_async_error()
    bad = np.asarray([[12, 12, 8], [1, 12, 8]], dtype=np.int32)        # second block leaves the volume
    disp, ncc = nrr.nrr_bm_match(_cuda(vol), _cuda(vol), _cuda(bad), (5, 5, 5), (3, 3, 3))
    with pytest.raises(nrr.NrrError) as ei:
        nrr.nrr_bm_check_async_error()
    assert ei.value.status == -8
    assert disp.cpu().numpy()[0].tolist() == [0, 0, 0] and np.isnan(ncc.cpu().numpy()[1])
    nrr.nrr_bm_check_async_error()                                       # flag was cleared


@pytest.mark.parametrize("b,r,rz", [(7, 5, 5), (5, 3, 3), (7, 5, 3), (9, 7, 7), (11, 9, 9), (5, 9, 9), (11, 3, 3)])
def test_match_every_candidate_row_can_win(b, r, rz):
    """Planted displacements covering every (dy, dz) candidate row and every dx of the window (nrr_inputs.planted)."""
    from nrr_inputs.planted import planted_pair
    fixed, moving, centres, want = planted_pair(b, r, rz)
    block, window = (b, b, b), (r, r, rz)
    assert nrr.nrr_bm_match_info(fixed.shape[::-1], block, window)["kernel"] == 2
    for opts in ({}, {"force_rows": 1}):
        disp, ncc = _with_options(opts, lambda: nrr.nrr_bm_match(_cuda(fixed), _cuda(moving), _cuda(centres), block, window))
        nrr.nrr_bm_check_async_error()
        assert np.array_equal(disp.cpu().numpy(), want), opts
        assert np.all(np.abs(ncc.cpu().numpy() - 1.0) < 1e-5)


def test_match_largest_fast_instantiation():
    dims, block, window = (64, 60, 56), (11, 11, 11), (9, 9, 9)
    vol = _smooth(dims, 41, sigma=2.0)
    mov = _shift_noise(vol, (4, -6, 5), 15.0, 42)
    sel = oracle.select(vol, block, (9, 9, 9), 0.4)
    ora = oracle.match(vol, mov, sel["centres"], block, window)
    assert nrr.nrr_bm_match_info(dims, block, window)["fast"]
    disp, ncc = nrr.nrr_bm_match(_cuda(vol), _cuda(mov), _cuda(sel["centres"]), block, window)
    assert_match_parity(disp.cpu().numpy(), ncc.cpu().numpy(), ora)


# ------------------------------------------------------------------------------------------- whole calls: host forms, register, plans, the BASELINE.json configs
def test_host_forms_equal_device_forms():
    cfg = CONFIGS["tiny"]
    fixed, moving, mask = pair("tiny")
    blocks, n, ncand = nrr.nrr_bm_select_blocks(_cuda(fixed), cfg.block, cfg.stride, cfg.frac)
    disp, ncc = nrr.nrr_bm_match(_cuda(fixed), _cuda(moving), blocks, cfg.block, cfg.window)
    hb, hn, hc, hv = nrr.nrr_bm_select_blocks_host(fixed, cfg.block, cfg.stride, cfg.frac)
    assert hn == n and hc == ncand and np.array_equal(hb, blocks.cpu().numpy())
    hd, hs = nrr.nrr_bm_match_host(fixed, moving, hb, cfg.block, cfg.window)
    assert np.array_equal(hd, disp.cpu().numpy()) and np.array_equal(hs, ncc.cpu().numpy())
    rb, rd, rs = nrr.nrr_bm_register_host(fixed, moving, cfg.block, cfg.stride, cfg.window, cfg.frac)
    assert np.array_equal(rb, hb) and np.array_equal(rd, hd) and np.array_equal(rs, hs)


@pytest.mark.parametrize("name", ["tiny", "intraop"])
def test_register_device_form_equals_select_then_match(name):
    """nrr_bm_register: no host synchronisation, K read on the device by kernels launched for an upper bound."""
    cfg = CONFIGS[name]
    fixed, moving, mask = pair(name)
    f, m, k = _cuda(fixed), _cuda(moving), _cuda(mask)
    blocks, n, ncand = nrr.nrr_bm_select_blocks(f, cfg.block, cfg.stride, cfg.frac, k)
    disp, ncc = nrr.nrr_bm_match(f, m, blocks, cfg.block, cfg.window)
    rb, rn, rd, rs = nrr.nrr_bm_register(f, m, cfg.block, cfg.stride, cfg.window, cfg.frac, k)
    nrr.nrr_bm_check_async_error()
    assert int(rn.item()) == n and rb.shape[0] >= n
    assert torch.equal(rb[:n], blocks) and torch.equal(rd[:n], disp) and torch.equal(rs[:n], ncc)
    # a capacity below K: the first `capacity` blocks are matched, K is still reported
    rb2, rn2, rd2, rs2 = nrr.nrr_bm_register(f, m, cfg.block, cfg.stride, cfg.window, cfg.frac, k, capacity=n // 2)
    torch.cuda.synchronize()
    assert int(rn2.item()) == n
    assert torch.equal(rb2, blocks[: n // 2]) and torch.equal(rd2, disp[: n // 2]) and torch.equal(rs2, ncc[: n // 2])


@pytest.mark.parametrize("name", ["tiny", "intraop", "fullres"])
def test_match_parity_configs_full(name):
    """BASELINE.json configs 1-3 at full size, every selected block, in the launch configuration bench.py uses."""
    cfg = CONFIGS[name]
    fixed, moving, mask = pair(name)
    blocks, n, ncand = nrr.nrr_bm_select_blocks(_cuda(fixed), cfg.block, cfg.stride, cfg.frac, _cuda(mask))
    disp, ncc = nrr.nrr_bm_match(_cuda(fixed), _cuda(moving), blocks, cfg.block, cfg.window)
    nrr.nrr_bm_check_async_error()
    ora = oracle.match(fixed, moving, blocks.cpu().numpy(), cfg.block, cfg.window)
    exempt = assert_match_parity(disp.cpu().numpy(), ncc.cpu().numpy(), ora, label=name)
    err = np.abs(ncc.cpu().numpy().astype(np.float64) - ora["ncc"])
    print("%s: %d blocks, %d inside the 1e-5 tie band (%d differ), max |dNCC| %.3g" % (
        name, n, int((ora["gap"] < 1e-5).sum()), exempt, err.max()))
    if name == "tiny":      # exact recovery of the constructed translation
        inside = np.all((blocks.cpu().numpy() - 2 + np.asarray(cfg.shift) >= np.maximum(cfg.shift, 0)) &
                        (blocks.cpu().numpy() + 3 + np.asarray(cfg.shift) <= np.asarray(cfg.dims) + np.minimum(cfg.shift, 0)), axis=1)
        assert np.all(disp.cpu().numpy()[inside] == np.asarray(cfg.shift))


@pytest.mark.parametrize("name", ["tiny", "intraop", "fullres"])
def test_plan_equals_select_then_match(name):
    """the pre-operative plan (selection + fixed-block records) and the intra-operative match give
    the bits of nrr_bm_select_blocks + nrr_bm_match; so do the host form's slab pipeline and a sharded block list."""
    cfg = CONFIGS[name]
    fixed, moving, mask = pair(name)
    f, m, k = _cuda(fixed), _cuda(moving), _cuda(mask)
    blocks, n, ncand = nrr.nrr_bm_select_blocks(f, cfg.block, cfg.stride, cfg.frac, k)
    disp, ncc = nrr.nrr_bm_match(f, m, blocks, cfg.block, cfg.window)
    plan = nrr.nrr_bm_plan_create(f, cfg.block, cfg.stride, cfg.window, cfg.frac, k)
    assert nrr.nrr_bm_plan_info(plan) == (n, ncand)
    assert np.array_equal(nrr.nrr_bm_plan_blocks_host(plan), blocks.cpu().numpy())
    assert torch.equal(nrr.nrr_bm_plan_blocks(plan), blocks)
    for _ in range(2):                                               # a plan serves many intra-operative volumes
        pd, pn = nrr.nrr_bm_plan_match(plan, m)
        nrr.nrr_bm_check_async_error()
        assert torch.equal(pd, disp) and torch.equal(pn, ncc)
    od = torch.full((n, 3), -99, dtype=torch.int32, device="cuda")
    on = torch.full((n,), -99.0, dtype=torch.float32, device="cuda")
    cuts = [0, n // 2, n]                                            # two "ranks", each its slice of the block list
    for a, b in zip(cuts[:-1], cuts[1:]):
        nrr.nrr_bm_plan_match_range(plan, m, od, on, first=a, count=b - a)
    nrr.nrr_bm_check_async_error()
    assert torch.equal(od, disp) and torch.equal(on, ncc)
    nrr.nrr_bm_plan_destroy(plan)
    hplan = nrr.nrr_bm_plan_create_host(fixed, cfg.block, cfg.stride, cfg.window, cfg.frac, mask)
    for slabs in (4, 1, 9):
        nrr.nrr_bm_set_option("plan_slabs", slabs)
        hd, hn = nrr.nrr_bm_plan_match_host(hplan, moving)
        assert np.array_equal(hd, disp.cpu().numpy()) and np.array_equal(hn, ncc.cpu().numpy()), slabs
    nrr.nrr_bm_set_option("plan_slabs", 4)
    nrr.nrr_bm_plan_destroy(hplan)


def test_register_then_regularise_then_warp_on_the_tiny_config():
    """The whole chain on the device: select + match -> biomechanical regularisation
     -> dense field -> warp.  The constructed translation (2,-1,1) is recovered
    at every mesh node and the warped intra-operative image lands on the pre-operative one."""
    cfg = CONFIGS["tiny"]
    fixed, moving, _ = pair("tiny")
    f, m = _cuda(fixed), _cuda(moving)
    blocks, n, _ = nrr.nrr_bm_select_blocks(f, cfg.block, cfg.stride, cfg.frac)
    disp, ncc = nrr.nrr_bm_match(f, m, blocks, cfg.block, cfg.window)
    fem = nrr.nrr_bm_fem_create(cfg.dims, (8, 8, 8), 1.0, 0.45)
    u, iters = nrr.nrr_bm_fem_solve(fem, blocks, disp, ncc, weight=1.0, n_iter=5)
    un = u.cpu().numpy()
    nn = np.asarray(fem.nodes)
    core = un.reshape(nn[2], nn[1], nn[0], 3)[1:-1, 1:-1, 1:-1]               # away from the hull (clamped shift, skipped candidates)
    dev = np.abs(core - np.asarray(cfg.shift))                                   # border blocks see the clamped shift
    assert np.median(dev) < 0.1 and np.max(dev) < 1.0, (np.median(dev), np.max(dev))
    field = nrr.nrr_bm_fem_dense_field(fem, u)
    warped = nrr.nrr_bm_warp(m, field).cpu().numpy()
    inner = (slice(6, -6), slice(8, -8), slice(8, -8))
    before = np.abs(moving[inner] - fixed[inner]).mean()
    after = np.abs(warped[inner] - fixed[inner]).mean()
    print("tiny chain: %d blocks, %d CG iterations, mean |moving - fixed| %.2f -> %.2f after the warp" % (n, iters, before, after))
    assert after < 0.5 * before
    nrr.nrr_bm_fem_destroy(fem)


def test_match_parity_highres_sampled():
    """Config 4 (512x512x176, 9^3, +-7): the full launch on the GPU, 400 sampled blocks on the oracle."""
    cfg = CONFIGS["highres"]
    fixed, moving, mask = pair("highres")
    blocks, n, ncand = nrr.nrr_bm_select_blocks(_cuda(fixed), cfg.block, cfg.stride, cfg.frac)
    assert (ncand, n) == (197568, 39514)
    disp, ncc = nrr.nrr_bm_match(_cuda(fixed), _cuda(moving), blocks, cfg.block, cfg.window)
    nrr.nrr_bm_check_async_error()
    idx = np.unique(np.concatenate([np.arange(40), np.arange(n - 40, n),
                                    np.random.default_rng(5).choice(n, 320, replace=False)]))
    ora = oracle.match(fixed, moving, blocks.cpu().numpy()[idx], cfg.block, cfg.window)
    exempt = assert_match_parity(disp.cpu().numpy()[idx], ncc.cpu().numpy()[idx], ora, label="highres")
    print("highres: %d blocks on the GPU, %d checked, %d exempt" % (n, len(idx), exempt))
    worst = assert_ncc_of_chosen_displacement(fixed, moving, blocks.cpu().numpy(), cfg.block, disp.cpu().numpy(), ncc.cpu().numpy(), "highres")
    print("highres: all %d blocks: max |ncc - oracle.ncc_at(disp)| %.3g" % (n, worst))
    # properties that hold at any size
    d = disp.cpu().numpy()
    assert np.all(np.abs(d) <= np.asarray(cfg.window))
    s = ncc.cpu().numpy()
    assert np.all(np.isfinite(s)) and np.all(s <= 1.0 + 1e-5) and np.all(s >= -1.0 - 1e-5)


def test_match_parity_batch_sampled():
    """Config 5: 32 settings on the fullres pair as ONE launch sequence that shares work (nrr_bm_register_batch: no
    host synchronisation; normalisers per block shape, variance keys per (block, stride), records per block list).
    Per setting the selection is checked in full, 48 sampled blocks against the full oracle search, and EVERY block's
    NCC against the oracle's NCC of the displacement it chose."""
    fixed, moving, mask = pair("fullres")
    f, m, k = _cuda(fixed), _cuda(moving), _cuda(mask)
    settings = list(batch_settings())
    assert len(settings) == 32
    results, out_n = nrr.nrr_bm_register_batch(f, m, settings, k)
    nrr.nrr_bm_check_async_error()                                   # the only synchronisation
    ns = out_n.cpu().numpy()
    total_exempt = total_blocks = 0
    worst = 0.0
    for si, (st, (rb, rd, rs)) in enumerate(zip(settings, results)):
        n = int(ns[si])
        ora_sel = oracle.select(fixed, st.block, st.stride, st.frac, mask)
        assert_select_parity(rb[:n].cpu().numpy(), n, ora_sel["n_candidates"], ora_sel)
        idx = np.sort(np.random.default_rng(1000 + si).choice(n, 48, replace=False))
        ora = oracle.match(fixed, moving, ora_sel["centres"][idx], st.block, st.window)
        total_exempt += assert_match_parity(rd[:n].cpu().numpy()[idx], rs[:n].cpu().numpy()[idx], ora, label=str(st))
        worst = max(worst, assert_ncc_of_chosen_displacement(fixed, moving, ora_sel["centres"], st.block, rd[:n].cpu().numpy(),
                                                             rs[:n].cpu().numpy(), str(st)))
        total_blocks += n
    print("batch: 32 settings, %d blocks, %d exempt blocks among the samples, all blocks: max |ncc - oracle.ncc_at(disp)| %.3g" % (
        total_blocks, total_exempt, worst))
    # the same sweep as 32 separate nrr_bm_register calls gives the same bits
    for si in (0, 13, 31):
        st = settings[si]
        rb, rn, rd, rs = nrr.nrr_bm_register(f, m, st.block, st.stride, st.window, st.frac, k)
        torch.cuda.synchronize()
        n = int(rn.item())
        assert n == int(ns[si]) and torch.equal(rb[:n], results[si][0][:n])
        assert torch.equal(rd[:n], results[si][1][:n]) and torch.equal(rs[:n], results[si][2][:n])


# ------------------------------------------------------------------------------------------- the bounded staging wait (last: it makes a kernel wait out its time bound)
def test_staging_timeout_reports_device_error_without_faulting():
    """The matching kernel's bounded wait: an over-programmed staging barrier must end as NRR_E_DEVICE (-12) with NaN
    results and a usable context afterwards -- never a trap."""
    cfg = CONFIGS["tiny"]
    fixed, moving, _ = pair("tiny")
    f, m = _cuda(fixed), _cuda(moving)
    blocks, n, _ = nrr.nrr_bm_select_blocks(f, cfg.block, cfg.stride, cfg.frac)
    good = nrr.nrr_bm_match(f, m, blocks[:8], cfg.block, cfg.window)
    nrr.nrr_bm_check_async_error()
    nrr.nrr_bm_set_option("debug_expect_tx_extra", 16)
    try:
        bad = nrr.nrr_bm_match(f, m, blocks[:8], cfg.block, cfg.window)        # 2 CTAs wait out the time bound (seconds)
        with pytest.raises(nrr.NrrError) as ei:
            nrr.nrr_bm_check_async_error()
        assert ei.value.status == -12
        assert torch.isnan(bad[1]).all()
    finally:
        nrr.nrr_bm_set_option("debug_expect_tx_extra", 0)
    again = nrr.nrr_bm_match(f, m, blocks[:8], cfg.block, cfg.window)
    nrr.nrr_bm_check_async_error()
    assert torch.equal(again[0], good[0]) and torch.equal(again[1], good[1])
