"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, no CUDA path involved).

Every check compares oracle/nrr_oracle.c with something other than itself: closed forms in tests/golden/,
numpy's own variance / corrcoef, invariants of Pearson's r, exact recovery of a constructed integer
translation, counting identities of the skip rule, and the independent naive evaluator oracle/naive.py.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from oracle import naive
from nrr_inputs import CONFIGS, make_mask, make_pair


def _rng(seed):
    return np.random.default_rng(seed)


def _smooth_volume(dims, seed, sigma=1.5):
    from scipy import ndimage
    nx, ny, nz = dims
    v = ndimage.gaussian_filter(_rng(seed).standard_normal((nz, ny, nx)), sigma, mode="reflect")
    v = (v - v.min()) / (v.max() - v.min()) * 1000.0
    return v.astype(np.float32)


# ----------------------------------------------------------------------------- variance / count / NCC
def test_variance_golden(golden):
    for row in golden("variance_small.txt"):
        k = row.index("|")
        vals = [float(t) for t in row[:k]]
        assert oracle.variance(vals) == pytest.approx(float(row[k + 1]), abs=1e-12)


def test_variance_matches_numpy_population_variance():
    r = _rng(1)
    for n in (2, 27, 125, 343, 729, 1331):
        a = r.uniform(0, 1000, size=n).astype(np.float32)
        assert oracle.variance(a) == pytest.approx(float(np.var(a.astype(np.float64))), rel=1e-12)
        # population, not sample, variance (reading Q7)
        assert oracle.variance(a) != pytest.approx(float(np.var(a.astype(np.float64), ddof=1)), rel=1e-6)


def test_count_rule_golden(golden):
    for n, frac, k in golden("count_rule.txt"):
        assert oracle.count(int(n), float(frac)) == int(k)


def test_ncc_golden(golden):
    for row in golden("ncc_small.txt"):
        i, j = [t for t, s in enumerate(row) if s == "|"]
        a = [float(t) for t in row[:i]]
        b = [float(t) for t in row[i + 1:j]]
        assert oracle.ncc(a, b) == pytest.approx(float(row[j + 1]), abs=1e-14)


def test_ncc_equals_numpy_corrcoef():
    """SPEC.md:681 acceptance #1: 10^4 random block pairs against an independently coded correlation."""
    r = _rng(2)
    for n in (3, 125, 343, 729, 1331):
        for _ in range(2000):
            a = r.uniform(0, 1000, size=n).astype(np.float32)
            b = (0.3 * a + r.normal(0, 200, size=n)).astype(np.float32)
            ref = float(np.corrcoef(a.astype(np.float64), b.astype(np.float64))[0, 1])
            assert oracle.ncc(a, b) == pytest.approx(ref, abs=1e-12)


def test_ncc_invariants():
    r = _rng(3)
    a = r.uniform(0, 1000, size=343)
    b = 0.5 * a + r.normal(0, 100, size=343)
    s = oracle.ncc(a, b)
    assert oracle.ncc(a, a) == pytest.approx(1.0, abs=1e-15)
    assert oracle.ncc(a, 3.5 * a + 17.0) == pytest.approx(1.0, abs=1e-12)
    assert oracle.ncc(a, -2.0 * a + 5.0) == pytest.approx(-1.0, abs=1e-12)
    assert oracle.ncc(b, a) == pytest.approx(s, abs=1e-15)                      # symmetry
    assert oracle.ncc(2.0 * a + 100.0, b) == pytest.approx(s, abs=1e-12)        # positive affine map, 1st arg
    assert oracle.ncc(a, 0.25 * b - 40.0) == pytest.approx(s, abs=1e-12)        # positive affine map, 2nd arg
    assert oracle.ncc(a, -b) == pytest.approx(-s, abs=1e-12)
    assert -1.0 <= s <= 1.0
    assert oracle.ncc(np.full(343, 7.0), b) == 0.0 and oracle.ncc(a, np.full(343, 7.0)) == 0.0
    assert oracle.ncc(a, b) == pytest.approx(naive.ncc(list(a), list(b)), abs=1e-13)


# ----------------------------------------------------------------------------- selection
def test_select_uniform_image_gives_first_k_indices():
    vol = np.full((12, 15, 20), 42.0, dtype=np.float32)      # nz, ny, nx
    res = oracle.select(vol, (3, 3, 3), (3, 3, 3), 0.25)
    g = oracle.grid((20, 15, 12), (3, 3, 3), (3, 3, 3))
    assert g == (6, 5, 4)
    n = g[0] * g[1] * g[2]
    k = math.floor(0.5 + n * 0.25)
    assert res["n_candidates"] == n and len(res["centres"]) == k
    assert np.all(res["var"] == 0.0)
    expect = [(1 + 3 * (q % 6), 1 + 3 * ((q // 6) % 5), 1 + 3 * (q // 30)) for q in range(k)]
    assert res["centres"].tolist() == [list(t) for t in expect]


def test_select_thousand_candidates_five_percent():
    vol = _smooth_volume((50, 50, 10), 4)                   # stride 5, block 5 -> 10 x 10 x 2 = 200 ... use stride 1
    res = oracle.select(vol, (5, 5, 5), (5, 5, 1), 0.05)    # grid 10 x 10 x 6 = 600
    assert res["n_candidates"] == 600 and len(res["centres"]) == 30
    vol2 = _smooth_volume((104, 54, 5), 5)                  # block 5, stride 1,5,1 -> 100 x 10 x 1 = 1000
    res2 = oracle.select(vol2, (5, 5, 5), (1, 5, 1), 0.05)
    assert res2["n_candidates"] == 1000 and len(res2["centres"]) == 50


def _bruteforce_select(vol, block, stride, frac, mask):
    nz, ny, nx = vol.shape
    bx, by, bz = block
    cents, var = [], []
    for oz, oy, ox in itertools.product(range(0, nz - bz + 1, stride[2]), range(0, ny - by + 1, stride[1]),
                                        range(0, nx - bx + 1, stride[0])):
        c = (ox + bx // 2, oy + by // 2, oz + bz // 2)
        if mask is not None and mask[c[2], c[1], c[0]] == 0:
            continue
        cents.append(c)
        var.append(np.var(vol[oz:oz + bz, oy:oy + by, ox:ox + bx].astype(np.float64)))
    var = np.asarray(var)
    k = int(math.floor(0.5 + len(cents) * frac))
    full = np.lexsort((np.arange(len(cents)), -var))
    order = full[:k]
    keep = np.sort(order)
    # K / K+1 variance margin: how far the last kept candidate is from the first one left out
    margin = float("nan") if k == 0 else (float("inf") if k == len(cents) else float(var[full[k - 1]] - var[full[k]]))
    _bruteforce_select.margin = margin
    return np.asarray(cents, dtype=np.int32)[keep], var[keep], len(cents)


@pytest.mark.parametrize("block,stride,frac,use_mask", [
    ((5, 5, 5), (5, 5, 5), 0.3, False),
    ((7, 7, 7), (5, 5, 5), 0.25, True),
    ((3, 5, 7), (4, 3, 2), 0.5, True),          # anisotropic: catches transposed axes
    ((9, 9, 9), (6, 6, 6), 1.0, False),         # frac = 1 keeps everything
])
def test_select_matches_numpy_bruteforce(block, stride, frac, use_mask):
    dims = (41, 37, 29)                         # ragged: not a multiple of anything
    vol = _smooth_volume(dims, 6)
    mask = None
    if use_mask:
        from nrr_inputs import spherical_mask
        mask = spherical_mask(dims, 15.0)
    res = oracle.select(vol, block, stride, frac, mask)
    cents, var, n = _bruteforce_select(vol, block, stride, frac, mask)
    assert res["n_candidates"] == n
    assert res["centres"].tolist() == cents.tolist()
    np.testing.assert_allclose(res["var"], var, rtol=1e-12)
    want_margin = _bruteforce_select.margin           # out_margin of nrr_oracle_select, against numpy
    if math.isinf(want_margin):
        assert math.isinf(res["margin"]) and res["margin"] > 0
    else:
        assert res["margin"] >= 0 and res["margin"] == pytest.approx(want_margin, rel=1e-9, abs=1e-9)
    lin = (res["centres"][:, 2].astype(np.int64) * dims[1] + res["centres"][:, 1]) * dims[0] + res["centres"][:, 0]
    assert np.all(np.diff(lin) > 0)             # canonical ascending order (Q8)


def test_select_matches_naive_evaluator():
    vol = _smooth_volume((24, 20, 14), 7)
    from nrr_inputs import spherical_mask
    mask = spherical_mask((24, 20, 14), 8.0)
    a = oracle.select(vol, (5, 3, 5), (3, 4, 2), 0.4, mask)
    b = naive.select(vol, (5, 3, 5), (3, 4, 2), 0.4, mask)
    assert a["n_candidates"] == b["n_candidates"]
    assert a["centres"].tolist() == b["centres"].tolist()
    np.testing.assert_allclose(a["var"], b["var"], rtol=1e-12)


def test_select_variance_ties_prefer_lower_index():
    # two identical bright patterns at different grid positions and a flat background: with K = 1 the
    # lower-index copy must win; with K = 2 both.
    vol = np.zeros((6, 6, 18), dtype=np.float32)            # nz, ny, nx ; block 3, stride 3 -> grid 6 x 2 x 2
    pat = np.arange(27, dtype=np.float32).reshape(3, 3, 3)
    vol[0:3, 0:3, 3:6] = pat                                # grid q = 1
    vol[3:6, 3:6, 12:15] = pat                              # grid q = 4 + 6 + 12 = 22
    r1 = oracle.select(vol, (3, 3, 3), (3, 3, 3), 1.0 / 24.0)
    assert r1["centres"].tolist() == [[4, 1, 1]]
    r2 = oracle.select(vol, (3, 3, 3), (3, 3, 3), 2.0 / 24.0)
    assert r2["centres"].tolist() == [[4, 1, 1], [13, 4, 4]]
    assert r2["var"][0] == r2["var"][1] == pytest.approx(np.var(np.arange(27.0)))


def test_config_candidate_counts_golden(golden):
    for name, ngrid, n, k, ncand in golden("config_counts.txt"):
        cfg = CONFIGS[name]
        g = oracle.grid(cfg.dims, cfg.block, cfg.stride)
        assert g[0] * g[1] * g[2] == int(ngrid)
        mask = make_mask(cfg)
        if mask is None:
            n_in = int(ngrid)
        else:
            cx = np.arange(g[0]) * cfg.stride[0] + cfg.block[0] // 2
            cy = np.arange(g[1]) * cfg.stride[1] + cfg.block[1] // 2
            cz = np.arange(g[2]) * cfg.stride[2] + cfg.block[2] // 2
            n_in = int(mask[np.ix_(cz, cy, cx)].astype(bool).sum())
        assert n_in == int(n)
        assert oracle.count(n_in, cfg.frac) == int(k)
        assert cfg.n_candidates == int(ncand)


# ----------------------------------------------------------------------------- matching
def _shifted(vol, s):
    """moving(p) = vol(clamp(p - s))  =>  vol(p) <-> moving(p + s)."""
    nz, ny, nx = vol.shape
    iz = np.clip(np.arange(nz) - s[2], 0, nz - 1)
    iy = np.clip(np.arange(ny) - s[1], 0, ny - 1)
    ix = np.clip(np.arange(nx) - s[0], 0, nx - 1)
    return np.ascontiguousarray(vol[np.ix_(iz, iy, ix)])


def _interior(centres, dims, block, shift):
    """Blocks whose translated box stays strictly away from the clamped border."""
    keep = []
    for c in centres:
        ok = True
        for a in range(3):
            o = c[a] - block[a] // 2 + shift[a]
            lo = max(shift[a], 0)
            hi = dims[a] + min(shift[a], 0)
            ok &= (o >= lo) and (o + block[a] <= hi)
        keep.append(ok)
    return np.asarray(keep)


@pytest.mark.parametrize("shift", [(2, -1, 1), (-3, 0, 2), (0, 3, -2)])
def test_match_recovers_integer_translation_exactly(shift):
    dims = (40, 36, 24)
    block, window = (5, 5, 5), (3, 3, 3)
    vol = _smooth_volume(dims, 8)
    moving = _shifted(vol, shift)
    sel = oracle.select(vol, block, (5, 5, 5), 0.5)
    res = oracle.match(vol, moving, sel["centres"], block, window)
    inside = _interior(sel["centres"], dims, block, shift)
    assert inside.sum() > 20
    assert np.all(res["disp"][inside] == np.asarray(shift))           # sign and axis order (Q15)
    np.testing.assert_allclose(res["ncc"][inside], 1.0, atol=1e-12)
    assert np.all(res["ncc"] <= 1.0 + 1e-12)


def test_match_identical_volumes_zero_displacement():
    vol = _smooth_volume((30, 30, 20), 9)
    sel = oracle.select(vol, (7, 7, 7), (5, 5, 5), 0.5)
    res = oracle.match(vol, vol, sel["centres"], (7, 7, 7), (2, 2, 2))
    assert np.all(res["disp"] == 0)
    np.testing.assert_allclose(res["ncc"], 1.0, atol=1e-12)
    assert np.all(res["gap"] > 0)


def test_match_argmax_invariant_to_positive_affine_intensity_map():
    dims = (32, 28, 20)
    vol = _smooth_volume(dims, 10)
    moving = (_shifted(vol, (1, 2, -1)) + _rng(11).normal(0, 20, size=vol.shape)).astype(np.float32)
    sel = oracle.select(vol, (5, 5, 5), (4, 4, 4), 0.3)
    a = oracle.match(vol, moving, sel["centres"], (5, 5, 5), (3, 3, 3))
    b = oracle.match(vol, (2.0 * moving + 64.0).astype(np.float32), sel["centres"], (5, 5, 5), (3, 3, 3))
    c = oracle.match((0.5 * vol + 8.0).astype(np.float32), moving, sel["centres"], (5, 5, 5), (3, 3, 3))
    sure = a["gap"] > 1e-6     # 2*m+64 and 0.5*f+8 are exact in fp32 only up to rounding; skip photo-finishes
    assert sure.sum() > 0.9 * len(sure)
    assert np.all(a["disp"][sure] == b["disp"][sure]) and np.all(a["disp"][sure] == c["disp"][sure])
    np.testing.assert_allclose(a["ncc"], b["ncc"], atol=1e-6)
    np.testing.assert_allclose(a["ncc"], c["ncc"], atol=1e-6)


def test_match_agrees_with_naive_evaluator_including_borders():
    dims = (16, 14, 12)
    vol = _smooth_volume(dims, 12, sigma=1.0)
    moving = (_shifted(vol, (1, -1, 1)) + _rng(13).normal(0, 30, size=vol.shape)).astype(np.float32)
    block, window = (3, 5, 3), (2, 1, 3)        # anisotropic block and window
    # every grid block, including the ones touching the border (skip rule, Q11)
    sel = oracle.select(vol, block, (4, 3, 3), 1.0)
    a = oracle.match(vol, moving, sel["centres"], block, window)
    b = naive.match(vol, moving, sel["centres"], block, window)
    assert a["disp"].tolist() == b["disp"].tolist()
    np.testing.assert_allclose(a["ncc"], b["ncc"], atol=1e-12)
    finite = np.isfinite(b["gap"])
    np.testing.assert_allclose(a["gap"][finite], b["gap"][finite], atol=1e-12)


def test_match_skip_rule_counts_valid_candidates():
    dims = (20, 18, 16)
    vol = _smooth_volume(dims, 14)
    block, window = (5, 5, 5), (3, 2, 4)
    centres = np.asarray([[2, 2, 2], [17, 15, 13], [10, 9, 8], [2, 9, 13], [4, 3, 2]], dtype=np.int32)
    res = oracle.match(vol, vol, centres, block, window)
    for c, nv in zip(centres, res["nvalid"]):
        expect = 1
        for a in range(3):
            o = c[a] - block[a] // 2
            lo = max(-window[a], -o)
            hi = min(window[a], dims[a] - block[a] - o)
            expect *= hi - lo + 1
        assert nv == expect
    assert res["nvalid"][2] == 7 * 5 * 9        # interior block: the whole window
    assert res["nvalid"][0] == 4 * 3 * 5        # corner block: only non-negative displacements


def test_match_equal_maxima_keep_lowest_linear_index():
    # a volume periodic with period 2 along x: displacements dx = -2, 0, +2 give bit-identical blocks,
    # so three candidates tie exactly; the lowest linear index (dx = -2, dy = dz = 0 is not lowest: the tie
    # set is {(-2,0,0),(0,0,0),(2,0,0)} and the rule picks dx = -2).
    nz, ny, nx = 9, 9, 16
    base = _rng(15).uniform(0, 1000, size=(nz, ny, 2)).astype(np.float32)
    vol = np.tile(base, (1, 1, nx // 2))
    centres = np.asarray([[8, 4, 4]], dtype=np.int32)
    res = oracle.match(vol, vol, centres, (3, 3, 3), (2, 0, 0))
    assert res["disp"].tolist() == [[-2, 0, 0]]
    assert res["ncc"][0] == pytest.approx(1.0, abs=1e-15)
    assert res["gap"][0] == 0.0                  # reported as a tie: inside the 1e-5 exemption band
    nv = naive.match(vol, vol, centres, (3, 3, 3), (2, 0, 0))
    assert nv["disp"].tolist() == [[-2, 0, 0]]


def test_match_constant_regions_score_zero():
    vol = _smooth_volume((20, 20, 12), 16)
    moving = vol.copy()
    moving[:, :, :] = 123.0                      # constant moving volume: every candidate has SSm = 0
    centres = np.asarray([[10, 10, 6]], dtype=np.int32)
    res = oracle.match(vol, moving, centres, (5, 5, 5), (2, 2, 2))
    assert res["ncc"][0] == 0.0 and res["disp"].tolist() == [[-2, -2, -2]]       # all tie at 0 -> index 0
    flat = np.full_like(vol, 55.0)
    res2 = oracle.match(flat, vol, centres, (5, 5, 5), (2, 2, 2))                 # constant fixed block
    assert res2["ncc"][0] == 0.0 and res2["disp"].tolist() == [[-2, -2, -2]]


def test_match_independent_of_thread_count():
    vol = _smooth_volume((36, 30, 22), 17)
    moving = (_shifted(vol, (1, 1, 0)) + _rng(18).normal(0, 25, size=vol.shape)).astype(np.float32)
    sel = oracle.select(vol, (5, 5, 5), (5, 5, 5), 0.6)
    a = oracle.match(vol, moving, sel["centres"], (5, 5, 5), (2, 2, 2), nthreads=1)
    b = oracle.match(vol, moving, sel["centres"], (5, 5, 5), (2, 2, 2), nthreads=4)
    assert a["disp"].tolist() == b["disp"].tolist()
    assert np.array_equal(a["ncc"], b["ncc"]) and np.array_equal(a["gap"], b["gap"])


def test_ncc_at_agrees_with_match_best():
    vol = _smooth_volume((26, 24, 18), 19)
    moving = (_shifted(vol, (-1, 2, 1)) + _rng(20).normal(0, 15, size=vol.shape)).astype(np.float32)
    sel = oracle.select(vol, (5, 5, 5), (5, 5, 5), 0.3)
    res = oracle.match(vol, moving, sel["centres"], (5, 5, 5), (3, 3, 3))
    for c, d, s in zip(sel["centres"], res["disp"], res["ncc"]):
        assert oracle.ncc_at(vol, moving, c, (5, 5, 5), d) == s
    assert math.isnan(oracle.ncc_at(vol, moving, (2, 2, 2), (5, 5, 5), (-1, 0, 0)))


def test_tiny_config_exact_recovery_with_noise():
    """BASELINE.json configs[0]: moving = fixed shifted by (2,-1,1) + N(0,10); the exhaustive search must
    return exactly that displacement for every block whose translated box stays inside the volume."""
    cfg = CONFIGS["tiny"]
    fixed, moving, mask = make_pair(cfg)
    assert mask is None and fixed.dtype == np.float32 and fixed.shape == (32, 64, 64)
    assert 0.0 <= fixed.min() and fixed.max() <= 1000.0
    sel = oracle.select(fixed, cfg.block, cfg.stride, cfg.frac, mask)
    assert sel["n_candidates"] == 864 and len(sel["centres"]) == 259
    res = oracle.match(fixed, moving, sel["centres"], cfg.block, cfg.window)
    inside = _interior(sel["centres"], cfg.dims, cfg.block, cfg.shift)
    assert inside.sum() >= 200
    assert np.all(res["disp"][inside] == np.asarray(cfg.shift))
    assert np.all(res["ncc"][inside] > 0.9)


# ------------------------------------------------------------------------- selection with a connectivity pattern
def _pruned_bruteforce(vol, block, stride, frac, mask, connectivity):
    """Independent restatement (numpy + python sets) of reading Q20: greedy by (variance desc, index asc).
    The per-candidate variance is taken from oracle.variance ON PURPOSE: that function is pinned on its own
    (closed forms, numpy.var) and using its bits keeps exact variance ties exact, so that this pin tests the walk
    (priority order, neighbourhood, stopping rule, output order) and nothing else."""
    nz, ny, nx = vol.shape
    g = [(n - b) // s + 1 for n, b, s in zip((nx, ny, nz), block, stride)]
    reach = {0: 0, 6: 1, 18: 2, 26: 3}[connectivity]
    cands = []
    for k in range(g[2]):
        for j in range(g[1]):
            for i in range(g[0]):
                o = (i * stride[0], j * stride[1], k * stride[2])
                c = tuple(o[a] + (block[a] - 1) // 2 for a in range(3))
                if mask is not None and mask[c[2], c[1], c[0]] == 0:
                    continue
                blk = vol[o[2]:o[2] + block[2], o[1]:o[1] + block[1], o[0]:o[0] + block[0]].astype(np.float64)
                # the variance itself is pinned elsewhere; taking the oracle's keeps exact ties exact here
                cands.append((oracle.variance(blk.ravel()), len(cands), (i, j, k), c))
    K = min(len(cands), int(math.floor(0.5 + len(cands) * frac)))
    kept, kept_pos = [], set()
    for var, q, gp, c in sorted(cands, key=lambda t: (-t[0], t[1])):
        if len(kept) == K:
            break
        nb = [(gp[0] + di, gp[1] + dj, gp[2] + dk) for di in (-1, 0, 1) for dj in (-1, 0, 1) for dk in (-1, 0, 1)
              if 0 < abs(di) + abs(dj) + abs(dk) <= reach]
        if any(p in kept_pos for p in nb):
            continue
        kept.append((q, c))
        kept_pos.add(gp)
    kept.sort()
    return np.asarray([c for _, c in kept], dtype=np.int32).reshape(-1, 3), len(cands)


def test_select_pruned_without_pattern_equals_plain_selection():
    vol = np.random.default_rng(3).uniform(0, 1000, (14, 13, 12)).astype(np.float32)
    a = oracle.select(vol, (3, 3, 3), (1, 1, 1), 0.2)
    b = oracle.select_pruned(vol, (3, 3, 3), (1, 1, 1), 0.2, None, 0)
    assert np.array_equal(a["centres"], b["centres"]) and np.array_equal(a["var"], b["var"])


def test_select_pruned_uniform_image_closed_forms():
    """All variances equal -> candidates are walked in index order, so the kept set has a closed form:
    face (6): i+j+k even; vertex (26): i, j, k all even; on a line every other candidate."""
    vol = np.full((9, 9, 9), 5.0, np.float32)                     # 7x7x7 grid of 3^3 blocks at stride 1
    c = oracle.select_pruned(vol, (3, 3, 3), (1, 1, 1), 1.0, None, 6)["centres"] - 1        # grid coordinates
    want = [(i, j, k) for k in range(7) for j in range(7) for i in range(7) if (i + j + k) % 2 == 0]
    assert c.tolist() == [list(t) for t in want]
    c = oracle.select_pruned(vol, (3, 3, 3), (1, 1, 1), 1.0, None, 26)["centres"] - 1
    want = [(i, j, k) for k in range(0, 7, 2) for j in range(0, 7, 2) for i in range(0, 7, 2)]
    assert c.tolist() == [list(t) for t in want]
    line = np.full((3, 3, 12), 5.0, np.float32)                   # a 10x1x1 grid
    for conn in (6, 18, 26):
        c = oracle.select_pruned(line, (3, 3, 3), (1, 1, 1), 1.0, None, conn)["centres"]
        assert c[:, 0].tolist() == [1, 3, 5, 7, 9]
    # the count rule stops the walk: K = floor(0.5 + 10 * 0.25) = 3 kept, the first three of the pattern
    c = oracle.select_pruned(line, (3, 3, 3), (1, 1, 1), 0.25, None, 6)["centres"]
    assert c[:, 0].tolist() == [1, 3, 5]


@pytest.mark.parametrize("conn", [6, 18, 26])
@pytest.mark.parametrize("stride,frac,use_mask", [((1, 1, 1), 0.1, False), ((1, 1, 1), 0.6, True), ((2, 1, 3), 0.5, False)])
def test_select_pruned_matches_bruteforce_and_is_an_independent_set(conn, stride, frac, use_mask):
    rng = np.random.default_rng(40 + conn)
    vol = rng.uniform(0, 1000, (11, 12, 13)).astype(np.float32)
    vol[:4] = np.round(vol[:4] / 250.0) * 250.0                   # many exact variance ties
    mask = (rng.uniform(size=vol.shape) < 0.7).astype(np.uint8) if use_mask else None
    got = oracle.select_pruned(vol, (3, 3, 3), stride, frac, mask, conn)
    want, ncand = _pruned_bruteforce(vol, (3, 3, 3), stride, frac, mask, conn)
    assert got["n_candidates"] == ncand
    assert np.array_equal(got["centres"], want)
    # invariant: no two kept centres are neighbours under the pattern (grid coordinates)
    gp = (got["centres"] - 1) // np.asarray(stride)
    d = np.abs(gp[:, None, :] - gp[None, :, :])
    near = (d.max(axis=2) <= 1) & (d.sum(axis=2) <= {6: 1, 18: 2, 26: 3}[conn]) & (d.sum(axis=2) > 0)
    assert not near.any()
    assert len(got["centres"]) <= oracle.count(ncand, frac)


def test_select_pruned_isolated_candidates_are_untouched():
    vol = np.random.default_rng(9).uniform(0, 1000, (12, 12, 12)).astype(np.float32)
    mask = np.zeros(vol.shape, np.uint8)
    mask[1::3, 1::3, 1::3] = 1                                    # candidates three voxels apart: never neighbours
    a = oracle.select(vol, (3, 3, 3), (1, 1, 1), 0.5, mask)
    b = oracle.select_pruned(vol, (3, 3, 3), (1, 1, 1), 0.5, mask, 26)
    assert np.array_equal(a["centres"], b["centres"])


# ------------------------------------------------------------------------------------ dense-field warp (Q21)
def test_warp_identity_and_integer_translation_are_exact():
    rng = np.random.default_rng(5)
    img = rng.uniform(0, 1000, (9, 10, 11)).astype(np.float32)
    zero = np.zeros((3,) + img.shape, np.float32)
    assert np.array_equal(oracle.warp(img, zero), img)
    f = zero.copy()
    f[0], f[1], f[2] = 2.0, -1.0, 3.0                             # out(p) = img(clamp(p + (2,-1,3)))
    nz, ny, nx = img.shape
    iz = np.clip(np.arange(nz) + 3, 0, nz - 1)
    iy = np.clip(np.arange(ny) - 1, 0, ny - 1)
    ix = np.clip(np.arange(nx) + 2, 0, nx - 1)
    assert np.array_equal(oracle.warp(img, f), img[np.ix_(iz, iy, ix)])


def test_warp_reproduces_affine_images_and_matches_scipy():
    from scipy import ndimage
    rng = np.random.default_rng(6)
    nz, ny, nx = 12, 13, 14
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    field = rng.uniform(-1.5, 1.5, (3, nz, ny, nx)).astype(np.float32)
    # trilinear interpolation reproduces affine functions wherever the sample stays inside the volume
    img = (3.0 * x - 2.0 * y + 0.5 * z + 7.0).astype(np.float32)
    sx, sy, sz = x + field[0].astype(np.float64), y + field[1].astype(np.float64), z + field[2].astype(np.float64)
    inside = (sx >= 0) & (sx <= nx - 1) & (sy >= 0) & (sy <= ny - 1) & (sz >= 0) & (sz <= nz - 1)
    got = oracle.warp(img, field).astype(np.float64)
    want = 3.0 * sx - 2.0 * sy + 0.5 * sz + 7.0
    assert np.max(np.abs(got - want)[inside]) < 1e-5
    # a library routine with the same definition: order-1 spline, coordinates clamped to the edge
    img2 = rng.uniform(0, 1000, (nz, ny, nx)).astype(np.float32)
    ref = ndimage.map_coordinates(img2.astype(np.float64), [sz, sy, sx], order=1, mode="nearest")
    # the oracle rounds its double result to float once: half an ulp at 1000 is 3.1e-5
    assert np.max(np.abs(oracle.warp(img2, field).astype(np.float64) - ref)) < 1e-4
