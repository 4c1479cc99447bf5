"""Property tests (-m "not gpu"): random volume shapes, block / stride / window triples, masks and options through the
emulated library (tests/cuda_emul) against the oracle.  The point is the shapes nobody wrote down: ragged tails, blocks
as large as the volume, windows wider than the volume, nx % 4 != 0 (plain staging) vs == 0 (TMA), partial last CTAs of
every grouping -- an index slip in any of them is an out-of-bounds access, i.e. a fault on a GPU."""
import os

import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings
from hypothesis import strategies as st

import oracle
import _emul
from _parity import assert_match_parity, assert_select_parity

# NRR_PROPERTY_EXAMPLES=<n>: a longer, randomised hunt (the suite's default is small and derandomised)
HUNT = int(os.environ.get("NRR_PROPERTY_EXAMPLES", "0"))
OPTIONS = ("force_rows", "force_generic", "disable_tma", "pair_blocks_per_cta", "select_generic", "boxstat_generic")


@pytest.fixture(autouse=True)
def _defaults():
    for name in OPTIONS:
        _emul.set_option(name, 0)
    yield
    for name in OPTIONS:
        _emul.set_option(name, 0)


def _volume(dims, seed):
    from scipy import ndimage
    nx, ny, nz = dims
    v = ndimage.gaussian_filter(np.random.default_rng(seed).standard_normal((nz, ny, nx)), 1.2, mode="reflect")
    return ((v - v.min()) / max(v.max() - v.min(), 1e-9) * 1000.0).astype(np.float32)


odd = lambda lo, hi: st.integers(lo, hi).map(lambda k: 2 * k + 1)


@st.composite
def generic_case(draw):
    block = (draw(odd(0, 3)), draw(odd(0, 3)), draw(odd(0, 2)))
    dims = tuple(draw(st.integers(b, b + 9)) for b in block)
    stride = tuple(draw(st.integers(1, 4)) for _ in range(3))
    window = tuple(draw(st.integers(0, 3)) for _ in range(3))
    return dims, block, stride, window, draw(st.sampled_from([0.2, 0.5, 1.0])), draw(st.booleans()), draw(st.integers(0, 10 ** 6))


@settings(max_examples=HUNT or 40, deadline=None, suppress_health_check=list(HealthCheck), derandomize=not HUNT, database=None)
@given(generic_case())
def test_any_shape_select_and_match_against_the_oracle(case):
    dims, block, stride, window, frac, use_mask, seed = case
    fixed = _volume(dims, seed)
    moving = _volume(dims, seed + 1) * 0.3 + fixed * 0.7
    mask = (np.random.default_rng(seed + 2).uniform(size=fixed.shape) < 0.7).astype(np.uint8) if use_mask else None
    ora_sel = oracle.select(fixed, block, stride, frac, mask)
    for generic in (0, 1):
        _emul.set_option("select_generic", generic)
        blocks, n, ncand, var = _emul.select(fixed, block, stride, frac, mask)
        assert_select_parity(blocks, n, ncand, ora_sel, var)
    _emul.set_option("select_generic", 0)
    if len(ora_sel["centres"]) == 0:
        return
    ora = oracle.match(fixed, moving.astype(np.float32), ora_sel["centres"], block, window)
    d, s = _emul.match(fixed, moving.astype(np.float32), ora_sel["centres"], block, window)
    assert_match_parity(d, s, ora, str(case))
    rb, rd, rs = _emul.register(fixed, moving.astype(np.float32), block, stride, window, frac, mask)
    assert np.array_equal(rb, ora_sel["centres"]) and np.array_equal(rd, d) and np.array_equal(rs, s)


@st.composite
def fast_case(draw):
    b = draw(st.sampled_from([5, 7, 9, 11]))
    r = draw(st.sampled_from([3, 5]))
    bz = draw(st.sampled_from([b, 3, 5]))
    rz = draw(st.integers(0, 3))
    nx = draw(st.integers(b + 2, b + 14))
    dims = (nx, draw(st.integers(b + 1, b + 10)), draw(st.integers(bz, bz + 8)))
    stride = (draw(st.integers(2, 6)), draw(st.integers(2, 6)), draw(st.integers(1, 4)))
    g = draw(st.sampled_from([0, 0, 1, 3, 5]))
    return dims, (b, b, bz), stride, (r, r, rz), g, draw(st.booleans()), draw(st.integers(0, 10 ** 6))


@settings(max_examples=HUNT or 30, deadline=None, suppress_health_check=list(HealthCheck), derandomize=not HUNT, database=None)
@given(fast_case())
def test_any_shape_through_the_pair_kernel_and_a_plan(case):
    dims, block, stride, window, g, no_tma, seed = case
    fixed = _volume(dims, seed)
    moving = (_volume(dims, seed + 1) * 0.2 + np.roll(fixed, 1, axis=2) * 0.8).astype(np.float32)
    sel = oracle.select(fixed, block, stride, 0.6, None)
    if len(sel["centres"]) == 0:
        return
    _emul.set_option("pair_blocks_per_cta", g)
    _emul.set_option("disable_tma", 1 if no_tma else 0)
    info = _emul.match_info(dims, block, window)
    ora = oracle.match(fixed, moving, sel["centres"], block, window)
    d, s = _emul.match(fixed, moving, sel["centres"], block, window)
    assert_match_parity(d, s, ora, "%s kernel %d" % (case, info["kernel"]))
    plan = _emul.Plan(fixed, block, stride, window, 0.6, None, host=True)
    _emul.set_option("plan_slabs", 3)
    pd, ps = plan.match_host(moving)
    _emul.set_option("plan_slabs", 4)
    plan.destroy()
    assert np.array_equal(pd, d) and np.array_equal(ps, s)
