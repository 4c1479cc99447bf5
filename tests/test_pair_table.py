"""Host logic of the pair matching kernel (no GPU): the lane -> task table must give every candidate row of every
block of a CTA's group to exactly one lane, keep the z-pair warps (rows (dy, 2p), (dy, 2p+1)) and the y-pair warps of
the last candidate plane (rows (dy, 2rz), (dy+1, 2rz); one row per block alone) apart, and keep the LDS.128 row
addresses of a quarter-warp on distinct 16-byte bank groups where the counts allow it
(paper_2308_10868_b200/csrc/nrr_match_pair.cu)."""
import numpy as np
import pytest

import paper_2308_10868_b200 as nrr

SHAPES = [(b, r, rz) for b in (5, 7, 9, 11) for r in (3, 5, 7, 9) for rz in (r,)] + [(7, 5, 3), (5, 3, 0), (9, 7, 1),
                                                                                       ((7, 3), 5, 2), ((11, 1), 9, 9)]


def _decode(tab):
    valid = (tab >> 31) & 1
    single = (tab >> 30) & 1          # y-pair warp: the last candidate plane, p = 1 if the row dy+1 belongs to the task
    g = (tab >> 16) & 0xFF
    dy = (tab >> 8) & 0xFF
    p = tab & 0xFF
    return valid.astype(bool), single.astype(bool), g.astype(int), dy.astype(int), p.astype(int)


@pytest.mark.parametrize("b,r,rz", SHAPES)
def test_every_candidate_row_has_exactly_one_lane(b, r, rz):
    b, bz = b if isinstance(b, tuple) else (b, b)
    tab, info = nrr.nrr_bm_pair_task_table((b, b, bz), (r, r, rz))
    valid, single, g, dy, p = _decode(tab)
    w, wz = 2 * r + 1, 2 * rz + 1
    assert info["threads"] == len(tab) and len(tab) % 32 == 0 and len(tab) <= 512
    assert info["smem_bytes"] <= 227 * 1024
    rows = []
    for v, s, gg, d, pp in zip(valid, single, g, dy, p):
        if not v:
            continue
        assert gg < info["blocks_per_cta"] and d < w
        if s:
            assert pp in (0, 1)
            rows.append((gg, d, wz - 1))
            if pp:
                assert d + 1 < w
                rows.append((gg, d + 1, wz - 1))
        else:
            assert 2 * pp + 1 <= wz - 2 + 1 and 2 * pp + 1 < wz
            rows += [(gg, d, 2 * pp), (gg, d, 2 * pp + 1)]
    want = sorted((gg, d, z) for gg in range(info["blocks_per_cta"]) for d in range(w) for z in range(wz))
    assert sorted(rows) == want                                   # each (block, dy, dz) row once, none missing
    # the role bit is uniform over a warp (the kernel branches on it per warp)
    for wi in range(len(tab) // 32):
        assert len(set(single[wi * 32:(wi + 1) * 32])) == 1


@pytest.mark.parametrize("b,r,rz", SHAPES)
def test_schedulers_are_balanced_and_quarter_warps_mostly_conflict_free(b, r, rz):
    b, bz = b if isinstance(b, tuple) else (b, b)
    tab, info = nrr.nrr_bm_pair_task_table((b, b, bz), (r, r, rz))
    valid, single, g, dy, p = _decode(tab)
    nw = len(tab) // 32
    wz = 2 * rz + 1
    # every warp carries two candidate rows per lane, whatever its role: at most one row per block is without a partner
    for gg in range(info["blocks_per_cta"]):
        alone = [i for i in range(len(tab)) if valid[i] and single[i] and g[i] == gg and p[i] == 0]
        assert len(alone) == 1
    # the y-pair warps come last, so that the z-pair warps fill the scheduler slots first (warp w issues from w % 4)
    roles = [bool(single[wi * 32]) for wi in range(nw)]
    assert roles == sorted(roles)
    # shared-memory wavefronts of one LDS.128 of moving voxels: per quarter-warp, the largest number of lanes whose
    # row address falls into the same 16-byte bank group (address in 16-byte units: base + P4*dy + PLANE4*dz)
    p4 = info["pitch"] // 4
    plane4 = p4 * info["rows_per_plane"]
    assert p4 % 2 == 1 and (info["union_stride"] // 16) % 8 == 0
    wavefronts = quarters = 0
    for q in range(0, len(tab), 8):
        lanes = [i for i in range(q, q + 8) if valid[i]]
        if not lanes:
            continue
        res = [(p4 * dy[i] + plane4 * ((wz - 1) if single[i] else 2 * p[i])) % 8 for i in lanes]
        wavefronts += max(np.bincount(res, minlength=8))
        quarters += 1
    assert wavefronts <= 1.25 * quarters, (wavefronts, quarters)


def test_config3_numbers_quoted_in_design_md():
    tab, info = nrr.nrr_bm_pair_task_table((7, 7, 7), (5, 5, 5))
    valid, single, g, dy, p = _decode(tab)
    assert info["blocks_per_cta"] == 4 and info["threads"] == 256 and info["pitch"] == 20
    assert 2 * (info["smem_bytes"] + 1024) <= 228 * 1024          # two CTAs per SM
    assert int(valid.sum()) == 4 * (55 + 6)                       # 55 z-pairs and 5 y-pairs + 1 row alone per block
    assert [wi for wi in range(8) if single[wi * 32]] == [7]       # 8 warps of 2 row-units: two per scheduler
    # the six y-pair tasks of a block start at rows 0, 2, 4, 6 (alone), 7, 9: distinct bank groups for pitch 5 x 16 B
    ys = sorted((int(dy[i]), int(p[i])) for i in range(len(tab)) if valid[i] and single[i] and g[i] == 0)
    assert ys == [(0, 1), (2, 1), (4, 1), (6, 0), (7, 1), (9, 1)]
