"""Second, independent, naive evaluator (TEST INFRASTRUCTURE) -- pure-Python triple loops for tiny inputs.

It exists to pin oracle/nrr_oracle.c: it is written differently on purpose (exactly-rounded sums via
math.fsum, Pearson's r through the raw-moment identity per candidate, all NCC values collected first
and the arg-max taken afterwards, selection through numpy.lexsort) so that an indexing, sign or
ordering mistake in the C oracle does not repeat here.  Same readings of the paper (Q1-Q15).
Citations: variance/selection PAPER.md:231-236, 376; NCC PAPER.md:243-246; search PAPER.md:659-667.
"""
from __future__ import annotations

import math
from typing import Optional

import numpy as np


def _block_values(vol: np.ndarray, origin, block):
    ox, oy, oz = origin
    bx, by, bz = block
    vals = []
    for z in range(oz, oz + bz):
        for y in range(oy, oy + by):
            for x in range(ox, ox + bx):
                vals.append(float(vol[z, y, x]))
    return vals


def variance(vals) -> float:
    n = len(vals)
    mean = math.fsum(vals) / n
    return math.fsum((v - mean) ** 2 for v in vals) / n


def ncc(a, b) -> float:
    """Pearson correlation through centred moments with exactly-rounded sums; 0 if either is constant."""
    n = len(a)
    ma = math.fsum(a) / n
    mb = math.fsum(b) / n
    saa = math.fsum((x - ma) * (x - ma) for x in a)
    sbb = math.fsum((y - mb) * (y - mb) for y in b)
    if saa == 0.0 or sbb == 0.0:
        return 0.0
    sab = math.fsum((x - ma) * (y - mb) for x, y in zip(a, b))
    return sab / math.sqrt(saa * sbb)


def select(fixed: np.ndarray, block, stride, frac: float, mask: Optional[np.ndarray] = None):
    nz, ny, nx = fixed.shape
    bx, by, bz = block
    sx, sy, sz = stride
    cents, vars_ = [], []
    oz = 0
    while oz + bz <= nz:
        oy = 0
        while oy + by <= ny:
            ox = 0
            while ox + bx <= nx:
                c = (ox + bx // 2, oy + by // 2, oz + bz // 2)
                if mask is None or mask[c[2], c[1], c[0]] != 0:
                    cents.append(c)
                    vars_.append(variance(_block_values(fixed, (ox, oy, oz), block)))
                ox += sx
            oy += sy
        oz += sz
    n = len(cents)
    k = int(math.floor(0.5 + n * frac))
    idx = np.arange(n)
    order = np.lexsort((idx, -np.asarray(vars_, dtype=np.float64)))  # primary: variance desc; then index asc
    keep = np.sort(order[:k])
    return {"centres": np.asarray([cents[i] for i in keep], dtype=np.int32).reshape(-1, 3),
            "var": np.asarray([vars_[i] for i in keep], dtype=np.float64), "n_candidates": n}


def match(fixed: np.ndarray, moving: np.ndarray, centres, block, window):
    nz, ny, nx = fixed.shape
    bx, by, bz = block
    rx, ry, rz = window
    disp, best_ncc, gaps = [], [], []
    for c in np.asarray(centres).reshape(-1, 3):
        o = (int(c[0]) - bx // 2, int(c[1]) - by // 2, int(c[2]) - bz // 2)
        f = _block_values(fixed, o, block)
        scores = np.full((2 * rz + 1, 2 * ry + 1, 2 * rx + 1), -np.inf)
        for dx in range(-rx, rx + 1):          # deliberately x-outermost: order must not matter
            for dy in range(-ry, ry + 1):
                for dz in range(-rz, rz + 1):
                    p = (o[0] + dx, o[1] + dy, o[2] + dz)
                    if min(p) < 0 or p[0] + bx > nx or p[1] + by > ny or p[2] + bz > nz:
                        continue
                    scores[dz + rz, dy + ry, dx + rx] = ncc(f, _block_values(moving, p, block))
        flat = scores.ravel()                   # linear candidate index, x fastest
        i = int(np.argmax(flat))                # first occurrence = lowest index among equal maxima
        kz, rem = divmod(i, (2 * ry + 1) * (2 * rx + 1))
        ky, kx = divmod(rem, 2 * rx + 1)
        disp.append((kx - rx, ky - ry, kz - rz))
        best_ncc.append(float(flat[i]))
        rest = np.delete(flat, i)
        rest = rest[np.isfinite(rest)]
        gaps.append(float(flat[i] - rest.max()) if rest.size else math.inf)
    return {"disp": np.asarray(disp, dtype=np.int32).reshape(-1, 3),
            "ncc": np.asarray(best_ncc, dtype=np.float64), "gap": np.asarray(gaps, dtype=np.float64)}
