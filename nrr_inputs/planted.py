"""Planted-displacement inputs: for block i an exact copy of the fixed block sits at displacement d_i in an
otherwise unrelated noise volume, with the d_i running over every (dy, dz) candidate row and every dx of the
window.  Input generation only (no method arithmetic): the expected result is the planted d_i with NCC = 1."""
import numpy as np


def planted_pair(b: int, r: int, rz: int, seed: int = 123, copies: int = 2):
    """Returns (fixed, moving, centres int32 [n][3], planted int32 [n][3]) for cubic blocks of edge b and the
    window (r, r, rz).  nx is a multiple of 4."""
    w, wz = 2 * r + 1, 2 * rz + 1
    n_min = copies * w * wz
    px, pz = b + 2 * r + 1, b + 2 * rz + 1            # windows of neighbouring blocks are disjoint
    gx = 7
    gy = 6
    gz = -(-n_min // (gx * gy))
    nx = -(-(gx * px + 2) // 4) * 4
    dims = (nx, gy * px + 4, gz * pz + 4)
    rng = np.random.default_rng(seed)
    fixed = rng.uniform(0, 1000, size=dims[::-1]).astype(np.float32)
    moving = rng.uniform(0, 1000, size=dims[::-1]).astype(np.float32)
    centres, want = [], []
    i = 0
    for kz in range(gz):
        for ky in range(gy):
            for kx in range(gx):
                o = np.array([kx * px + r, ky * px + r, kz * pz + rz])
                d = np.array([(i * 4) % w - r, i % w - r, (i // w) % wz - rz])      # (dx, dy, dz)
                p = o + d
                moving[p[2]:p[2] + b, p[1]:p[1] + b, p[0]:p[0] + b] = fixed[o[2]:o[2] + b, o[1]:o[1] + b, o[0]:o[0] + b]
                centres.append(o + (b - 1) // 2)
                want.append(d)
                i += 1
    return fixed, moving, np.asarray(centres, np.int32), np.asarray(want, np.int32)
