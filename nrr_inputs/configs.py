"""Parameter sets of the five BASELINE.json workloads (plus the readings of SURVEY.md 8(c) Q10).

All triples are in (x, y, z) order, matching the C ABI. Volumes are stored [z][y][x] (x fastest).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

Triple = Tuple[int, int, int]


@dataclass(frozen=True)
class Config:
    name: str
    dims: Triple                 # (nx, ny, nz)
    block: Triple                # full odd edge length per axis
    stride: Triple
    window: Triple               # displacement half-range r per axis; candidates = prod(2r+1)
    frac: float                  # selection fraction F_s
    sigma: float                 # Gaussian smoothing of the N(0,1) field, voxels
    n_blobs: int
    mask_radius: Optional[float]  # spherical mask radius in voxels, None = no mask
    moving: str                  # "shift" | "rbf"
    shift: Triple = (0, 0, 0)    # for moving == "shift"
    rbf_amplitude: float = 0.0   # max |u| in voxels for moving == "rbf"
    noise: str = "gauss"         # "gauss" | "rician" | "none"
    noise_sigma: float = 0.0
    seed: int = 0

    @property
    def n_candidates(self) -> int:
        rx, ry, rz = self.window
        return (2 * rx + 1) * (2 * ry + 1) * (2 * rz + 1)


CONFIGS = {
    # BASELINE.json configs[0]
    "tiny": Config("tiny", (64, 64, 32), (5, 5, 5), (5, 5, 5), (3, 3, 3), 0.30,
                   sigma=2.0, n_blobs=0, mask_radius=None, moving="shift", shift=(2, -1, 1),
                   noise="gauss", noise_sigma=10.0),
    # configs[1]
    "intraop": Config("intraop", (256, 256, 60), (7, 7, 7), (7, 7, 7), (5, 5, 3), 0.20,
                      sigma=3.0, n_blobs=4, mask_radius=110.0, moving="rbf", rbf_amplitude=5.0,
                      noise="gauss", noise_sigma=15.0),
    # configs[2] -- the config BASELINE.json's metric is quoted on (256x256x124)
    "fullres": Config("fullres", (256, 256, 124), (7, 7, 7), (5, 5, 5), (5, 5, 5), 0.25,
                      sigma=3.0, n_blobs=4, mask_radius=110.0, moving="rbf", rbf_amplitude=8.0,
                      noise="rician", noise_sigma=20.0),
    # configs[3]
    "highres": Config("highres", (512, 512, 176), (9, 9, 9), (6, 6, 6), (7, 7, 7), 0.20,
                      sigma=3.0, n_blobs=6, mask_radius=None, moving="rbf", rbf_amplitude=12.0,
                      noise="gauss", noise_sigma=10.0),
}


@dataclass(frozen=True)
class BatchSetting:
    block: Triple
    window: Triple
    frac: float
    stride: Triple = (5, 5, 5)


def batch_settings() -> List[BatchSetting]:
    """configs[4]: 32 settings = block {5,7,9,11} x window half-width {3,5,7,9} x frac {0.1,0.3},
    all on the "fullres" pair with its mask and stride 5."""
    out = []
    for b in (5, 7, 9, 11):
        for w in (3, 5, 7, 9):
            for f in (0.10, 0.30):
                out.append(BatchSetting((b, b, b), (w, w, w), f))
    return out


def get_config(name: str) -> Config:
    return CONFIGS[name]
