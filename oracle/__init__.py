"""CPU oracle (TEST INFRASTRUCTURE, NOT PRODUCT) -- ctypes front-end of oracle/nrr_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares nothing with paper_2308_10868_b200/ and never imports it.

The C file is compiled on first use with gcc (-O2 -ffp-contract=off -fopenmp) into oracle/build/.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nrr_oracle.c")
_BUILD = os.path.join(_HERE, "build")
# NRR_ORACLE_SANITIZE=1 (tests/test_oracle_sanitized.py): the same source under AddressSanitizer + UBSan
_SANITIZE = os.environ.get("NRR_ORACLE_SANITIZE", "0") == "1"
_SO = os.path.join(_BUILD, "libnrr_oracle_san.so" if _SANITIZE else "libnrr_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/nrr_oracle.c -> oracle/build/libnrr_oracle.so (idempotent)."""
    os.makedirs(_BUILD, exist_ok=True)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        if _SANITIZE:
            cmd[1:2] = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    c_int_p = ctypes.POINTER(ctypes.c_int)
    c_dbl_p = ctypes.POINTER(ctypes.c_double)
    c_flt_p = ctypes.POINTER(ctypes.c_float)
    c_u8_p = ctypes.POINTER(ctypes.c_ubyte)
    lib.nrr_oracle_variance_f32.restype = ctypes.c_double
    lib.nrr_oracle_variance_f32.argtypes = [c_flt_p, ctypes.c_long]
    lib.nrr_oracle_ncc_f32.restype = ctypes.c_double
    lib.nrr_oracle_ncc_f32.argtypes = [c_flt_p, c_flt_p, ctypes.c_long]
    lib.nrr_oracle_variance.restype = ctypes.c_double
    lib.nrr_oracle_variance.argtypes = [c_dbl_p, ctypes.c_long]
    lib.nrr_oracle_ncc.restype = ctypes.c_double
    lib.nrr_oracle_ncc.argtypes = [c_dbl_p, c_dbl_p, ctypes.c_long]
    lib.nrr_oracle_count.restype = ctypes.c_int
    lib.nrr_oracle_count.argtypes = [ctypes.c_long, ctypes.c_double]
    lib.nrr_oracle_grid.restype = None
    lib.nrr_oracle_grid.argtypes = [c_int_p, c_int_p, c_int_p, c_int_p]
    lib.nrr_oracle_select.restype = ctypes.c_int
    lib.nrr_oracle_select.argtypes = [c_flt_p, c_int_p, c_int_p, c_int_p, ctypes.c_double, c_u8_p,
                                      c_int_p, ctypes.c_int, c_int_p, c_dbl_p, c_int_p, c_dbl_p]
    lib.nrr_oracle_select_pruned.restype = ctypes.c_int
    lib.nrr_oracle_select_pruned.argtypes = [c_flt_p, c_int_p, c_int_p, c_int_p, ctypes.c_double, c_u8_p, ctypes.c_int,
                                             c_int_p, ctypes.c_int, c_int_p, c_dbl_p, c_int_p]
    lib.nrr_oracle_warp.restype = ctypes.c_int
    lib.nrr_oracle_warp.argtypes = [c_flt_p, c_int_p, c_flt_p, c_flt_p]
    lib.nrr_oracle_match.restype = ctypes.c_int
    lib.nrr_oracle_match.argtypes = [c_flt_p, c_flt_p, c_int_p, c_int_p, ctypes.c_int, c_int_p, c_int_p,
                                     c_int_p, c_dbl_p, c_dbl_p, c_int_p, ctypes.c_int]
    lib.nrr_oracle_ncc_at.restype = ctypes.c_double
    lib.nrr_oracle_ncc_at.argtypes = [c_flt_p, c_flt_p, c_int_p, c_int_p, c_int_p, c_int_p]
    lib.nrr_oracle_max_threads.restype = ctypes.c_int
    lib.nrr_oracle_max_threads.argtypes = []
    _lib = lib
    return lib


def _i3(t):
    return (ctypes.c_int * 3)(int(t[0]), int(t[1]), int(t[2]))


def _f32(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


def _ptr(a: np.ndarray, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def _dims_of(vol: np.ndarray) -> Tuple[int, int, int]:
    nz, ny, nx = vol.shape
    return (nx, ny, nz)


def variance(values) -> float:
    """Population variance of a flat array."""
    a = np.ascontiguousarray(values, dtype=np.float64).ravel()
    return float(_load().nrr_oracle_variance(_ptr(a, ctypes.c_double), a.size))


def ncc(a, b) -> float:
    """NCC of two equally long arrays."""
    a = np.ascontiguousarray(a, dtype=np.float64).ravel()
    b = np.ascontiguousarray(b, dtype=np.float64).ravel()
    if a.size != b.size:
        raise ValueError("length mismatch")
    return float(_load().nrr_oracle_ncc(_ptr(a, ctypes.c_double), _ptr(b, ctypes.c_double), a.size))


def count(n_candidates: int, frac: float) -> int:
    """K = floor(0.5 + N*frac)."""
    return int(_load().nrr_oracle_count(int(n_candidates), float(frac)))


def grid(dims, block, stride) -> Tuple[int, int, int]:
    g = (ctypes.c_int * 3)()
    _load().nrr_oracle_grid(_i3(dims), _i3(block), _i3(stride), g)
    return (g[0], g[1], g[2])


def select(fixed: np.ndarray, block, stride, frac: float, mask: Optional[np.ndarray] = None):
    """Returns dict(centres int32 [K][3], var float64 [K], n_candidates, margin)."""
    fixed = _f32(fixed)
    dims = _dims_of(fixed)
    g = grid(dims, block, stride)
    cap = max(1, g[0] * g[1] * g[2])
    centres = np.empty((cap, 3), dtype=np.int32)
    var = np.empty(cap, dtype=np.float64)
    n = ctypes.c_int(0)
    ncand = ctypes.c_int(0)
    margin = ctypes.c_double(0.0)
    mptr = None
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        if mask.shape != fixed.shape:
            raise ValueError("mask shape mismatch")
        mptr = _ptr(mask, ctypes.c_ubyte)
    rc = _load().nrr_oracle_select(_ptr(fixed, ctypes.c_float), _i3(dims), _i3(block), _i3(stride),
                                   float(frac), mptr, _ptr(centres, ctypes.c_int), cap,
                                   ctypes.byref(n), _ptr(var, ctypes.c_double), ctypes.byref(ncand),
                                   ctypes.byref(margin))
    if rc != 0:
        raise RuntimeError("nrr_oracle_select failed: %d" % rc)
    k = n.value
    return {"centres": centres[:k].copy(), "var": var[:k].copy(), "n_candidates": ncand.value,
            "margin": margin.value}


def select_pruned(fixed: np.ndarray, block, stride, frac: float, mask: Optional[np.ndarray] = None,
                  connectivity: int = 6):
    """Selection under the paper's connectivity pattern (reading Q20: greedy in (variance desc,
    index asc) order on the candidate grid).  Returns dict(centres int32 [n][3], var float64 [n], n_candidates)."""
    fixed = _f32(fixed)
    dims = _dims_of(fixed)
    g = grid(dims, block, stride)
    cap = max(1, g[0] * g[1] * g[2])
    centres = np.empty((cap, 3), dtype=np.int32)
    var = np.empty(cap, dtype=np.float64)
    n = ctypes.c_int(0)
    ncand = ctypes.c_int(0)
    mptr = None
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        if mask.shape != fixed.shape:
            raise ValueError("mask shape mismatch")
        mptr = _ptr(mask, ctypes.c_ubyte)
    rc = _load().nrr_oracle_select_pruned(_ptr(fixed, ctypes.c_float), _i3(dims), _i3(block), _i3(stride),
                                          float(frac), mptr, int(connectivity), _ptr(centres, ctypes.c_int), cap,
                                          ctypes.byref(n), _ptr(var, ctypes.c_double), ctypes.byref(ncand))
    if rc != 0:
        raise RuntimeError("nrr_oracle_select_pruned failed: %d" % rc)
    k = n.value
    return {"centres": centres[:k].copy(), "var": var[:k].copy(), "n_candidates": ncand.value}


def match(fixed: np.ndarray, moving: np.ndarray, centres: np.ndarray, block, window, nthreads: int = 0):
    """Returns dict(disp int32 [n][3], ncc float64 [n], gap float64 [n], nvalid int32 [n])."""
    fixed = _f32(fixed)
    moving = _f32(moving)
    if fixed.shape != moving.shape:
        raise ValueError("volume shape mismatch")
    dims = _dims_of(fixed)
    centres = np.ascontiguousarray(centres, dtype=np.int32).reshape(-1, 3)
    n = centres.shape[0]
    disp = np.zeros((n, 3), dtype=np.int32)
    val = np.zeros(n, dtype=np.float64)
    gap = np.zeros(n, dtype=np.float64)
    nvalid = np.zeros(n, dtype=np.int32)
    rc = _load().nrr_oracle_match(_ptr(fixed, ctypes.c_float), _ptr(moving, ctypes.c_float), _i3(dims),
                                  _ptr(centres, ctypes.c_int), n, _i3(block), _i3(window),
                                  _ptr(disp, ctypes.c_int), _ptr(val, ctypes.c_double),
                                  _ptr(gap, ctypes.c_double), _ptr(nvalid, ctypes.c_int), int(nthreads))
    if rc != 0:
        raise RuntimeError("nrr_oracle_match failed: %d" % rc)
    return {"disp": disp, "ncc": val, "gap": gap, "nvalid": nvalid}


def warp(image: np.ndarray, field: np.ndarray) -> np.ndarray:
    """out(p) = trilinear(image, clamp(p + v(p))); field is float32 [3][nz][ny][nx], components (vx, vy, vz) in voxels
    (reading Q21)."""
    image = _f32(image)
    field = np.ascontiguousarray(field, dtype=np.float32)
    if field.shape != (3,) + image.shape:
        raise ValueError("field must be [3][nz][ny][nx]")
    out = np.empty_like(image)
    rc = _load().nrr_oracle_warp(_ptr(image, ctypes.c_float), _i3(_dims_of(image)), _ptr(field, ctypes.c_float),
                                 _ptr(out, ctypes.c_float))
    if rc != 0:
        raise RuntimeError("nrr_oracle_warp failed: %d" % rc)
    return out


def ncc_at(fixed: np.ndarray, moving: np.ndarray, centre, block, d) -> float:
    """NCC of one (block, displacement) pair; nan if the skip rule removes the candidate."""
    fixed = _f32(fixed)
    moving = _f32(moving)
    dims = _dims_of(fixed)
    return float(_load().nrr_oracle_ncc_at(_ptr(fixed, ctypes.c_float), _ptr(moving, ctypes.c_float),
                                           _i3(dims), _i3(centre), _i3(block), _i3(d)))


def max_threads() -> int:
    return int(_load().nrr_oracle_max_threads())
