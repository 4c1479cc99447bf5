"""Thin ctypes binding of libnrr_bm.so (include/nrr_bm.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch appears here only as the owner of
device memory and streams.  There is no CPU fallback: if the library is missing or no CUDA device is
present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnrr_bm.so")

NRR_OK = 0
NRR_E_NULL, NRR_E_DIMS, NRR_E_BLOCK, NRR_E_STRIDE, NRR_E_WINDOW, NRR_E_FRAC = -1, -2, -3, -4, -5, -6
NRR_E_CAPACITY, NRR_E_BOUNDS, NRR_E_SMEM, NRR_E_CUDA, NRR_E_ARG, NRR_E_DEVICE, NRR_E_NOCONV = -7, -8, -9, -10, -11, -12, -13

EXPORTS = [
    "nrr_bm_select_blocks", "nrr_bm_select_blocks_pruned", "nrr_bm_select_blocks_pruned_host", "nrr_bm_match", "nrr_bm_register", "nrr_bm_check_async_error", "nrr_bm_moving_stats", "nrr_bm_moving_stats_host", "nrr_bm_warp", "nrr_bm_warp_host",
    "nrr_bm_select_blocks_host", "nrr_bm_match_host", "nrr_bm_register_host",
    "nrr_bm_profile_enable", "nrr_bm_profile_read", "nrr_bm_launch_count", "nrr_bm_match_info", "nrr_bm_match_info_n",
    "nrr_bm_capacity_bound", "nrr_bm_plan_create", "nrr_bm_plan_create_host", "nrr_bm_plan_info", "nrr_bm_plan_blocks_host",
    "nrr_bm_plan_blocks_device", "nrr_bm_plan_blocks", "nrr_bm_plan_match", "nrr_bm_plan_match_range", "nrr_bm_plan_match_host", "nrr_bm_plan_destroy",
    "nrr_bm_register_batch",
    "nrr_bm_fem_create", "nrr_bm_fem_info", "nrr_bm_fem_solve", "nrr_bm_fem_solve_host", "nrr_bm_fem_dense_field",
    "nrr_bm_fem_dense_field_host", "nrr_bm_fem_destroy",
    "nrr_bm_fp32_peak", "nrr_bm_fp32_microbench", "nrr_bm_pair_task_table", "nrr_bm_set_option", "nrr_bm_last_error", "nrr_bm_status_string", "nrr_bm_version",
]


class NrrError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s (%d): %s" % (_status_name(status), status, message))
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libnrr_bm.so (built in-tree by paper_2308_10868_b200/build.py). Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libnrr_bm.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "or `python paper_2308_10868_b200/build.py` (there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    i3 = ctypes.POINTER(ctypes.c_int)
    L.nrr_bm_select_blocks.restype = ci
    L.nrr_bm_select_blocks.argtypes = [vp, i3, i3, i3, cd, vp, vp, ci, i3, vp, i3, vp]
    L.nrr_bm_match.restype = ci
    L.nrr_bm_match.argtypes = [vp, vp, i3, vp, ci, i3, i3, vp, vp, vp]
    L.nrr_bm_select_blocks_pruned.restype = ci
    L.nrr_bm_select_blocks_pruned.argtypes = [vp, i3, i3, i3, cd, vp, ci, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci), vp]
    L.nrr_bm_select_blocks_pruned_host.restype = ci
    L.nrr_bm_select_blocks_pruned_host.argtypes = [vp, i3, i3, i3, cd, vp, ci, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci)]
    L.nrr_bm_register.restype = ci
    L.nrr_bm_register.argtypes = [vp, vp, i3, i3, i3, i3, cd, vp, vp, ci, vp, vp, vp, vp]
    L.nrr_bm_warp.restype = ci
    L.nrr_bm_warp.argtypes = [vp, i3, vp, vp, vp]
    L.nrr_bm_warp_host.restype = ci
    L.nrr_bm_warp_host.argtypes = [vp, i3, vp, vp]
    L.nrr_bm_moving_stats.restype = ci
    L.nrr_bm_moving_stats.argtypes = [vp, i3, i3, vp, vp]
    L.nrr_bm_moving_stats_host.restype = ci
    L.nrr_bm_moving_stats_host.argtypes = [vp, i3, i3, vp]
    L.nrr_bm_check_async_error.restype = ci
    L.nrr_bm_check_async_error.argtypes = [vp]
    L.nrr_bm_select_blocks_host.restype = ci
    L.nrr_bm_select_blocks_host.argtypes = [vp, i3, i3, i3, cd, vp, vp, ci, i3, vp, i3]
    L.nrr_bm_match_host.restype = ci
    L.nrr_bm_match_host.argtypes = [vp, vp, i3, vp, ci, i3, i3, vp, vp]
    L.nrr_bm_register_host.restype = ci
    L.nrr_bm_register_host.argtypes = [vp, vp, i3, i3, i3, i3, cd, vp, vp, ci, i3, vp, vp]
    L.nrr_bm_capacity_bound.restype = ci
    L.nrr_bm_capacity_bound.argtypes = [i3, i3, i3, cd, i3, i3]
    pp = ctypes.POINTER(vp)
    L.nrr_bm_plan_create.restype = ci
    L.nrr_bm_plan_create.argtypes = [vp, i3, i3, i3, i3, cd, vp, ci, vp, pp]
    L.nrr_bm_plan_create_host.restype = ci
    L.nrr_bm_plan_create_host.argtypes = [vp, i3, i3, i3, i3, cd, vp, ci, pp]
    L.nrr_bm_plan_info.restype = ci
    L.nrr_bm_plan_info.argtypes = [vp, i3, i3]
    L.nrr_bm_plan_blocks_host.restype = ci
    L.nrr_bm_plan_blocks_host.argtypes = [vp, vp, vp]
    L.nrr_bm_plan_blocks.restype = ci
    L.nrr_bm_plan_blocks.argtypes = [vp, vp, vp, vp]
    L.nrr_bm_plan_blocks_device.restype = vp
    L.nrr_bm_plan_blocks_device.argtypes = [vp]
    L.nrr_bm_plan_match.restype = ci
    L.nrr_bm_plan_match.argtypes = [vp, vp, vp, vp, vp]
    L.nrr_bm_plan_match_range.restype = ci
    L.nrr_bm_plan_match_range.argtypes = [vp, vp, ci, ci, vp, vp, vp]
    L.nrr_bm_plan_match_host.restype = ci
    L.nrr_bm_plan_match_host.argtypes = [vp, vp, vp, vp]
    L.nrr_bm_plan_destroy.restype = ci
    L.nrr_bm_plan_destroy.argtypes = [vp]
    L.nrr_bm_register_batch.restype = ci
    L.nrr_bm_register_batch.argtypes = [vp, vp, i3, vp, vp, ci, pp, i3, vp, pp, pp, vp]
    L.nrr_bm_fem_create.restype = ci
    L.nrr_bm_fem_create.argtypes = [i3, i3, cd, cd, pp]
    L.nrr_bm_fem_info.restype = ci
    L.nrr_bm_fem_info.argtypes = [vp, i3, i3]
    L.nrr_bm_fem_solve.restype = ci
    L.nrr_bm_fem_solve.argtypes = [vp, vp, vp, vp, ci, cd, ci, cd, ci, vp, i3, vp]
    L.nrr_bm_fem_solve_host.restype = ci
    L.nrr_bm_fem_solve_host.argtypes = [vp, vp, vp, vp, ci, cd, ci, cd, ci, vp, i3]
    L.nrr_bm_fem_dense_field.restype = ci
    L.nrr_bm_fem_dense_field.argtypes = [vp, vp, vp, vp]
    L.nrr_bm_fem_dense_field_host.restype = ci
    L.nrr_bm_fem_dense_field_host.argtypes = [vp, vp, vp]
    L.nrr_bm_fem_destroy.restype = ci
    L.nrr_bm_fem_destroy.argtypes = [vp]
    L.nrr_bm_profile_enable.restype = ci
    L.nrr_bm_profile_enable.argtypes = [ci]
    L.nrr_bm_profile_read.restype = ci
    L.nrr_bm_profile_read.argtypes = [ctypes.POINTER(cd), i3]
    L.nrr_bm_launch_count.restype = ctypes.c_longlong
    L.nrr_bm_launch_count.argtypes = [ci]
    L.nrr_bm_match_info.restype = ci
    L.nrr_bm_match_info.argtypes = [i3, i3, i3, i3]
    L.nrr_bm_match_info_n.restype = ci
    L.nrr_bm_match_info_n.argtypes = [i3, i3, i3, ci, i3]
    L.nrr_bm_pair_task_table.restype = ci
    L.nrr_bm_pair_task_table.argtypes = [i3, i3, vp, ci, ctypes.POINTER(ci)]
    L.nrr_bm_fp32_peak.restype = ci
    L.nrr_bm_fp32_peak.argtypes = [ctypes.POINTER(cd), vp]
    L.nrr_bm_fp32_microbench.restype = ci
    L.nrr_bm_fp32_microbench.argtypes = [ctypes.POINTER(cd), vp]
    L.nrr_bm_set_option.restype = ci
    L.nrr_bm_set_option.argtypes = [ctypes.c_char_p, cd]
    L.nrr_bm_last_error.restype = ctypes.c_char_p
    L.nrr_bm_last_error.argtypes = []
    L.nrr_bm_status_string.restype = ctypes.c_char_p
    L.nrr_bm_status_string.argtypes = [ci]
    L.nrr_bm_version.restype = ci
    L.nrr_bm_version.argtypes = []
    _lib = L
    return L


def _status_name(status: int) -> str:
    try:
        return lib().nrr_bm_status_string(int(status)).decode()
    except Exception:  # pragma: no cover
        return "NRR_E_?"


def _check(status: int, allow: Sequence[int] = ()) -> int:
    if status != NRR_OK and status not in allow:
        raise NrrError(status, lib().nrr_bm_last_error().decode())
    return status


def _i3(t) -> ctypes.Array:
    return (ctypes.c_int * 3)(int(t[0]), int(t[1]), int(t[2]))


def _dims_of(vol) -> Tuple[int, int, int]:
    nz, ny, nx = vol.shape
    return (int(nx), int(ny), int(nz))


def _stream_ptr(stream) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _dev(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor (no CPU fallback)" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous %s tensor" % (name, dtype))
    return t


# --------------------------------------------------------------------------------------------- device API
def nrr_bm_select_blocks(fixed, block, stride, frac: float, mask=None, capacity: Optional[int] = None,
                         want_var: bool = False, stream=None):
    """Device form. fixed: CUDA fp32 [nz][ny][nx]; mask: CUDA uint8 same shape or None.
    Returns (blocks int32 CUDA [K][3], K, N[, var float64 CUDA [K]])."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    dims = _dims_of(fixed)
    if mask is not None:
        mask = _dev(mask, torch.uint8, "mask")
        if tuple(mask.shape) != tuple(fixed.shape):
            raise ValueError("mask shape mismatch")
    if capacity is None:
        capacity = 1
        for a in range(3):
            capacity *= max(0, (dims[a] - int(block[a])) // max(1, int(stride[a])) + 1)
        capacity = max(1, capacity)
    out_blocks = torch.empty((capacity, 3), dtype=torch.int32, device=fixed.device)
    out_var = torch.empty((capacity,), dtype=torch.float64, device=fixed.device) if want_var else None
    n = ctypes.c_int(0)
    ncand = ctypes.c_int(0)
    with torch.cuda.device(fixed.device):
        _check(lib().nrr_bm_select_blocks(fixed.data_ptr(), _i3(dims), _i3(block), _i3(stride), float(frac),
                                          mask.data_ptr() if mask is not None else None, out_blocks.data_ptr(),
                                          int(capacity), ctypes.byref(n), out_var.data_ptr() if want_var else None,
                                          ctypes.byref(ncand), _stream_ptr(stream)))
    k = n.value
    if want_var:
        return out_blocks[:k], k, ncand.value, out_var[:k]
    return out_blocks[:k], k, ncand.value


def nrr_bm_select_blocks_pruned(fixed, block, stride, frac: float, mask=None, connectivity: int = 6,
                                capacity: Optional[int] = None, want_var: bool = False, stream=None):
    """Device form of the selection under a connectivity pattern (0, 6, 18, 26). Same returns as nrr_bm_select_blocks."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    dims = _dims_of(fixed)
    if mask is not None:
        mask = _dev(mask, torch.uint8, "mask")
        if tuple(mask.shape) != tuple(fixed.shape):
            raise ValueError("mask shape mismatch")
    if capacity is None:
        capacity = 1
        for a in range(3):
            capacity *= max(0, (dims[a] - int(block[a])) // max(1, int(stride[a])) + 1)
        capacity = max(1, capacity)
    out_blocks = torch.empty((capacity, 3), dtype=torch.int32, device=fixed.device)
    out_var = torch.empty((capacity,), dtype=torch.float64, device=fixed.device) if want_var else None
    n = ctypes.c_int(0)
    ncand = ctypes.c_int(0)
    with torch.cuda.device(fixed.device):
        _check(lib().nrr_bm_select_blocks_pruned(fixed.data_ptr(), _i3(dims), _i3(block), _i3(stride), float(frac),
                                                 mask.data_ptr() if mask is not None else None, int(connectivity),
                                                 out_blocks.data_ptr(), int(capacity), ctypes.byref(n),
                                                 out_var.data_ptr() if want_var else None, ctypes.byref(ncand),
                                                 _stream_ptr(stream)))
    k = n.value
    if want_var:
        return out_blocks[:k], k, ncand.value, out_var[:k]
    return out_blocks[:k], k, ncand.value


def nrr_bm_match(fixed, moving, blocks, block, window, out_disp=None, out_ncc=None, stream=None):
    """Device form, asynchronous. Returns (disp int32 CUDA [n][3], ncc fp32 CUDA [n])."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    moving = _dev(moving, torch.float32, "moving")
    if tuple(fixed.shape) != tuple(moving.shape):
        raise ValueError("volume shape mismatch")
    blocks = _dev(blocks, torch.int32, "blocks")
    n = int(blocks.shape[0])
    if out_disp is None:
        out_disp = torch.empty((n, 3), dtype=torch.int32, device=fixed.device)
    if out_ncc is None:
        out_ncc = torch.empty((n,), dtype=torch.float32, device=fixed.device)
    with torch.cuda.device(fixed.device):
        _check(lib().nrr_bm_match(fixed.data_ptr(), moving.data_ptr(), _i3(_dims_of(fixed)), blocks.data_ptr(), n,
                                  _i3(block), _i3(window), out_disp.data_ptr(), out_ncc.data_ptr(), _stream_ptr(stream)))
    return out_disp, out_ncc


def nrr_bm_register(fixed, moving, block, stride, window, frac: float, mask=None, capacity: Optional[int] = None,
                    out_blocks=None, out_n=None, out_disp=None, out_ncc=None, stream=None):
    """Device form, fully asynchronous: select + match of one pair with no host synchronisation.
    Returns (blocks [capacity][3], n (CUDA int32 scalar tensor: K), disp [capacity][3], ncc [capacity]); rows
    beyond K are untouched.  Read n (e.g. int(n)) only after the work on `stream` may be waited for."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    moving = _dev(moving, torch.float32, "moving")
    if tuple(fixed.shape) != tuple(moving.shape):
        raise ValueError("volume shape mismatch")
    dims = _dims_of(fixed)
    if mask is not None:
        mask = _dev(mask, torch.uint8, "mask")
    if capacity is None:
        capacity = max(1, nrr_bm_capacity_bound(dims, block, stride, frac)[1])
    dev = fixed.device
    if out_blocks is None:
        out_blocks = torch.empty((capacity, 3), dtype=torch.int32, device=dev)
    if out_disp is None:
        out_disp = torch.empty((capacity, 3), dtype=torch.int32, device=dev)
    if out_ncc is None:
        out_ncc = torch.empty((capacity,), dtype=torch.float32, device=dev)
    if out_n is None:
        out_n = torch.empty((), dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        _check(lib().nrr_bm_register(fixed.data_ptr(), moving.data_ptr(), _i3(dims), _i3(block), _i3(stride), _i3(window),
                                     float(frac), mask.data_ptr() if mask is not None else None, out_blocks.data_ptr(),
                                     int(capacity), out_n.data_ptr(), out_disp.data_ptr(), out_ncc.data_ptr(),
                                     _stream_ptr(stream)))
    return out_blocks, out_n, out_disp, out_ncc


def nrr_bm_capacity_bound(dims, block, stride, frac: float) -> Tuple[int, int]:
    """(stride-grid positions, upper bound on K) -- the library's own count rule; no device needed."""
    g, b = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().nrr_bm_capacity_bound(_i3(dims), _i3(block), _i3(stride), float(frac), ctypes.byref(g), ctypes.byref(b)))
    return g.value, b.value


class nrr_bm_setting(ctypes.Structure):
    """One parameter setting of nrr_bm_register_batch (include/nrr_bm.h)."""
    _fields_ = [("block", ctypes.c_int * 3), ("stride", ctypes.c_int * 3), ("window", ctypes.c_int * 3), ("frac", ctypes.c_double)]


def nrr_bm_register_batch(fixed, moving, settings, mask=None, stream=None):
    """One volume pair under many settings in ONE launch sequence (no host synchronisation).  `settings`: objects with
    .block, .stride, .window, .frac.  Returns (results, n) with results[s] = (blocks [cap][3], disp [cap][3], ncc [cap])
    CUDA tensors and n a CUDA int32 tensor [len(settings)] holding K per setting; rows beyond K are untouched."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    moving = _dev(moving, torch.float32, "moving")
    if tuple(fixed.shape) != tuple(moving.shape):
        raise ValueError("volume shape mismatch")
    if mask is not None:
        mask = _dev(mask, torch.uint8, "mask")
    dims = _dims_of(fixed)
    ns = len(settings)
    arr = (nrr_bm_setting * max(1, ns))()
    caps = (ctypes.c_int * max(1, ns))()
    pb, pd, pn = (ctypes.c_void_p * max(1, ns))(), (ctypes.c_void_p * max(1, ns))(), (ctypes.c_void_p * max(1, ns))()
    results = []
    dev = fixed.device
    for i, st in enumerate(settings):
        arr[i].block[:] = [int(v) for v in st.block]
        arr[i].stride[:] = [int(v) for v in st.stride]
        arr[i].window[:] = [int(v) for v in st.window]
        arr[i].frac = float(st.frac)
        cap = max(1, nrr_bm_capacity_bound(dims, st.block, st.stride, st.frac)[1])
        caps[i] = cap
        b = torch.empty((cap, 3), dtype=torch.int32, device=dev)
        d = torch.empty((cap, 3), dtype=torch.int32, device=dev)
        c = torch.empty((cap,), dtype=torch.float32, device=dev)
        pb[i], pd[i], pn[i] = b.data_ptr(), d.data_ptr(), c.data_ptr()
        results.append((b, d, c))
    out_n = torch.zeros((max(1, ns),), dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        _check(lib().nrr_bm_register_batch(fixed.data_ptr(), moving.data_ptr(), _i3(dims),
                                           mask.data_ptr() if mask is not None else None, arr, ns, pb, caps,
                                           out_n.data_ptr(), pd, pn, _stream_ptr(stream)))
    return results, out_n[:ns]


class NrrPlan:
    """Handle of an nrr_bm_plan (include/nrr_bm.h "PLANS").  Keeps the `fixed` tensor alive for the device form."""

    def __init__(self, handle, dims, keep=None):
        self.handle, self.dims, self._keep = handle, dims, keep
        n, ncand = ctypes.c_int(0), ctypes.c_int(0)
        _check(lib().nrr_bm_plan_info(handle, ctypes.byref(n), ctypes.byref(ncand)))
        self.n, self.ncand = n.value, ncand.value

    def __del__(self):
        try:
            nrr_bm_plan_destroy(self)
        except Exception:  # pragma: no cover
            pass


def nrr_bm_plan_create(fixed, block, stride, window, frac: float, mask=None, connectivity: int = 0, stream=None) -> NrrPlan:
    """PRE-OPERATIVE, device form: selection + fixed-block records.  fixed / mask: CUDA tensors (fixed is kept)."""
    import torch
    fixed = _dev(fixed, torch.float32, "fixed")
    if mask is not None:
        mask = _dev(mask, torch.uint8, "mask")
    h = ctypes.c_void_p()
    with torch.cuda.device(fixed.device):
        _check(lib().nrr_bm_plan_create(fixed.data_ptr(), _i3(_dims_of(fixed)), _i3(block), _i3(stride), _i3(window),
                                        float(frac), mask.data_ptr() if mask is not None else None, int(connectivity),
                                        _stream_ptr(stream), ctypes.byref(h)))
    return NrrPlan(h, _dims_of(fixed), keep=fixed)


def _host_ptr(a):
    return None if a is None else (a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())


def nrr_bm_plan_create_host(fixed, block, stride, window, frac: float, mask=None, connectivity: int = 0) -> NrrPlan:
    """PRE-OPERATIVE, host form: fixed / mask are numpy arrays or (pinned) CPU tensors; the plan owns the device copies."""
    h = ctypes.c_void_p()
    _check(lib().nrr_bm_plan_create_host(_host_ptr(fixed), _i3(_dims_of(fixed)), _i3(block), _i3(stride), _i3(window),
                                         float(frac), _host_ptr(mask), int(connectivity), ctypes.byref(h)))
    return NrrPlan(h, _dims_of(fixed))


def nrr_bm_plan_info(plan: NrrPlan) -> Tuple[int, int]:
    return plan.n, plan.ncand


def nrr_bm_plan_blocks_host(plan: NrrPlan, want_var: bool = False):
    blocks = np.empty((plan.n, 3), dtype=np.int32)
    var = np.empty((plan.n,), dtype=np.float64) if want_var else None
    _check(lib().nrr_bm_plan_blocks_host(plan.handle, blocks.ctypes.data, var.ctypes.data if want_var else None))
    return (blocks, var) if want_var else blocks


def nrr_bm_plan_blocks(plan: NrrPlan, device=None, want_var: bool = False, stream=None):
    """The plan's block centres as a CUDA int32 tensor [n][3] (a copy), optionally with the variances (float64 [n])."""
    import torch
    dev = device if device is not None else torch.device("cuda", torch.cuda.current_device())
    blocks = torch.empty((plan.n, 3), dtype=torch.int32, device=dev)
    var = torch.empty((plan.n,), dtype=torch.float64, device=dev) if want_var else None
    with torch.cuda.device(dev):
        _check(lib().nrr_bm_plan_blocks(plan.handle, blocks.data_ptr(), var.data_ptr() if want_var else None, _stream_ptr(stream)))
    return (blocks, var) if want_var else blocks


def nrr_bm_plan_match(plan: NrrPlan, moving, out_disp=None, out_ncc=None, stream=None, first: int = 0, count: Optional[int] = None):
    """INTRA-OPERATIVE, device form, asynchronous.  With first/count: nrr_bm_plan_match_range (rows outside untouched)."""
    import torch
    moving = _dev(moving, torch.float32, "moving")
    if _dims_of(moving) != tuple(plan.dims):
        raise ValueError("volume shape mismatch")
    if out_disp is None:
        out_disp = torch.empty((plan.n, 3), dtype=torch.int32, device=moving.device)
    if out_ncc is None:
        out_ncc = torch.empty((plan.n,), dtype=torch.float32, device=moving.device)
    with torch.cuda.device(moving.device):
        if count is None and first == 0:
            _check(lib().nrr_bm_plan_match(plan.handle, moving.data_ptr(), out_disp.data_ptr(), out_ncc.data_ptr(), _stream_ptr(stream)))
        else:
            cnt = plan.n - first if count is None else count
            _check(lib().nrr_bm_plan_match_range(plan.handle, moving.data_ptr(), int(first), int(cnt), out_disp.data_ptr(),
                                                 out_ncc.data_ptr(), _stream_ptr(stream)))
    return out_disp, out_ncc


nrr_bm_plan_match_range = nrr_bm_plan_match


def nrr_bm_plan_match_host(plan: NrrPlan, moving, out_disp=None, out_ncc=None):
    """INTRA-OPERATIVE, host form: moving / outputs are numpy arrays or pinned CPU tensors; synchronises."""
    if out_disp is None:
        out_disp = np.empty((plan.n, 3), dtype=np.int32)
    if out_ncc is None:
        out_ncc = np.empty((plan.n,), dtype=np.float32)
    _check(lib().nrr_bm_plan_match_host(plan.handle, _host_ptr(moving), _host_ptr(out_disp), _host_ptr(out_ncc)))
    return out_disp, out_ncc


def nrr_bm_plan_destroy(plan: NrrPlan) -> None:
    if plan.handle is not None and plan.handle.value:
        h, plan.handle = plan.handle, None
        _check(lib().nrr_bm_plan_destroy(h))
    plan._keep = None


class NrrFem:
    """Handle of an nrr_bm_fem model (include/nrr_bm.h "BIOMECHANICAL REGULARISATION")."""

    def __init__(self, handle, dims):
        self.handle, self.dims = handle, tuple(int(v) for v in dims)
        nodes = (ctypes.c_int * 3)()
        n = ctypes.c_int(0)
        _check(lib().nrr_bm_fem_info(handle, nodes, ctypes.byref(n)))
        self.nodes, self.n_nodes = (nodes[0], nodes[1], nodes[2]), n.value

    def __del__(self):
        try:
            nrr_bm_fem_destroy(self)
        except Exception:  # pragma: no cover
            pass


def nrr_bm_fem_create(dims, spacing, young: float, poisson: float) -> NrrFem:
    h = ctypes.c_void_p()
    _check(lib().nrr_bm_fem_create(_i3(dims), _i3(spacing), float(young), float(poisson), ctypes.byref(h)))
    return NrrFem(h, dims)


def nrr_bm_fem_solve(fem: NrrFem, blocks, disp, ncc, weight: float = 1.0, n_iter: int = 1, tol: float = 1e-10,
                     max_cg: int = 2000, out_u=None, stream=None):
    """Device form: blocks/disp int32 CUDA [n][3], ncc fp32 CUDA [n].  Returns (U float64 CUDA [n_nodes][3], CG iterations)."""
    import torch
    blocks = _dev(blocks, torch.int32, "blocks")
    disp = _dev(disp, torch.int32, "disp")
    ncc = _dev(ncc, torch.float32, "ncc")
    n = int(blocks.shape[0])
    if out_u is None:
        out_u = torch.empty((fem.n_nodes, 3), dtype=torch.float64, device=blocks.device)
    iters = ctypes.c_int(0)
    with torch.cuda.device(blocks.device):
        _check(lib().nrr_bm_fem_solve(fem.handle, blocks.data_ptr(), disp.data_ptr(), ncc.data_ptr(), n, float(weight),
                                      int(n_iter), float(tol), int(max_cg), out_u.data_ptr(), ctypes.byref(iters), _stream_ptr(stream)))
    return out_u, iters.value


def nrr_bm_fem_solve_host(fem: NrrFem, blocks: np.ndarray, disp: np.ndarray, ncc: np.ndarray, weight: float = 1.0,
                          n_iter: int = 1, tol: float = 1e-10, max_cg: int = 2000):
    blocks, disp, ncc = _np(blocks, np.int32, "blocks"), _np(disp, np.int32, "disp"), _np(ncc, np.float32, "ncc")
    out_u = np.empty((fem.n_nodes, 3), dtype=np.float64)
    iters = ctypes.c_int(0)
    _check(lib().nrr_bm_fem_solve_host(fem.handle, blocks.ctypes.data, disp.ctypes.data, ncc.ctypes.data, int(blocks.shape[0]),
                                       float(weight), int(n_iter), float(tol), int(max_cg), out_u.ctypes.data, ctypes.byref(iters)))
    return out_u, iters.value


def nrr_bm_fem_dense_field(fem: NrrFem, u, out_field=None, stream=None):
    """Device form, asynchronous: u float64 CUDA [n_nodes][3] -> field fp32 CUDA [3][nz][ny][nx] (what nrr_bm_warp takes)."""
    import torch
    u = _dev(u, torch.float64, "u")
    nx, ny, nz = fem.dims
    if out_field is None:
        out_field = torch.empty((3, nz, ny, nx), dtype=torch.float32, device=u.device)
    with torch.cuda.device(u.device):
        _check(lib().nrr_bm_fem_dense_field(fem.handle, u.data_ptr(), out_field.data_ptr(), _stream_ptr(stream)))
    return out_field


def nrr_bm_fem_dense_field_host(fem: NrrFem, u: np.ndarray) -> np.ndarray:
    u = _np(u, np.float64, "u")
    nx, ny, nz = fem.dims
    out = np.empty((3, nz, ny, nx), dtype=np.float32)
    _check(lib().nrr_bm_fem_dense_field_host(fem.handle, u.ctypes.data, out.ctypes.data))
    return out


def nrr_bm_fem_destroy(fem: NrrFem) -> None:
    if fem.handle is not None and fem.handle.value:
        h, fem.handle = fem.handle, None
        _check(lib().nrr_bm_fem_destroy(h))


def nrr_bm_warp(image, field, out=None, stream=None):
    """Device form, asynchronous: out(p) = trilinear(image, clamp(p + v(p))); field is CUDA fp32 [3][nz][ny][nx]."""
    import torch
    image = _dev(image, torch.float32, "image")
    field = _dev(field, torch.float32, "field")
    if tuple(field.shape) != (3,) + tuple(image.shape):
        raise ValueError("field must be [3][nz][ny][nx]")
    if out is None:
        out = torch.empty_like(image)
    out = _dev(out, torch.float32, "out")
    with torch.cuda.device(image.device):
        _check(lib().nrr_bm_warp(image.data_ptr(), _i3(_dims_of(image)), field.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
    return out


def nrr_bm_moving_stats(moving, block, out_inv_sd=None, stream=None):
    """Device form, asynchronous. Returns inv_sd fp32 CUDA [nz][ny][nx] (entries whose block leaves the volume untouched)."""
    import torch
    moving = _dev(moving, torch.float32, "moving")
    if out_inv_sd is None:
        out_inv_sd = torch.zeros_like(moving)
    out_inv_sd = _dev(out_inv_sd, torch.float32, "out_inv_sd")
    with torch.cuda.device(moving.device):
        _check(lib().nrr_bm_moving_stats(moving.data_ptr(), _i3(_dims_of(moving)), _i3(block), out_inv_sd.data_ptr(),
                                         _stream_ptr(stream)))
    return out_inv_sd


def nrr_bm_check_async_error(stream=None) -> None:
    _check(lib().nrr_bm_check_async_error(_stream_ptr(stream)))


# --------------------------------------------------------------------------------------------- host API
def _np(a, dtype, name):
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise TypeError("%s must be a C-contiguous numpy %s array" % (name, np.dtype(dtype).name))
    return a


def nrr_bm_select_blocks_host(fixed: np.ndarray, block, stride, frac: float, mask: Optional[np.ndarray] = None,
                              capacity: Optional[int] = None):
    fixed = _np(fixed, np.float32, "fixed")
    dims = _dims_of(fixed)
    if mask is not None:
        mask = _np(mask, np.uint8, "mask")
    if capacity is None:
        capacity = max(1, int(np.prod([max(0, (dims[a] - block[a]) // stride[a] + 1) for a in range(3)])))
    out_blocks = np.empty((capacity, 3), dtype=np.int32)
    out_var = np.empty((capacity,), dtype=np.float64)
    n, ncand = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().nrr_bm_select_blocks_host(fixed.ctypes.data, _i3(dims), _i3(block), _i3(stride), float(frac),
                                           mask.ctypes.data if mask is not None else None, out_blocks.ctypes.data,
                                           int(capacity), ctypes.byref(n), out_var.ctypes.data, ctypes.byref(ncand)))
    return out_blocks[:n.value], n.value, ncand.value, out_var[:n.value]


def nrr_bm_match_host(fixed: np.ndarray, moving: np.ndarray, blocks: np.ndarray, block, window):
    fixed = _np(fixed, np.float32, "fixed")
    moving = _np(moving, np.float32, "moving")
    blocks = _np(blocks, np.int32, "blocks")
    n = int(blocks.shape[0])
    disp = np.empty((n, 3), dtype=np.int32)
    ncc = np.empty((n,), dtype=np.float32)
    _check(lib().nrr_bm_match_host(fixed.ctypes.data, moving.ctypes.data, _i3(_dims_of(fixed)), blocks.ctypes.data, n,
                                   _i3(block), _i3(window), disp.ctypes.data, ncc.ctypes.data))
    return disp, ncc


def nrr_bm_register_host(fixed, moving, block, stride, window, frac: float, mask=None, out_blocks=None,
                         out_disp=None, out_ncc=None):
    """select + match of one pair from HOST buffers (numpy arrays or pinned CPU torch tensors).
    Returns (blocks [K][3], disp [K][3], ncc [K]) as views of the output buffers."""
    def ptr(a):
        return None if a is None else (a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())
    dims = _dims_of(fixed)
    cap = int(np.prod([max(0, (dims[a] - block[a]) // stride[a] + 1) for a in range(3)]))
    if out_blocks is None:
        out_blocks = np.empty((cap, 3), dtype=np.int32)
        out_disp = np.empty((cap, 3), dtype=np.int32)
        out_ncc = np.empty((cap,), dtype=np.float32)
    cap = int(out_blocks.shape[0])
    n = ctypes.c_int(0)
    _check(lib().nrr_bm_register_host(ptr(fixed), ptr(moving), _i3(dims), _i3(block), _i3(stride), _i3(window),
                                      float(frac), ptr(mask), ptr(out_blocks), cap, ctypes.byref(n), ptr(out_disp),
                                      ptr(out_ncc)))
    k = n.value
    return out_blocks[:k], out_disp[:k], out_ncc[:k]


# --------------------------------------------------------------------------------------------- instrumentation
def nrr_bm_profile_enable(on: bool) -> None:
    _check(lib().nrr_bm_profile_enable(1 if on else 0))


def nrr_bm_profile_read():
    ms = (ctypes.c_double * 4)()
    calls = (ctypes.c_int * 4)()
    _check(lib().nrr_bm_profile_read(ms, calls))
    return {"select_ms": ms[0], "moving_stats_ms": ms[1], "match_ms": ms[2], "prep_ms": ms[3],
            "select_calls": calls[0], "moving_stats_calls": calls[1], "match_calls": calls[2], "prep_calls": calls[3]}


def nrr_bm_launch_count(reset: bool = False) -> int:
    return int(lib().nrr_bm_launch_count(1 if reset else 0))


def nrr_bm_match_info(dims, block, window, n: int = 0):
    """Which matching kernel (and launch shape) a (dims, block, window) triple dispatches to, for a launch of n blocks."""
    info = (ctypes.c_int * 6)()
    _check(lib().nrr_bm_match_info_n(_i3(dims), _i3(block), _i3(window), int(n), info))
    return {"fast": bool(info[0]), "kernel": info[0], "threads": info[1], "smem_bytes": info[2], "tma": bool(info[3]),
            "candidates": info[4], "blocks_per_cta": info[5]}


def nrr_bm_pair_task_table(block, window):
    """Returns (table uint32 [threads], info dict) of the pair kernel's lane -> task assignment. No device needed."""
    info = (ctypes.c_int * 6)()
    tab = np.zeros(1024, dtype=np.uint32)
    _check(lib().nrr_bm_pair_task_table(_i3(block), _i3(window), tab.ctypes.data, tab.size, info))
    return tab[: info[0]].copy(), {"threads": info[0], "blocks_per_cta": info[1], "pitch": info[2], "rows_per_plane": info[3],
                                   "union_stride": info[4], "smem_bytes": info[5]}


def nrr_bm_fp32_peak(stream=None) -> float:
    out = ctypes.c_double(0.0)
    _check(lib().nrr_bm_fp32_peak(ctypes.byref(out), _stream_ptr(stream)))
    return out.value


def nrr_bm_fp32_microbench(stream=None):
    """TFLOP/s of the FP32 microbenchmarks (include/nrr_bm.h): register-only FFMA / FFMA2 and three main-loop bodies."""
    out = (ctypes.c_double * 7)()
    _check(lib().nrr_bm_fp32_microbench(out, _stream_ptr(stream)))
    names = ("ffma_chain", "ffma_tile", "ffma2_packed", "ffma2_scalar", "loop_1row_ffma_useful", "loop_2row_ffma_useful", "loop_2row_ffma2_useful")
    return dict(zip(names, [float(v) for v in out]))


def nrr_bm_set_option(name: str, value: float) -> None:
    _check(lib().nrr_bm_set_option(name.encode(), float(value)))


def nrr_bm_version() -> int:
    return int(lib().nrr_bm_version())
