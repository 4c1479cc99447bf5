"""TEST INFRASTRUCTURE ONLY: ctypes access to tests/cuda_emul/libnrr_bm_emul.so, the product's .cu sources
compiled as plain C++ against a fiber-per-thread CUDA emulation (see tests/cuda_emul/include/cuda_runtime.h).
It exercises the kernels' logic on the CPU through the same C-ABI host entry points; it is not a product path
(the package never loads it, and without a CUDA device the product library returns NRR_E_CUDA)."""
import ctypes
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


def lib():
    global _lib
    if _lib is None:
        spec = importlib.util.spec_from_file_location("build_emul", os.path.join(_HERE, "cuda_emul", "build_emul.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        L = ctypes.CDLL(mod.build())
        L.nrr_bm_last_error.restype = ctypes.c_char_p
        L.nrr_bm_set_option.argtypes = [ctypes.c_char_p, ctypes.c_double]
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        i3 = ctypes.POINTER(ctypes.c_int)
        L.nrr_bm_select_blocks_host.argtypes = [vp, i3, i3, i3, cd, vp, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci)]
        L.nrr_bm_select_blocks_pruned_host.argtypes = [vp, i3, i3, i3, cd, vp, ci, vp, ci, ctypes.POINTER(ci), vp, ctypes.POINTER(ci)]
        L.nrr_bm_warp_host.argtypes = [vp, i3, vp, vp]
        L.nrr_bm_match_host.argtypes = [vp, vp, i3, vp, ci, i3, i3, vp, vp]
        L.nrr_bm_match_info.argtypes = [i3, i3, i3, i3]
        L.nrr_bm_moving_stats_host.argtypes = [vp, i3, i3, vp]
        L.nrr_bm_register_host.argtypes = [vp, vp, i3, i3, i3, i3, cd, vp, vp, ci, ctypes.POINTER(ci), vp, vp]
        _lib = L
    return _lib


def _i3(t):
    return (ctypes.c_int * 3)(int(t[0]), int(t[1]), int(t[2]))


def _check(rc):
    if rc != 0:
        raise RuntimeError("emulated libnrr_bm status %d: %s" % (rc, lib().nrr_bm_last_error().decode()))


def set_option(name, value):
    _check(lib().nrr_bm_set_option(name.encode(), float(value)))


def match_info(dims, block, window):
    info = (ctypes.c_int * 6)()
    _check(lib().nrr_bm_match_info(_i3(dims), _i3(block), _i3(window), info))
    return {"kernel": info[0], "threads": info[1], "smem_bytes": info[2], "tma": info[3], "candidates": info[4]}


def select(fixed, block, stride, frac, mask=None):
    nz, ny, nx = fixed.shape
    cap = max(1, int(np.prod([max(0, ((nx, ny, nz)[a] - block[a]) // stride[a] + 1) for a in range(3)])))
    blocks = np.empty((cap, 3), np.int32)
    var = np.empty((cap,), np.float64)
    n, ncand = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().nrr_bm_select_blocks_host(fixed.ctypes.data, _i3((nx, ny, nz)), _i3(block), _i3(stride), float(frac),
                                           None if mask is None else mask.ctypes.data, blocks.ctypes.data, cap,
                                           ctypes.byref(n), var.ctypes.data, ctypes.byref(ncand)))
    return blocks[:n.value], n.value, ncand.value, var[:n.value]


def match(fixed, moving, blocks, block, window):
    nz, ny, nx = fixed.shape
    blocks = np.ascontiguousarray(blocks, np.int32)
    n = blocks.shape[0]
    disp = np.empty((n, 3), np.int32)
    ncc = np.empty((n,), np.float32)
    _check(lib().nrr_bm_match_host(fixed.ctypes.data, moving.ctypes.data, _i3((nx, ny, nz)), blocks.ctypes.data, n,
                                   _i3(block), _i3(window), disp.ctypes.data, ncc.ctypes.data))
    return disp, ncc


def moving_stats(moving, block, fill=-7.0):
    nz, ny, nx = moving.shape
    out = np.full(moving.shape, fill, np.float32)
    _check(lib().nrr_bm_moving_stats_host(moving.ctypes.data, _i3((nx, ny, nz)), _i3(block), out.ctypes.data))
    return out


def register(fixed, moving, block, stride, window, frac, mask=None):
    nz, ny, nx = fixed.shape
    cap = max(1, int(np.prod([max(0, ((nx, ny, nz)[a] - block[a]) // stride[a] + 1) for a in range(3)])))
    blocks = np.full((cap, 3), -99, np.int32)
    disp = np.full((cap, 3), -99, np.int32)
    ncc = np.full((cap,), -99.0, np.float32)
    n = ctypes.c_int(0)
    _check(lib().nrr_bm_register_host(fixed.ctypes.data, moving.ctypes.data, _i3((nx, ny, nz)), _i3(block), _i3(stride),
                                      _i3(window), float(frac), None if mask is None else mask.ctypes.data,
                                      blocks.ctypes.data, cap, ctypes.byref(n), disp.ctypes.data, ncc.ctypes.data))
    return blocks[:n.value], disp[:n.value], ncc[:n.value]


def select_pruned(fixed, block, stride, frac, mask, connectivity):
    nz, ny, nx = fixed.shape
    cap = max(1, int(np.prod([max(0, ((nx, ny, nz)[a] - block[a]) // stride[a] + 1) for a in range(3)])))
    blocks = np.empty((cap, 3), np.int32)
    var = np.empty((cap,), np.float64)
    n, ncand = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().nrr_bm_select_blocks_pruned_host(fixed.ctypes.data, _i3((nx, ny, nz)), _i3(block), _i3(stride),
                                                  float(frac), None if mask is None else mask.ctypes.data,
                                                  int(connectivity), blocks.ctypes.data, cap, ctypes.byref(n),
                                                  var.ctypes.data, ctypes.byref(ncand)))
    return blocks[:n.value], n.value, ncand.value, var[:n.value]


def warp(image, field):
    nz, ny, nx = image.shape
    field = np.ascontiguousarray(field, np.float32)
    out = np.empty_like(image)
    _check(lib().nrr_bm_warp_host(image.ctypes.data, _i3((nx, ny, nz)), field.ctypes.data, out.ctypes.data))
    return out


# ---- plans, the parameter sweep, the capacity bound (in the emulation a "device" pointer is a host pointer)
class Setting(ctypes.Structure):
    _fields_ = [("block", ctypes.c_int * 3), ("stride", ctypes.c_int * 3), ("window", ctypes.c_int * 3), ("frac", ctypes.c_double)]


def capacity_bound(dims, block, stride, frac):
    g, b = ctypes.c_int(0), ctypes.c_int(0)
    L = lib()
    L.nrr_bm_capacity_bound.argtypes = [ctypes.POINTER(ctypes.c_int)] * 3 + [ctypes.c_double] + [ctypes.POINTER(ctypes.c_int)] * 2
    _check(L.nrr_bm_capacity_bound(_i3(dims), _i3(block), _i3(stride), float(frac), ctypes.byref(g), ctypes.byref(b)))
    return g.value, b.value


class Plan:
    def __init__(self, fixed, block, stride, window, frac, mask=None, connectivity=0, host=True):
        L = lib()
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        i3 = ctypes.POINTER(ctypes.c_int)
        L.nrr_bm_plan_create_host.argtypes = [vp, i3, i3, i3, i3, cd, vp, ci, ctypes.POINTER(vp)]
        L.nrr_bm_plan_create.argtypes = [vp, i3, i3, i3, i3, cd, vp, ci, vp, ctypes.POINTER(vp)]
        L.nrr_bm_plan_info.argtypes = [vp, i3, i3]
        L.nrr_bm_plan_blocks_host.argtypes = [vp, vp, vp]
        L.nrr_bm_plan_match.argtypes = [vp, vp, vp, vp, vp]
        L.nrr_bm_plan_match_range.argtypes = [vp, vp, ci, ci, vp, vp, vp]
        L.nrr_bm_plan_match_host.argtypes = [vp, vp, vp, vp]
        L.nrr_bm_plan_destroy.argtypes = [vp]
        nz, ny, nx = fixed.shape
        self.fixed, self.mask = fixed, mask      # the device form keeps the caller's pointer
        self.h = vp()
        mp = None if mask is None else mask.ctypes.data
        if host:
            _check(L.nrr_bm_plan_create_host(fixed.ctypes.data, _i3((nx, ny, nz)), _i3(block), _i3(stride), _i3(window),
                                             float(frac), mp, int(connectivity), ctypes.byref(self.h)))
        else:
            _check(L.nrr_bm_plan_create(fixed.ctypes.data, _i3((nx, ny, nz)), _i3(block), _i3(stride), _i3(window),
                                        float(frac), mp, int(connectivity), None, ctypes.byref(self.h)))
        n, nc = ctypes.c_int(0), ctypes.c_int(0)
        _check(L.nrr_bm_plan_info(self.h, ctypes.byref(n), ctypes.byref(nc)))
        self.n, self.ncand = n.value, nc.value

    def blocks(self):
        b = np.empty((self.n, 3), np.int32)
        v = np.empty((self.n,), np.float64)
        _check(lib().nrr_bm_plan_blocks_host(self.h, b.ctypes.data, v.ctypes.data))
        return b, v

    def match(self, moving, first=None, count=None, out=None):
        disp, ncc = out if out is not None else (np.full((self.n, 3), -99, np.int32), np.full((self.n,), -99.0, np.float32))
        if first is None:
            _check(lib().nrr_bm_plan_match(self.h, moving.ctypes.data, disp.ctypes.data, ncc.ctypes.data, None))
        else:
            _check(lib().nrr_bm_plan_match_range(self.h, moving.ctypes.data, int(first), int(count), disp.ctypes.data, ncc.ctypes.data, None))
        _check(lib().nrr_bm_check_async_error(None))
        return disp, ncc

    def match_host(self, moving):
        disp = np.full((self.n, 3), -99, np.int32)
        ncc = np.full((self.n,), -99.0, np.float32)
        _check(lib().nrr_bm_plan_match_host(self.h, moving.ctypes.data, disp.ctypes.data, ncc.ctypes.data))
        return disp, ncc

    def destroy(self):
        if self.h:
            _check(lib().nrr_bm_plan_destroy(self.h))
            self.h = None


def register_batch(fixed, moving, settings, mask=None):
    """settings: iterable of (block, stride, window, frac).  Returns [(blocks, disp, ncc)] trimmed to K per setting."""
    L = lib()
    vp, ci = ctypes.c_void_p, ctypes.c_int
    i3 = ctypes.POINTER(ctypes.c_int)
    pp = ctypes.POINTER(vp)
    L.nrr_bm_register_batch.argtypes = [vp, vp, i3, vp, vp, ci, pp, i3, vp, pp, pp, vp]
    nz, ny, nx = fixed.shape
    ns = len(settings)
    arr = (Setting * ns)()
    caps = (ci * ns)()
    pb, pd, pn = (vp * ns)(), (vp * ns)(), (vp * ns)()
    keep = []
    for i, (block, stride, window, frac) in enumerate(settings):
        arr[i].block[:] = list(block)
        arr[i].stride[:] = list(stride)
        arr[i].window[:] = list(window)
        arr[i].frac = float(frac)
        cap = max(1, capacity_bound((nx, ny, nz), block, stride, frac)[1])
        caps[i] = cap
        b = np.full((cap, 3), -99, np.int32)
        d = np.full((cap, 3), -99, np.int32)
        c = np.full((cap,), -99.0, np.float32)
        pb[i], pd[i], pn[i] = b.ctypes.data, d.ctypes.data, c.ctypes.data
        keep.append((b, d, c))
    out_n = np.zeros((ns,), np.int32)
    _check(L.nrr_bm_register_batch(fixed.ctypes.data, moving.ctypes.data, _i3((nx, ny, nz)),
                                   None if mask is None else mask.ctypes.data, arr, ns, pb, caps, out_n.ctypes.data, pd, pn, None))
    _check(L.nrr_bm_check_async_error(None))
    return [(b[:k], d[:k], c[:k]) for (b, d, c), k in zip(keep, out_n)], out_n


# ---- biomechanical regularisation (nrr_fem.cu)
class Fem:
    def __init__(self, dims, spacing, young, poisson):
        L = lib()
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        i3 = ctypes.POINTER(ctypes.c_int)
        L.nrr_bm_fem_create.argtypes = [i3, i3, cd, cd, ctypes.POINTER(vp)]
        L.nrr_bm_fem_info.argtypes = [vp, i3, i3]
        L.nrr_bm_fem_solve_host.argtypes = [vp, vp, vp, vp, ci, cd, ci, cd, ci, vp, i3]
        L.nrr_bm_fem_solve.argtypes = [vp, vp, vp, vp, ci, cd, ci, cd, ci, vp, i3, vp]
        L.nrr_bm_fem_dense_field_host.argtypes = [vp, vp, vp]
        L.nrr_bm_fem_destroy.argtypes = [vp]
        self.dims = tuple(dims)
        self.h = vp()
        _check(L.nrr_bm_fem_create(_i3(dims), _i3(spacing), float(young), float(poisson), ctypes.byref(self.h)))
        nodes = (ci * 3)()
        n = ci(0)
        _check(L.nrr_bm_fem_info(self.h, nodes, ctypes.byref(n)))
        self.nodes, self.n_nodes = tuple(nodes), n.value

    def solve(self, blocks, disp, ncc, weight=1.0, n_iter=1, tol=1e-12, max_cg=5000, allow_noconv=False):
        blocks = np.ascontiguousarray(blocks, np.int32)
        disp = np.ascontiguousarray(disp, np.int32)
        ncc = np.ascontiguousarray(ncc, np.float32)
        u = np.full((self.n_nodes, 3), np.nan)
        iters = ctypes.c_int(0)
        rc = lib().nrr_bm_fem_solve_host(self.h, blocks.ctypes.data, disp.ctypes.data, ncc.ctypes.data, len(blocks), float(weight),
                                         int(n_iter), float(tol), int(max_cg), u.ctypes.data, ctypes.byref(iters))
        if not (allow_noconv and rc == -13):
            _check(rc)
        return u, iters.value, rc

    def dense_field(self, u):
        nx, ny, nz = self.dims
        out = np.empty((3, nz, ny, nx), np.float32)
        u = np.ascontiguousarray(u, np.float64)
        _check(lib().nrr_bm_fem_dense_field_host(self.h, u.ctypes.data, out.ctypes.data))
        return out

    def destroy(self):
        if self.h:
            _check(lib().nrr_bm_fem_destroy(self.h))
            self.h = None
