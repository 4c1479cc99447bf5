"""TEST INFRASTRUCTURE ONLY: a stand-in for the `paper_2308_10868_b200` binding that forwards to the emulated
library (tests/cuda_emul) and works on CPU tensors, plus the torch patches that let tests/test_gpu_parity.py run
without a GPU.  tests/test_gpu_suite_dryrun.py runs a quick subset of the GPU tests this way, in a subprocess, so
that a mistake in the GPU tests themselves (a wrong signature, a stale expectation) is found here and not on the
GPU box.  Importing this module patches torch for the whole process: only run.py imports it."""
import sys, types, os
import numpy as np
import torch
ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
import _emul

class NrrError(RuntimeError):
    def __init__(self, status, msg=""):
        super().__init__(msg); self.status = status

def _wrap(fn):
    def g(*a, **k):
        try:
            return fn(*a, **k)
        except RuntimeError as e:
            import re
            m = re.search(r"status (-?\d+)", str(e))
            raise NrrError(int(m.group(1)) if m else -999, str(e))
    return g

fake = types.ModuleType("paper_2308_10868_b200")
fake.NrrError = NrrError
fake.lib = _emul.lib
fake.nrr_bm_set_option = _emul.set_option
_pending = {"err": None}
def _np(t): return None if t is None else t.numpy()
def select(fixed, block, stride, frac, mask=None, capacity=None, want_var=False, stream=None):
    b, n, nc, v = _emul.select(_np(fixed), block, stride, frac, _np(mask))
    if capacity is not None and n > capacity: raise NrrError(-7, "capacity")
    r = (torch.from_numpy(b.copy()), n, nc)
    return r + (torch.from_numpy(v.copy()),) if want_var else r
def select_pruned(fixed, block, stride, frac, mask=None, connectivity=6, capacity=None, want_var=False, stream=None):
    b, n, nc, v = _emul.select_pruned(_np(fixed), block, stride, frac, _np(mask), connectivity)
    r = (torch.from_numpy(b.copy()), n, nc)
    return r + (torch.from_numpy(v.copy()),) if want_var else r
def match(fixed, moving, blocks, block, window, out_disp=None, out_ncc=None, stream=None):
    if blocks.shape[0] == 0:
        return torch.empty((0,3),dtype=torch.int32), torch.empty((0,),dtype=torch.float32)
    try:
        d, s = _emul.match(_np(fixed), _np(moving), _np(blocks), block, window)
    except RuntimeError as e:
        if "leaves the volume" in str(e) or "status -12" in str(e):      # sticky device flags: reported by the next check
            _pending["err"] = NrrError(-12 if "status -12" in str(e) else -8, str(e))
            n = blocks.shape[0]
            return torch.zeros((n,3),dtype=torch.int32), torch.full((n,), float("nan"))
        raise
    return torch.from_numpy(d), torch.from_numpy(s)
def check_async(stream=None):
    e, _pending["err"] = _pending["err"], None
    if e: raise e
def register(fixed, moving, block, stride, window, frac, mask=None, capacity=None, **kw):
    b, d, s = _emul.register(_np(fixed), _np(moving), block, stride, window, frac, _np(mask))
    n = len(b)
    cap = n if capacity is None else capacity
    k = min(n, cap)
    return torch.from_numpy(b[:k].copy()), torch.tensor(n, dtype=torch.int32), torch.from_numpy(d[:k].copy()), torch.from_numpy(s[:k].copy())
def moving_stats(moving, block, out=None, stream=None):
    fill = -7.0
    r = _emul.moving_stats(_np(moving), block, fill)
    return torch.from_numpy(r)
def match_info(dims, block, window):
    i = _emul.match_info(dims, block, window)
    return {"fast": bool(i["kernel"]), "kernel": i["kernel"], "threads": i["threads"], "smem_bytes": i["smem_bytes"], "tma": bool(i["tma"]), "candidates": i["candidates"], "blocks_per_cta": 0}
class _Plan:
    def __init__(self, p): self.p, self.n, self.ncand = p, p.n, p.ncand
def plan_create(fixed, block, stride, window, frac, mask=None, connectivity=0, stream=None):
    return _Plan(_emul.Plan(_np(fixed), block, stride, window, frac, _np(mask), connectivity, host=False))
def plan_create_host(fixed, block, stride, window, frac, mask=None, connectivity=0):
    return _Plan(_emul.Plan(fixed, block, stride, window, frac, mask, connectivity, host=True))
def plan_match(plan, moving, out_disp=None, out_ncc=None, stream=None, first=0, count=None):
    out = None if out_disp is None else (out_disp.numpy(), out_ncc.numpy())
    if count is None and first == 0:
        d, s = plan.p.match(_np(moving), out=out)
    else:
        d, s = plan.p.match(_np(moving), first, plan.n - first if count is None else count, out=out)
    return (torch.from_numpy(d), torch.from_numpy(s)) if out is None else (out_disp, out_ncc)
def register_batch(fixed, moving, settings, mask=None, stream=None):
    got, out_n = _emul.register_batch(_np(fixed), _np(moving), [(st.block, st.stride, st.window, st.frac) for st in settings], _np(mask))
    return [tuple(torch.from_numpy(a.copy()) for a in g) for g in got], torch.from_numpy(out_n)
fake.nrr_bm_plan_create = plan_create
fake.nrr_bm_plan_create_host = plan_create_host
fake.nrr_bm_plan_info = lambda plan: (plan.n, plan.ncand)
fake.nrr_bm_plan_blocks_host = lambda plan, want_var=False: plan.p.blocks() if want_var else plan.p.blocks()[0]
fake.nrr_bm_plan_blocks = lambda plan, device=None, want_var=False, stream=None: torch.from_numpy(plan.p.blocks()[0])
fake.nrr_bm_plan_match = plan_match
fake.nrr_bm_plan_match_range = plan_match
fake.nrr_bm_plan_match_host = lambda plan, moving, out_disp=None, out_ncc=None: plan.p.match_host(moving)
fake.nrr_bm_plan_destroy = lambda plan: plan.p.destroy()
class _Fem:
    def __init__(self, f): self.f, self.nodes, self.n_nodes, self.dims = f, f.nodes, f.n_nodes, f.dims
def fem_solve(fem, blocks, disp, ncc, weight=1.0, n_iter=1, tol=1e-10, max_cg=2000, out_u=None, stream=None):
    u, it, _ = fem.f.solve(_np(blocks), _np(disp), _np(ncc), weight, n_iter, tol, max_cg)
    return torch.from_numpy(u), it
fake.nrr_bm_fem_create = lambda dims, spacing, young, poisson: _Fem(_emul.Fem(dims, spacing, young, poisson))
fake.nrr_bm_fem_solve = fem_solve
fake.nrr_bm_fem_solve_host = lambda fem, b, d, c, weight=1.0, n_iter=1, tol=1e-10, max_cg=2000: fem.f.solve(b, d, c, weight, n_iter, tol, max_cg)[:2]
fake.nrr_bm_fem_dense_field = lambda fem, u, out_field=None, stream=None: torch.from_numpy(fem.f.dense_field(u.numpy()))
fake.nrr_bm_fem_destroy = lambda fem: fem.f.destroy()
fake.nrr_bm_register_batch = register_batch
fake.nrr_bm_capacity_bound = _emul.capacity_bound
fake.nrr_bm_select_blocks = select
fake.nrr_bm_select_blocks_pruned = select_pruned
fake.nrr_bm_match = match
fake.nrr_bm_check_async_error = check_async
fake.nrr_bm_register = register
fake.nrr_bm_moving_stats = moving_stats
fake.nrr_bm_match_info = match_info
fake.nrr_bm_warp = lambda img, field, out=None, stream=None: torch.from_numpy(_emul.warp(img.numpy(), field.numpy()))
fake.nrr_bm_select_blocks_host = lambda f, b, s, fr, mask=None, capacity=None: _emul.select(f, b, s, fr, mask)
fake.nrr_bm_match_host = lambda f, m, bl, b, w: _emul.match(f, m, bl, b, w)
fake.nrr_bm_register_host = lambda f, m, b, s, w, fr, mask=None, *a: _emul.register(f, m, b, s, w, fr, mask)
sys.modules["paper_2308_10868_b200"] = fake
torch.Tensor.cuda = lambda self, *a, **k: self
torch.cuda.is_available = lambda: True
torch.cuda.synchronize = lambda *a, **k: None
_orig_empty, _orig_full = torch.empty, torch.full
def _strip(fn):
    def g(*a, **k):
        k.pop("device", None); return fn(*a, **k)
    return g
torch.empty = _strip(_orig_empty); torch.full = _strip(_orig_full)
