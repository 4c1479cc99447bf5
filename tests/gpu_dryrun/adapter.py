"""TEST INFRASTRUCTURE ONLY: lets tests/test_gpu_parity.py run without a GPU, against the CPU emulation of the kernels
(tests/cuda_emul), THROUGH THE REAL BINDING.  `paper_2308_10868_b200.binding` is imported unchanged; only its three
device-facing helpers are patched -- the library path (the emulated build exports the same C ABI), the "must be a CUDA
tensor" check and the stream lookup -- so every marshalling line of binding.py that the GPU tests will execute on the
GPU box has executed here first.  In the emulation a "device" pointer is a host pointer, so CPU tensors serve as device
memory.  tests/test_gpu_suite_dryrun.py runs a quick subset of the GPU tests this way, in a subprocess.  Importing this
module patches torch for the whole process: only run.py imports it."""
import contextlib
import importlib.util
import os
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

spec = importlib.util.spec_from_file_location("build_emul", os.path.join(ROOT, "tests", "cuda_emul", "build_emul.py"))
_be = importlib.util.module_from_spec(spec)
spec.loader.exec_module(_be)

import paper_2308_10868_b200.binding as B  # noqa: E402

B.LIB_PATH = _be.build()                     # the product's sources, compiled for the CPU


def _dev(t, dtype, name):
    if not isinstance(t, torch.Tensor):
        raise TypeError("%s must be a tensor" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous %s tensor" % (name, dtype))
    return t


B._dev = _dev
B._stream_ptr = lambda stream=None: 0

# torch: "cuda" means this process's memory
torch.Tensor.cuda = lambda self, *a, **k: self
torch.cuda.is_available = lambda: True
torch.cuda.synchronize = lambda *a, **k: None
torch.cuda.current_device = lambda: 0
torch.cuda.device = lambda *a, **k: contextlib.nullcontext()
_orig_device = torch.device


def _strip(fn):
    def g(*a, **k):
        dev = k.get("device")
        if dev is not None and "cuda" in str(dev):
            k.pop("device")
        return fn(*a, **k)
    return g


for _name in ("empty", "full", "zeros", "zeros_like", "empty_like"):
    setattr(torch, _name, _strip(getattr(torch, _name)))
