"""pytest plugin: run the `-m gpu` test FILES against the host-model library, on a machine without a GPU.

TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  It tests the tests (their expectations, sizes, generators) and the ctypes
marshalling of paper_2511_02742_b200/hough.py: the binding is pointed at tests/emu/libhough_emu.so, `.cuda()` becomes the
identity and "cuda" devices become the CPU, for the duration of this pytest process only.  Nothing here is importable from the
product, and the product binding itself has no CPU path.

    PYTHONPATH=tests/emu python -m pytest tests/test_gpu_parity.py tests/test_gpu_track.py -m gpu -p emu_plugin -q
"""
import ctypes, os, sys
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for _p in (HERE, ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

_real_device = torch.device
def _dev(*a, **k):
    if a and isinstance(a[0], str) and a[0].startswith("cuda"):
        return _real_device("cpu")
    return _real_device(*a, **k)
torch.device = _dev
torch.Tensor.cuda = lambda self, *a, **k: self
torch.Tensor.pin_memory = lambda self: self
torch.cuda.synchronize = lambda *a, **k: None
torch.cuda.device_count = lambda: 1
class _S: cuda_stream = 0
torch.cuda.current_stream = lambda *a, **k: _S()
def _wrap(fn):
    def w(*a, **k):
        d = k.get("device")
        if isinstance(d, str) and d.startswith("cuda"):
            k["device"] = "cpu"
        return fn(*a, **k)
    return w
for name in ("zeros", "empty", "full", "tensor", "ones"):
    setattr(torch, name, _wrap(getattr(torch, name)))

import hough_emu as E
from paper_2511_02742_b200 import hough as H
H.load_library(E.lib()._name)

def _devptr(plan, t, dtype, name):
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous {dtype} tensor, got {t.dtype}")
    return ctypes.c_void_p(t.data_ptr())
H._dev = _devptr
H._stream_ptr = lambda plan, stream: None
