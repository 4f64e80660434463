"""Device-side generator of BASELINE.json configs[4] (gen/_gen_cuda.cu): the throughput-sweep points too large for the host.
Input generation only; bit-identical to gen.config5_sweep_point (checked by the GPU tests on small points)."""
from __future__ import annotations

import ctypes
import os
import subprocess

from .workloads import SEED0

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "_gen_cuda.cu")
_LIB = os.path.join(_HERE, "_gen_cuda.so")
_lib = None


def build_cuda(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(["nvcc", "-O3", "-fmad=false", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def config5_on_device(log2m: int, k: int, device="cuda:0", seed: int = SEED0 + 5):
    """Returns dict(m, n, nnz, rowptr, col, val, lb, ub, lo, hi, x0, x_true) of torch tensors on `device` (fp32 / int32 / int64)."""
    import torch

    global _lib
    if _lib is None:
        build_cuda()
        _lib = ctypes.CDLL(_LIB)
        _lib.gen_cfg5_device.argtypes = [ctypes.c_int64, ctypes.c_int, ctypes.c_uint64] + [ctypes.c_void_p] * 7
    m = 1 << log2m
    n = m // 2
    assert n % k == 0
    dev = torch.device(device)
    with torch.cuda.device(dev):
        rowptr = torch.empty(m + 1, dtype=torch.int64, device=dev)
        col = torch.empty(m * k, dtype=torch.int32, device=dev)
        val = torch.empty(m * k, dtype=torch.float32, device=dev)
        xs = torch.empty(n, dtype=torch.float32, device=dev)
        lb = torch.empty(m, dtype=torch.float32, device=dev)
        ub = torch.empty(m, dtype=torch.float32, device=dev)
        rc = _lib.gen_cfg5_device(m, k, seed, rowptr.data_ptr(), col.data_ptr(), val.data_ptr(), xs.data_ptr(), lb.data_ptr(), ub.data_ptr(),
                                  ctypes.c_void_p(torch.cuda.current_stream(dev).cuda_stream))
        if rc:
            raise RuntimeError(f"gen_cfg5_device: CUDA error {rc}")
        torch.cuda.synchronize(dev)
    return dict(m=m, n=n, nnz=m * k, k=k, rowptr=rowptr, col=col, val=val, lb=lb, ub=ub, lo=torch.zeros(n, dtype=torch.float32, device=dev),
                hi=torch.ones(n, dtype=torch.float32, device=dev), x0=torch.zeros(n, dtype=torch.float32, device=dev), x_true=xs)
