"""Random 32-byte-sector gather probe (harness/gather_probe.cu -> harness/libpeek_harness.so)."""
from __future__ import annotations

import ctypes
import os
import subprocess

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gather_probe.cu")
_LIB = os.path.join(_HERE, "libpeek_harness.so")
_lib = None


def build(force: bool = False) -> str:
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                    "-Xcompiler", "-fPIC", "-shared", _SRC, "-o", _LIB], check=True)
    return _LIB


def random_gather(buf: torch.Tensor, reads: int, seed: int = 1) -> torch.Tensor:
    """Enqueue `reads` random 32-byte-sector reads over `buf` on the current stream."""
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.harness_random_gather.restype = ctypes.c_int32
        _lib.harness_random_gather.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_uint64,
                                               ctypes.c_void_p, ctypes.c_void_p]
    sink = torch.zeros(1, dtype=torch.uint64, device=buf.device)
    st = _lib.harness_random_gather(ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size(), int(reads),
                                    int(seed), ctypes.c_void_p(sink.data_ptr()),
                                    ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != 0:
        raise RuntimeError("harness_random_gather failed: %d" % st)
    return sink
