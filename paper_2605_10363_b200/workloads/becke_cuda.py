"""ctypes wrapper of workloads/becke.cu (input generation only; see generate.becke_weights)."""
from __future__ import annotations

import ctypes
import os

import numpy as np

_LIB = None
_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libkldi_workloads.so")


def available() -> bool:
    return os.path.exists(_PATH)


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(_PATH)
        _LIB.wl_becke_partition.restype = ctypes.c_int
        _LIB.wl_becke_partition.argtypes = [ctypes.c_void_p] * 5 + [ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p]
    return _LIB


def becke_partition(atom_xyz: np.ndarray, pts: np.ndarray, owner: np.ndarray) -> np.ndarray:
    import torch

    dev = torch.device("cuda")
    a = torch.as_tensor(np.ascontiguousarray(atom_xyz, dtype=np.float64), device=dev)
    rab = torch.cdist(a, a)
    rab.fill_diagonal_(1.0)
    inv = (1.0 / rab).contiguous()
    p = torch.as_tensor(np.ascontiguousarray(pts, dtype=np.float64), device=dev)
    o = torch.as_tensor(np.ascontiguousarray(owner, dtype=np.int32), device=dev)
    out = torch.empty(p.shape[0], dtype=torch.float64, device=dev)
    rc = _lib().wl_becke_partition(a.data_ptr(), inv.data_ptr(), p.data_ptr(), o.data_ptr(), out.data_ptr(),
                                   p.shape[0], a.shape[0], torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"wl_becke_partition failed rc={rc}")
    torch.cuda.synchronize()
    return out.cpu().numpy()
