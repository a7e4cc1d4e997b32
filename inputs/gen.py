"""ctypes wrapper over inputs/libgen.so (counter-based normal generator, bf16 conversions)."""
import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        u64, dbl, vp = ctypes.c_uint64, ctypes.c_double, ctypes.c_void_p
        _lib.gen_normal_f32.argtypes = [u64, u64, u64, u64, dbl, dbl, vp]
        _lib.gen_normal_bf16.argtypes = [u64, u64, u64, u64, dbl, dbl, vp]
        _lib.gen_f32_to_bf16.argtypes = [vp, u64, vp]
        _lib.gen_bf16_to_f32.argtypes = [vp, u64, vp]
        for f in (_lib.gen_normal_f32, _lib.gen_normal_bf16, _lib.gen_f32_to_bf16, _lib.gen_bf16_to_f32):
            f.restype = None
    return _lib


def normal(seed: int, tid: int, shape, std: float = 1.0, mean: float = 0.0, bf16: bool = False,
           out: np.ndarray | None = None, i0: int = 0) -> np.ndarray:
    """Tensor `tid` of seed `seed`: fl32(mean + std*N(0,1)); bf16=True returns the bf16 bits as uint16."""
    n = int(np.prod(shape))
    dt = np.uint16 if bf16 else np.float32
    if out is None:
        out = np.empty(shape, dtype=dt)
    assert out.dtype == dt and out.size == n and out.flags.c_contiguous
    fn = lib().gen_normal_bf16 if bf16 else lib().gen_normal_f32
    fn(seed, tid, i0, n, mean, std, out.ctypes.data)
    return out


def f32_to_bf16(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    out = np.empty(a.shape, dtype=np.uint16)
    lib().gen_f32_to_bf16(a.ctypes.data, a.size, out.ctypes.data)
    return out


def bf16_to_f32(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint16)
    out = np.empty(a.shape, dtype=np.float32)
    lib().gen_bf16_to_f32(a.ctypes.data, a.size, out.ctypes.data)
    return out
