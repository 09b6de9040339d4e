"""Measurement aids for bench.py (ceilings/libvipir_ceilings.so, built from ceilings.cu): what the part does at
best on the unit a libvipir kernel is bound by.  Bench-only: not product code, no arithmetic of the method."""
from __future__ import annotations

import ctypes
from pathlib import Path

_LIB_PATH = Path(__file__).resolve().parent / "libvipir_ceilings.so"
_lib = None


def _load():
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2606_11536_b200.build`")
        lib = ctypes.CDLL(str(_LIB_PATH))
        lib.vipir_ceiling_mma_i8.restype = ctypes.c_int
        lib.vipir_ceiling_mma_i8.argtypes = [ctypes.c_uint32, ctypes.POINTER(ctypes.c_uint32), ctypes.c_void_p]
        lib.vipir_ceiling_butterflies.restype = ctypes.c_int
        lib.vipir_ceiling_butterflies.argtypes = [ctypes.c_uint32, ctypes.c_uint32, ctypes.POINTER(ctypes.c_uint32),
                                                  ctypes.c_void_p]
        _lib = lib
    return _lib


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def mma_i8(iters: int) -> float:
    """Enqueue the pure tcgen05.mma.kind::i8 loop; returns the int8 ops (2 per MAC) the launch executes."""
    pairs = ctypes.c_uint32(0)
    rc = _load().vipir_ceiling_mma_i8(iters, ctypes.byref(pairs), _stream())
    if rc:
        raise RuntimeError(f"vipir_ceiling_mma_i8 failed: {rc}")
    return float(pairs.value) * iters * 4 * 2.0 * 256 * 256 * 32


def butterflies(iters: int, q: int) -> float:
    """Enqueue the register-only Harvey butterfly loop; returns the butterflies the launch executes."""
    blocks = ctypes.c_uint32(0)
    rc = _load().vipir_ceiling_butterflies(iters, q, ctypes.byref(blocks), _stream())
    if rc:
        raise RuntimeError(f"vipir_ceiling_butterflies failed: {rc}")
    return float(blocks.value) * 512 * iters * 32
