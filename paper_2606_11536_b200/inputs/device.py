"""Device twin of generator.py: fills torch CUDA tensors with the same seeded streams
(inputs/libvipir_inputs.so, built from generator.cu).  No arithmetic of the method."""
from __future__ import annotations

import ctypes
from pathlib import Path

from . import generator as g

_LIB_PATH = Path(__file__).resolve().parent / "libvipir_inputs.so"
_lib = None


def _load():
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2606_11536_b200.build`")
        lib = ctypes.CDLL(str(_LIB_PATH))
        lib.vipir_inputs_fill_bytes.restype = ctypes.c_int
        lib.vipir_inputs_fill_bytes.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_void_p]
        lib.vipir_inputs_fill_mod.restype = ctypes.c_int
        lib.vipir_inputs_fill_mod.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64,
                                              ctypes.c_uint32, ctypes.c_void_p]
        lib.vipir_inputs_read_only.restype = ctypes.c_int
        lib.vipir_inputs_read_only.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p]
        _lib = lib
    return _lib


def read_only(t):
    """Measurement aid: stream the tensor once with plain loads, discarding the data (bench.py's
    read-only HBM ceiling)."""
    rc = _load().vipir_inputs_read_only(t.data_ptr(), t.numel() * t.element_size(), None, _stream())
    if rc:
        raise RuntimeError(f"vipir_inputs_read_only failed: {rc}")


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def db(seed: int, rows: int, cols: int, db_bits: int, device="cuda"):
    """The rows x cols database on the device: torch.uint8 tensor of shape [rows, cols*db_bits/8]
    (the byte view; a u16 DB is its little-endian bytes)."""
    import torch
    nbytes = rows * cols * (db_bits // 8)
    assert nbytes % 8 == 0
    t = torch.empty(nbytes, dtype=torch.uint8, device=device)
    rc = _load().vipir_inputs_fill_bytes(t.data_ptr(), nbytes, g.stream_key(seed, g.STREAM_DB), _stream())
    if rc:
        raise RuntimeError(f"vipir_inputs_fill_bytes failed: {rc}")
    return t.view(rows, cols * (db_bits // 8))


def query(seed: int, cols: int, batch: int, moduli=None, device="cuda"):
    """Q [T][batch][cols] as a torch.int32 tensor holding the u32 words bit for bit."""
    import torch
    key = g.stream_key(seed, g.STREAM_QUERY)
    T = 1 if not moduli else len(moduli)
    t = torch.empty((T, batch, cols), dtype=torch.int32, device=device)
    lib = _load()
    if not moduli:
        assert (4 * batch * cols) % 8 == 0
        rc = lib.vipir_inputs_fill_bytes(t.data_ptr(), 4 * batch * cols, key, _stream())
    else:
        n = batch * cols
        rc = 0
        for i, p in enumerate(moduli):
            rc |= lib.vipir_inputs_fill_mod(t[i].data_ptr(), n, key, i * n, int(p), _stream())
    if rc:
        raise RuntimeError(f"vipir_inputs fill failed: {rc}")
    return t


def modgemm_operand(seed: int, stream: int, moduli, n_coeff: int, per_problem: int, device="cuda"):
    """Device twin of generator.modgemm_operand: [T][n_coeff][per_problem] torch.int32 (u32 bits)."""
    import torch
    key = g.stream_key(seed, stream)
    t = torch.empty((len(moduli), n_coeff, per_problem), dtype=torch.int32, device=device)
    lib = _load()
    n = n_coeff * per_problem
    rc = 0
    for i, p in enumerate(moduli):
        rc |= lib.vipir_inputs_fill_mod(t[i].data_ptr(), n, key, i * n, int(p), _stream())
    if rc:
        raise RuntimeError(f"vipir_inputs fill failed: {rc}")
    return t
