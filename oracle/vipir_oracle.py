"""Python face of the CPU oracle (oracle/vipir_oracle.c) -- TEST INFRASTRUCTURE ONLY.

``dbmul`` is the plain definition  A[t][b][r] = (sum_k D[r][k] * Q[t][b][k]) mod q_t
(section 2.5; modulus PAPER.md:238 section 4; residues PAPER.md:95-97);
``dbmul_limbs`` follows the paper's four-limb method (section 4.1);
``dbmul_bruteforce`` is a pure-Python big-integer triple loop for tiny shapes only.

Nothing here imports the CUDA package; arrays are numpy, on the host.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "vipir_oracle.c"
_SRCS = [_SRC, _HERE / "vipir_modgemm_oracle.c",  # NEXT-4: parallel modular GEMMs (own file, same library)
         _HERE / "vipir_ntt_oracle.c"]             # lift + forward NTT producing G and H (own file, same library)
_LIB = _HERE / "libvipir_oracle.so"
_lib = None


def lib_path() -> Path:
    return _LIB


def build(force: bool = False) -> Path:
    """Compile oracle/*.c with gcc (plain C, -O2, OpenMP for the outer loop)."""
    if force or not _LIB.exists() or any(_LIB.stat().st_mtime < f.stat().st_mtime for f in _SRCS):
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.run(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
             "-o", str(tmp), *map(str, _SRCS)],
            check=True,
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        u64, u32, i32, vp = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, ctypes.c_void_p
        lib.vipir_oracle_dbmul.restype = ctypes.c_int
        lib.vipir_oracle_dbmul.argtypes = [u64, u64, u32, i32, u32, vp, vp, vp, vp, i32]
        lib.vipir_oracle_dbmul_limbs.restype = ctypes.c_int
        lib.vipir_oracle_dbmul_limbs.argtypes = [u64, u64, u32, i32, u32, vp, vp, vp, vp, u64]
        lib.vipir_oracle_dbmul_signed.restype = ctypes.c_int
        lib.vipir_oracle_dbmul_signed.argtypes = [u64, u64, u32, i32, u32, vp, vp, vp, vp]
        lib.vipir_oracle_modswitch.restype = ctypes.c_int
        lib.vipir_oracle_modswitch.argtypes = [vp, u64, i32]
        lib.vipir_oracle_modgemm.restype = ctypes.c_int
        lib.vipir_oracle_modgemm.argtypes = [u32, u64, u64, u64, u64, u64, vp, vp, vp, vp, vp, i32]
        lib.vipir_oracle_modgemm_lazy.restype = ctypes.c_int
        lib.vipir_oracle_modgemm_lazy.argtypes = [u32, u64, u64, u64, u64, u64, vp, vp, vp, vp, vp, u32]
        lib.vipir_oracle_ntt_lift.restype = ctypes.c_int
        lib.vipir_oracle_ntt_lift.argtypes = [u32, u32, u32, u32, vp, vp, vp, u32, i32, i32, vp, vp, i32]
        _lib = lib
    return _lib


def _prep(D, Q, moduli):
    D = np.ascontiguousarray(D)
    if D.dtype == np.uint8:
        db_bits = 8
    elif D.dtype == np.uint16:
        db_bits = 16
    else:
        raise TypeError("D must be uint8 or uint16")
    if D.ndim != 2:
        raise ValueError("D must be rows x cols")
    rows, cols = D.shape
    mods = None if moduli is None or len(moduli) == 0 else np.ascontiguousarray(moduli, dtype=np.uint32)
    T = 1 if mods is None else int(mods.size)
    Q = np.ascontiguousarray(Q, dtype=np.uint32)
    if Q.ndim == 1:
        Q = Q.reshape(1, 1, -1)
    elif Q.ndim == 2:
        Q = Q.reshape(1, *Q.shape)
    if Q.ndim != 3 or Q.shape[0] != T or Q.shape[2] != cols:
        raise ValueError(f"Q must be [T={T}][batch][cols={cols}], got {Q.shape}")
    batch = Q.shape[1]
    A = np.zeros((T, batch, rows), dtype=np.uint32)
    return D, Q, mods, db_bits, rows, cols, batch, T, A


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def dbmul(D, Q, moduli=None, nthreads: int = 1) -> np.ndarray:
    """The definition.  D rows x cols (u8/u16), Q [T][B][cols] u32 -> A [T][B][rows] u32."""
    D, Q, mods, db_bits, rows, cols, batch, T, A = _prep(D, Q, moduli)
    rc = _load().vipir_oracle_dbmul(rows, cols, batch, db_bits, 0 if mods is None else T,
                                    _ptr(mods), _ptr(D), _ptr(Q), _ptr(A), int(nthreads))
    if rc != 0:
        raise ValueError(f"vipir_oracle_dbmul failed: {rc}")
    return A


def dbmul_limbs(D, Q, moduli=None, k_chunk: int = 32768) -> np.ndarray:
    """The paper's limb method; raises OverflowError if an INT32
    partial product would have overflowed for this k_chunk."""
    D, Q, mods, db_bits, rows, cols, batch, T, A = _prep(D, Q, moduli)
    rc = _load().vipir_oracle_dbmul_limbs(rows, cols, batch, db_bits, 0 if mods is None else T,
                                          _ptr(mods), _ptr(D), _ptr(Q), _ptr(A), int(k_chunk))
    if rc == -2:
        raise OverflowError("an INT32 limb accumulator overflowed; k_chunk too large")
    if rc != 0:
        raise ValueError(f"vipir_oracle_dbmul_limbs failed: {rc}")
    return A


def dbmul_signed(D, Q, moduli=None) -> np.ndarray:
    """The definition with SIGNED database elements (D given as uint8/uint16 bit patterns or as
    int8/int16); centred plaintexts."""
    D = np.ascontiguousarray(D)
    if D.dtype in (np.int8, np.int16):
        D = D.view(np.uint8 if D.dtype == np.int8 else np.uint16)
    D, Q, mods, db_bits, rows, cols, batch, T, A = _prep(D, Q, moduli)
    rc = _load().vipir_oracle_dbmul_signed(rows, cols, batch, db_bits, 0 if mods is None else T,
                                           _ptr(mods), _ptr(D), _ptr(Q), _ptr(A))
    if rc != 0:
        raise ValueError(f"vipir_oracle_dbmul_signed failed: {rc}")
    return A


def modswitch(A, bits: int = 18) -> np.ndarray:
    """Scalar-HE modulus switch 2^32 -> 2^bits of every word; returns a copy."""
    out = np.ascontiguousarray(A, dtype=np.uint32).copy()
    rc = _load().vipir_oracle_modswitch(_ptr(out), out.size, int(bits))
    if rc != 0:
        raise ValueError(f"vipir_oracle_modswitch failed: {rc}")
    return out


def dbmul_bruteforce(D, Q, moduli=None):
    """Pure-Python big-integer triple loop; tiny shapes only (pins the C routine)."""
    D = np.asarray(D)
    Q = np.asarray(Q)
    mods = [1 << 32] if moduli is None or len(moduli) == 0 else [int(m) for m in moduli]
    if Q.ndim == 1:
        Q = Q.reshape(1, 1, -1)
    elif Q.ndim == 2:
        Q = Q.reshape(1, *Q.shape)
    rows, cols = D.shape
    out = np.zeros((len(mods), Q.shape[1], rows), dtype=np.uint32)
    for t, q in enumerate(mods):
        for b in range(Q.shape[1]):
            for r in range(rows):
                s = 0
                for k in range(cols):
                    s += int(D[r, k]) * int(Q[t, b, k])
                out[t, b, r] = s % q
    return out
