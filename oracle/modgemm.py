"""Python face of oracle/vipir_modgemm_oracle.c -- TEST INFRASTRUCTURE ONLY.

``modgemm`` is the plain definition of VIPIR's parallel INT32 modular GEMMs
``Out = H*C + (0 | G) mod q_t`` (PAPER.md:216 section 3.5.2; :261-265 section 4.2);
``modgemm_lazy`` follows the paper's lazy-reduction method;
``modgemm_bruteforce`` is a pure-Python big-integer loop for tiny shapes only.

Layouts (uint32, numpy, host):  H [T][NC][M][K],  C [T][NC][ncols][K],  G [T][NC][gcols][M] or
None,  Out [T][NC][ncols][M].  G is added to the LAST gcols columns.  Nothing here imports the
CUDA package.
"""
from __future__ import annotations

import numpy as np

from .vipir_oracle import _load, _ptr


def _prep(H, C, G, moduli):
    mods = np.ascontiguousarray(moduli, dtype=np.uint32).reshape(-1)
    H = np.ascontiguousarray(H, dtype=np.uint32)
    C = np.ascontiguousarray(C, dtype=np.uint32)
    if H.ndim != 4 or C.ndim != 4:
        raise ValueError("H must be [T][NC][M][K] and C [T][NC][ncols][K]")
    T, NC, M, K = H.shape
    if mods.size != T or C.shape[0] != T or C.shape[1] != NC or C.shape[3] != K:
        raise ValueError(f"shape mismatch: H {H.shape}, C {C.shape}, {mods.size} moduli")
    ncols = C.shape[2]
    gcols = 0
    if G is not None:
        G = np.ascontiguousarray(G, dtype=np.uint32)
        if G.ndim != 4 or G.shape[0] != T or G.shape[1] != NC or G.shape[3] != M or G.shape[2] > ncols:
            raise ValueError(f"G must be [T][NC][gcols<=ncols][M], got {G.shape}")
        gcols = G.shape[2]
    Out = np.zeros((T, NC, ncols, M), dtype=np.uint32)
    return mods, H, C, G, Out, T, NC, M, K, ncols, gcols


def modgemm(H, C, G, moduli, nthreads: int = 1) -> np.ndarray:
    """The definition."""
    mods, H, C, G, Out, T, NC, M, K, ncols, gcols = _prep(H, C, G, moduli)
    rc = _load().vipir_oracle_modgemm(T, NC, M, K, ncols, gcols, _ptr(mods), _ptr(H), _ptr(C), _ptr(G),
                                      _ptr(Out), int(nthreads))
    if rc != 0:
        raise ValueError(f"vipir_oracle_modgemm failed: {rc}")
    return Out


def modgemm_lazy(H, C, G, moduli, defer: int = 32) -> np.ndarray:
    """The paper's method: 64-bit accumulators, one reduction per `defer` MACs.
    Raises OverflowError when its precondition (q < 2^29, inputs < q, defer <= 32) fails."""
    mods, H, C, G, Out, T, NC, M, K, ncols, gcols = _prep(H, C, G, moduli)
    rc = _load().vipir_oracle_modgemm_lazy(T, NC, M, K, ncols, gcols, _ptr(mods), _ptr(H), _ptr(C), _ptr(G),
                                           _ptr(Out), int(defer))
    if rc == -3:
        raise OverflowError("lazy reduction precondition violated (q >= 2^29, input >= q or defer > 32)")
    if rc != 0:
        raise ValueError(f"vipir_oracle_modgemm_lazy failed: {rc}")
    return Out


def modgemm_bruteforce(H, C, G, moduli) -> np.ndarray:
    """Pure-Python big-integer loops; tiny shapes only (pins the C routine)."""
    H = np.asarray(H)
    C = np.asarray(C)
    T, NC, M, K = H.shape
    ncols = C.shape[2]
    gcols = 0 if G is None else np.asarray(G).shape[2]
    out = np.zeros((T, NC, ncols, M), dtype=np.uint32)
    for t in range(T):
        q = int(moduli[t])
        for c in range(NC):
            for j in range(ncols):
                for m in range(M):
                    s = 0
                    for k in range(K):
                        s += int(H[t, c, m, k]) * int(C[t, c, j, k])
                    if j >= ncols - gcols:
                        s += int(G[t, c, j - (ncols - gcols), m])
                    out[t, c, j, m] = s % q
    return out
