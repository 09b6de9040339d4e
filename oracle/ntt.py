"""Python face of oracle/vipir_ntt_oracle.c -- TEST INFRASTRUCTURE ONLY.

``ntt_lift`` is the plain definition of the lift + forward negacyclic NTT that turns the scan's
scalar-HE output (and the hint) into the polynomial matrices G and H of the ring-packing stage
(PAPER.md:214 section 3.5.2, :667 Appendix C.1, :95-101 section 2.3), written in the layout of
the modular GEMMs' operands.  ``smallest_psi`` is the reading taken for the
root of unity (R24).  Nothing here imports the CUDA package.
"""
from __future__ import annotations

import numpy as np

from .vipir_oracle import _load, _ptr

LAYOUT_G, LAYOUT_H = 0, 1


def smallest_psi(N: int, q: int) -> int:
    """The smallest positive integer psi with psi^N = -1 mod q (a primitive 2N-th root of unity)."""
    if (q - 1) % (2 * N) != 0:
        raise ValueError("q != 1 mod 2N")
    for x in range(2, q):
        if pow(x, N, q) == q - 1:
            return x
    raise ValueError("no primitive 2N-th root of unity")


def ntt_lift(X, N: int, moduli, psi, scale, p_bits: int, centered: bool = False, out_layout: int = LAYOUT_G,
             nthreads: int = 1) -> np.ndarray:
    """X [n_a][M*N] u32 words < 2^p_bits  ->  O [T][N][n_a][M] (LAYOUT_G) or [T][N][M][n_a] (LAYOUT_H)."""
    X = np.ascontiguousarray(X, dtype=np.uint32)
    if X.ndim != 2 or X.shape[1] % N != 0:
        raise ValueError("X must be [n_a][M*N]")
    n_a, M = X.shape[0], X.shape[1] // N
    mods = np.ascontiguousarray(moduli, dtype=np.uint32).reshape(-1)
    ps = np.ascontiguousarray(psi, dtype=np.uint32).reshape(-1)
    sc = np.ascontiguousarray(scale, dtype=np.uint32).reshape(-1)
    T = mods.size
    if ps.size != T or sc.size != T:
        raise ValueError("one psi and one scale per modulus")
    shape = (T, N, n_a, M) if out_layout == LAYOUT_G else (T, N, M, n_a)
    O = np.zeros(shape, dtype=np.uint32)
    lib = _load()
    rc = lib.vipir_oracle_ntt_lift(T, n_a, M, N, _ptr(mods), _ptr(ps), _ptr(sc), int(p_bits), int(bool(centered)),
                                   int(out_layout), _ptr(X), _ptr(O), int(nthreads))
    if rc == -2:
        raise ValueError("psi is not a primitive 2N-th root of unity")
    if rc == -3:
        raise ValueError("an input word is >= 2^p_bits")
    if rc != 0:
        raise ValueError(f"vipir_oracle_ntt_lift failed: {rc}")
    return O
