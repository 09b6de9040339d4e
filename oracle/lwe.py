"""Toy LWE scalar-HE client, used only to pin the oracle end to end -- TEST INFRASTRUCTURE.

Follows PAPER.md:498-526 (Appendix A.1) with the paper's parameters p = 2^8, q = 2^32,
Delta = q/p = 2^24, sigma = 3.2, ternary secret; the LWE degree n is a free argument
(the paper uses n = 1280; tests use a small n -- the product's arithmetic does not
depend on it).

  Encrypt(m) -> ct = (a, b) in Z_q^{n+1} with  b + a^T s = Delta*m + e  (mod q)   (:502-504)
  phase(ct)  =  b + a^T s                                                         (:508)
  Decrypt    =  round(phase / Delta)  ->  m  provided |e| < Delta/2               (:512-514)

SimplePIR query for column i* (section 2.5): D0 ciphertexts, the i*-th
encrypts one and the others zero; together a D0 x (n+1) matrix.  In the library's layout
(query-major, [batch][cols]) that is Q[j][k] = a_k[j] for j < n and Q[n][k] = b_k.
The server's product D*Q then holds, for row r, the ciphertext (H[r][0..n-1], ans[r]) of
D[r][i*], whose noise is sum_k D[r][k]*e_k.

Readings: R12 sign convention is the paper's (b = Delta*m + e - a^T s);
R13 the error is a rounded N(0, sigma^2) draw, resampled while |e| >= 6*sigma;
R14 decryption is ((phase + 2^23) >> 24) & 0xFF in wrapping 32-bit arithmetic.
"""
from __future__ import annotations

import numpy as np

P_BITS = 8
Q_BITS = 32
DELTA = 1 << (Q_BITS - P_BITS)  # 2^24
SIGMA = 3.2
MASK = (1 << Q_BITS) - 1


def keygen(n: int, rng: np.random.Generator) -> np.ndarray:
    """Uniform ternary secret in {-1,0,1}^n."""
    return rng.integers(-1, 2, size=n, dtype=np.int64)


def sample_error(shape, rng: np.random.Generator) -> np.ndarray:
    """Rounded Gaussian, sigma = 3.2, clipped so |e| < 6 sigma by resampling (:500, R13)."""
    e = np.rint(rng.normal(0.0, SIGMA, size=shape)).astype(np.int64)
    bad = np.abs(e) >= 6 * SIGMA
    while bad.any():
        e[bad] = np.rint(rng.normal(0.0, SIGMA, size=int(bad.sum()))).astype(np.int64)
        bad = np.abs(e) >= 6 * SIGMA
    return e


def simplepir_query(cols: int, i_star: int, s: np.ndarray, rng: np.random.Generator):
    """Encrypted one-hot of i_star.  Returns (Q [n+1][cols] uint32, e [cols] int64)."""
    n = s.size
    a = rng.integers(0, 1 << Q_BITS, size=(cols, n), dtype=np.uint64)  # a_k uniform in Z_q
    e = sample_error(cols, rng)
    m = np.zeros(cols, dtype=np.int64)
    m[i_star] = 1
    # a_k^T s with Python-int exactness (object dtype), then b_k = Delta*m_k + e_k - a_k^T s mod q
    a_dot_s = (a.astype(object) * s.astype(object)[None, :]).sum(axis=1)
    b = np.array([(DELTA * int(m[k]) + int(e[k]) - int(a_dot_s[k])) & MASK for k in range(cols)],
                 dtype=np.uint64)
    Q = np.empty((n + 1, cols), dtype=np.uint32)
    Q[:n, :] = a.T.astype(np.uint32)
    Q[n, :] = b.astype(np.uint32)
    return Q, e


def decrypt_answer(A: np.ndarray, s: np.ndarray) -> np.ndarray:
    """A is the server's answer [n+1][rows] (hint part rows 0..n-1, b part row n).
    Returns the decrypted plaintext byte per DB row (R14)."""
    n = s.size
    rows = A.shape[1]
    out = np.empty(rows, dtype=np.uint8)
    s_obj = [int(x) for x in s]
    for r in range(rows):
        phase = int(A[n, r])
        for j in range(n):
            phase += int(A[j, r]) * s_obj[j]
        phase &= MASK
        out[r] = ((phase + (DELTA >> 1)) >> (Q_BITS - P_BITS)) & 0xFF
    return out


def worst_case_noise_ok(cols: int) -> bool:
    """|sum_k D[r][k] e_k| <= 255 * 19 * cols must stay below Delta/2 = 2^23."""
    return 255 * 19 * cols < (DELTA >> 1)


def decrypt_answer_switched(A_sw: np.ndarray, s: np.ndarray, bits: int = 18) -> np.ndarray:
    """Decrypt an answer whose words were modulus-switched to 2^bits:
    same phase computation mod 2^bits with scale Delta' = 2^bits / p."""
    n = s.size
    rows = A_sw.shape[1]
    q2 = 1 << bits
    delta2 = q2 >> P_BITS
    out = np.empty(rows, dtype=np.uint8)
    s_obj = [int(x) for x in s]
    for r in range(rows):
        phase = int(A_sw[n, r])
        for j in range(n):
            phase += int(A_sw[j, r]) * s_obj[j]
        phase %= q2
        out[r] = ((phase + (delta2 >> 1)) // delta2) & 0xFF
    return out
