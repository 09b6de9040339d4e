"""Seeded synthetic inputs for the VIPIR database scan (host twin, numpy).

This module holds NO arithmetic of the method (no products, limbs or reductions of the
scan): it only produces the bytes of D and the words of Q.  It is the one piece of code the
CPU oracle's tests and the CUDA path's tests both use, so that both see the same inputs.

Generator: the SplitMix64 sequence with random access.
    fin(z)        = z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^ z>>31
    word(key, i)  = fin(key + (i+1) * 0x9E3779B97F4A7C15)          (all mod 2^64)
    key(seed, s)  = word(word(seed, 0) ^ (s * 0xD1342543DE82EF95), 0)   s = stream id
Byte n of a "uniform bytes" buffer is byte (n & 7) of word(key, n >> 3), little-endian, so
u8 / u16 / u32 buffers are all the same byte stream reinterpreted.  Residues mod p are
word(key, n) % p, one word per element.

The paper uses no dataset: the DB is arbitrary bytes and PIR cost is data-independent
(PAPER.md:22, :331), so uniform random bytes are its workload; shapes follow its
SimplePIR-style square layouts D0 ~ sqrt(D).  See DESIGN.md "Input recipe".
The device twin is generator.cu (same functions, tested equal in tests/).
"""
from __future__ import annotations

import numpy as np

GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_STREAM_MUL = 0xD1342543DE82EF95
_MASK64 = (1 << 64) - 1

STREAM_DB = 1
STREAM_QUERY = 2
STREAM_MG_H = 3  # parallel modular GEMMs: H, C, G residues
STREAM_MG_C = 4
STREAM_MG_G = 5


def _fin(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def words(key: int, start: int, count: int) -> np.ndarray:
    """word(key, i) for i in [start, start+count) as uint64."""
    with np.errstate(over="ignore"):
        i = np.arange(start + 1, start + 1 + count, dtype=np.uint64)
        return _fin(np.uint64(key) + i * GAMMA)


def _word_scalar(key: int, i: int) -> int:
    z = (key + (i + 1) * int(GAMMA)) & _MASK64
    z ^= z >> 30
    z = (z * int(_M1)) & _MASK64
    z ^= z >> 27
    z = (z * int(_M2)) & _MASK64
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int) -> int:
    return _word_scalar(_word_scalar(seed & _MASK64, 0) ^ ((stream * _STREAM_MUL) & _MASK64), 0)


def uniform_bytes(key: int, start_byte: int, nbytes: int) -> np.ndarray:
    """Bytes [start_byte, start_byte + nbytes) of the stream, as uint8."""
    w0 = start_byte >> 3
    w1 = (start_byte + nbytes + 7) >> 3
    buf = words(key, w0, w1 - w0).astype("<u8").view(np.uint8)
    off = start_byte - (w0 << 3)
    return buf[off:off + nbytes].copy()


def residues(key: int, start: int, count: int, p: int) -> np.ndarray:
    """word(key, n) % p for n in [start, start+count), as uint32."""
    return (words(key, start, count) % np.uint64(p)).astype(np.uint32)


# ---- the workloads' tensors --------------------------------------------------------------

def db_rows(seed: int, rows: int, cols: int, db_bits: int, row0: int = 0, nrows: int | None = None):
    """Rows [row0, row0+nrows) of the rows x cols database, uniform over the element range."""
    nrows = rows - row0 if nrows is None else nrows
    eb = db_bits // 8
    key = stream_key(seed, STREAM_DB)
    raw = uniform_bytes(key, row0 * cols * eb, nrows * cols * eb)
    dt = np.uint8 if db_bits == 8 else np.dtype("<u2")
    return raw.view(dt).reshape(nrows, cols)


def query(seed: int, cols: int, batch: int, moduli=None) -> np.ndarray:
    """Q [T][batch][cols] uint32: uniform words (q = 2^32) or uniform residues mod each p_t."""
    key = stream_key(seed, STREAM_QUERY)
    if moduli is None or len(moduli) == 0:
        return uniform_bytes(key, 0, 4 * batch * cols).view("<u4").reshape(1, batch, cols).astype(np.uint32)
    n = batch * cols
    out = np.empty((len(moduli), batch, cols), dtype=np.uint32)
    for t, p in enumerate(moduli):
        out[t] = residues(key, t * n, n, int(p)).reshape(batch, cols)
    return out


def modgemm_operand(seed: int, stream: int, moduli, n_coeff: int, per_problem: int,
                    c0: int = 0, nc: int | None = None) -> np.ndarray:
    """Operand of the parallel modular GEMMs H*C + (0|G): uniform residues mod
    q_t, flat index ((t*n_coeff + c)*per_problem + i) -> word(key, index) % q_t.  Returns
    [T][nc][per_problem] uint32 for coefficients [c0, c0+nc) (the caller reshapes the last axis)."""
    nc = n_coeff - c0 if nc is None else nc
    key = stream_key(seed, stream)
    out = np.empty((len(moduli), nc, per_problem), dtype=np.uint32)
    for t, p in enumerate(moduli):
        start = (t * n_coeff + c0) * per_problem
        out[t] = residues(key, start, nc * per_problem, int(p)).reshape(nc, per_problem)
    return out


# ---- RNS primes for config 5 ---------------------------------------------------------------

def _is_prime(n: int) -> bool:
    if n < 2:
        return False
    for p in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        if n % p == 0:
            return n == p
    d, s = n - 1, 0
    while d % 2 == 0:
        d //= 2
        s += 1
    for a in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):  # deterministic below 3.3e24
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(s - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def rns_primes(seed: int = 0, count: int = 2, below: int = 1 << 30, modulus: int = 8192):
    """The seed-th .. (seed+count-1)-th primes of the descending list of primes p < below
    with p = 1 (mod modulus).  BASELINE.json config 5: "two distinct primes below 2^30
    (q = 1 mod 8192, fixed by the build from the seed and recorded)"; 8192 = 2N for the
    paper's N = 2^12 (q_i = 1 mod 2N)."""
    out = []
    skip = seed
    p = ((below - 2) // modulus) * modulus + 1
    while len(out) < count and p > 1:
        if _is_prime(p):
            if skip > 0:
                skip -= 1
            else:
                out.append(p)
        p -= modulus
    return out
