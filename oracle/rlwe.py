"""Toy RLWE poly-HE client and naive negacyclic NTT, used only to pin the modular-GEMM oracle end
to end -- TEST INFRASTRUCTURE.

Ring and scheme follow PAPER.md:528-559 (Appendix A.2): R_q = Z_q[X]/(X^N + 1), ternary secret
s(X), uniform a(X), small error e(X),

    Encrypt(m(X)) -> ct = (a(X), b(X))  with  a(X)*s(X) + b(X) = Delta*m(X) + e(X)  (mod q),
    phase(ct) = a*s + b,   Decrypt = round(phase / Delta)  given |e_i| < Delta/2,
    Delta = floor(q / p).

Prime selection follows PAPER.md:578-589 (Appendix A.4): q = 1 mod 2N ("a sufficient condition
for enabling NTT") and q = 1 mod p, so Delta*p + 1 = q.

Tiptoe-style ring packing follows PAPER.md:633-667 (Appendix C.1), eq. (3):
    (0, Delta*iota(b)) + sum_i iota(A_i) * ct_Pack,i  ->  ct_res,   ct_Pack,i = Encrypt(s_i),
whose phase is Delta*iota(b + sum_i A_i s_i) + sum_i iota(A_i)*e_i(X) = Delta*iota(m) + noise.
In the NTT domain this is the server's  H*C + (0 | G): H = NTT(iota(A_i)) per
group of N LWE ciphertexts, C = NTT of the n x 2 polynomial matrix [a_i | b_i], G = NTT(Delta*iota(b)).

The NTT here is the definition, O(N^2): evaluation at the odd powers of a primitive 2N-th root of
unity psi, X -> psi^(2c+1), c = 0..N-1 (these are the roots of X^N + 1, so products in R_q become
point-wise products; section 2.3).  Everything is Python big integers.
"""
from __future__ import annotations

import numpy as np


def is_prime(n: int) -> bool:
    if n < 2:
        return False
    if n % 2 == 0:
        return n == 2
    f = 3
    while f * f <= n:
        if n % f == 0:
            return False
        f += 2
    return True


def find_prime(N: int, p: int, below: int) -> int:
    """Largest prime q < below with q = 1 mod 2N and q = 1 mod p."""
    step = np.lcm(2 * N, p)
    q = (below - 2) // int(step) * int(step) + 1
    while q > 1:
        if is_prime(q):
            return int(q)
        q -= int(step)
    raise ValueError("no such prime")


def primitive_2n_root(N: int, q: int) -> int:
    """psi with psi^N = -1 mod q (so psi has order exactly 2N)."""
    assert (q - 1) % (2 * N) == 0
    for g in range(2, q):
        psi = pow(g, (q - 1) // (2 * N), q)
        if pow(psi, N, q) == q - 1:
            return psi
    raise ValueError("no root found")


def ntt(poly, q: int, psi: int):
    """[poly(psi^(2c+1)) mod q for c < N] -- the negacyclic NTT by its definition."""
    N = len(poly)
    out = []
    for c in range(N):
        x = pow(psi, 2 * c + 1, q)
        acc, xp = 0, 1
        for j in range(N):
            acc = (acc + int(poly[j]) * xp) % q
            xp = xp * x % q
        out.append(acc)
    return out


def intt(vals, q: int, psi: int):
    """Inverse of ntt(): coefficient j = N^-1 * sum_c vals[c] * psi^(-(2c+1) j)."""
    N = len(vals)
    n_inv = pow(N, -1, q)
    psi_inv = pow(psi, -1, q)
    out = []
    for j in range(N):
        acc = 0
        for c in range(N):
            acc = (acc + int(vals[c]) * pow(psi_inv, (2 * c + 1) * j, q)) % q
        out.append(acc * n_inv % q)
    return out


def negacyclic_mul(f, g, q: int):
    """Schoolbook product in Z_q[X]/(X^N + 1): X^N = -1."""
    N = len(f)
    out = [0] * N
    for i in range(N):
        for j in range(N):
            k = i + j
            term = int(f[i]) * int(g[j])
            if k >= N:
                out[k - N] = (out[k - N] - term) % q
            else:
                out[k] = (out[k] + term) % q
    return out


def keygen(N: int, rng: np.random.Generator):
    """Uniform ternary secret polynomial."""
    return [int(x) for x in rng.integers(-1, 2, size=N)]


def encrypt(m_poly, s_poly, q: int, delta: int, rng: np.random.Generator, err_bound: int = 1):
    """(a, b) with a*s + b = Delta*m + e mod q; e uniform in [-err_bound, err_bound] (a small
    error stands in for the sigma = 3.2 Gaussian: only |e| < Delta/2 matters)."""
    N = len(s_poly)
    if q < (1 << 62):
        a = [int(x) for x in rng.integers(0, q, size=N)]
    else:  # an RNS modulus q = q_0 q_1 q_2 ~ 2^87: 128 random bits reduced mod q
        a = [int.from_bytes(rng.bytes(16), "little") % q for _ in range(N)]
    e = [int(x) for x in rng.integers(-err_bound, err_bound + 1, size=N)]
    a_s = negacyclic_mul(a, [x % q for x in s_poly], q)
    b = [(delta * int(m_poly[j]) + e[j] - a_s[j]) % q for j in range(N)]
    return a, b


def phase(a, b, s_poly, q: int):
    """a*s + b mod q, centred to [-(q-1)/2, (q-1)/2]."""
    a_s = negacyclic_mul(a, [x % q for x in s_poly], q)
    out = []
    for j in range(len(b)):
        v = (a_s[j] + int(b[j])) % q
        out.append(v - q if v > (q - 1) // 2 else v)
    return out


def decrypt(a, b, s_poly, q: int, delta: int, p: int):
    """round(phase / Delta) mod p."""
    return [((2 * v + delta) // (2 * delta)) % p for v in phase(a, b, s_poly, q)]
