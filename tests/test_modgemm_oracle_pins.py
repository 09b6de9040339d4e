"""Pins for the CPU oracle of the parallel modular GEMMs  Out = H*C + (0|G) mod q_t
(SURVEY.md 8(f) NEXT-4; PAPER.md:216 section 3.5.2, :261-265 section 4.2).  No GPU.

Each test checks oracle/ against something the paper or the mathematics fixes -- never against
the oracle's formula retyped and never against the CUDA path: Python big-integer brute force,
closed forms, identity, numpy int64 matmul where nothing can wrap, linearity, the meaning of the
point-wise products as negacyclic polynomial products (naive NTT), a toy RLWE
ring-packing round trip of eq. (3) that must decrypt to the packed LWE
plaintexts, and CRT consistency across RNS primes.
"""
import numpy as np
import pytest

import oracle
from oracle import rlwe
from paper_2606_11536_b200 import inputs

P29 = [536608769, 533463041]          # < 2^29, = 1 mod 2^18
P30 = [1073692673, 1073668097]        # < 2^30, = 1 mod 8192 (BASELINE.json configs[4])


def rng(seed):
    return np.random.default_rng(seed)


def rand_u32(g, shape, hi=1 << 32):
    return g.integers(0, hi, size=shape, dtype=np.uint64).astype(np.uint32)


# ---- brute force on tiny shapes -----------------------------------------------------------------

@pytest.mark.parametrize("NC,M,K,ncols,gcols", [(1, 1, 1, 1, 0), (2, 3, 5, 4, 2), (3, 2, 7, 2, 1), (1, 4, 3, 3, 3),
                                              (2, 5, 2, 6, 0)])
@pytest.mark.parametrize("moduli", [[97], P29, P30, [2, (1 << 30) - 1, 65537]])
def test_bruteforce_tiny(NC, M, K, ncols, gcols, moduli):
    g = rng(NC * 1000 + M * 100 + K * 10 + ncols + gcols)
    T = len(moduli)
    H = rand_u32(g, (T, NC, M, K))          # any u32 is legal, also >= q
    C = rand_u32(g, (T, NC, ncols, K))
    G = rand_u32(g, (T, NC, gcols, M)) if gcols else None
    H[0, 0, 0, 0] = 0xFFFFFFFF
    C[0, 0, 0, 0] = 0xFFFFFFFF
    want = oracle.modgemm_bruteforce(H, C, G, moduli)
    assert np.array_equal(oracle.modgemm(H, C, G, moduli), want)
    for t, q in enumerate(moduli):
        assert (want[t] < q).all()           # canonical range


def test_hand_example():
    # q = 7: H = [[1,2],[3,4]], C columns (1,1) and (2,0), G = [5,6] on the last column:
    # col 0: [1+2, 3+4] = [3, 7] -> [3, 0];  col 1: [2, 6] + [5, 6] = [7, 12] -> [0, 5]
    H = np.array([[[[1, 2], [3, 4]]]], dtype=np.uint32)
    C = np.array([[[[1, 1], [2, 0]]]], dtype=np.uint32)
    G = np.array([[[[5, 6]]]], dtype=np.uint32)
    out = oracle.modgemm(H, C, G, [7])
    assert out[0, 0].tolist() == [[3, 0], [0, 5]]


# ---- closed forms ------------------------------------------------------------------------------

@pytest.mark.parametrize("q", P29 + P30)
def test_all_ones_times_minus_one(q):
    K, M, ncols = 1280, 3, 4                 # K = n = 1280
    H = np.ones((1, 2, M, K), dtype=np.uint32)
    C = np.full((1, 2, ncols, K), q - 1, dtype=np.uint32)
    G = np.full((1, 2, 2, M), 5, dtype=np.uint32)
    out = oracle.modgemm(H, C, G, [q])
    assert (out[0, :, :2, :] == (q - K) % q).all()            # -K mod q, left half: no G
    assert (out[0, :, 2:, :] == (q - K + 5) % q).all()        # right half: + G


def test_all_max_words():
    # every word 2^32-1: sum = K * (2^32-1)^2, G = 2^32-1
    q, K = P30[0], 777
    H = np.full((1, 1, 2, K), 0xFFFFFFFF, dtype=np.uint32)
    C = np.full((1, 1, 2, K), 0xFFFFFFFF, dtype=np.uint32)
    G = np.full((1, 1, 1, 2), 0xFFFFFFFF, dtype=np.uint32)
    out = oracle.modgemm(H, C, G, [q])
    w = (1 << 32) - 1
    assert (out[0, 0, 0] == (K * w * w) % q).all()
    assert (out[0, 0, 1] == (K * w * w + w) % q).all()


def test_identity_h_returns_c_plus_g():
    g = rng(3)
    q, n = P29[0], 6
    H = np.zeros((1, 2, n, n), dtype=np.uint32)
    H[0, :, np.arange(n), np.arange(n)] = 1
    C = rand_u32(g, (1, 2, 4, n), q)
    G = rand_u32(g, (1, 2, 2, n), q)
    out = oracle.modgemm(H, C, G, [q])
    assert np.array_equal(out[0, :, :2, :], C[0, :, :2, :])
    want = (C[0, :, 2:, :].astype(np.uint64) + G[0]) % q
    assert np.array_equal(out[0, :, 2:, :], want.astype(np.uint32))


def test_transposition_probe():
    # H one-hot at (m, pi(m)), C[j][k] = 100*j + k + 1  ->  Out[j][m] = 100*j + pi(m) + 1
    g = rng(4)
    M = K = 9
    pi = g.permutation(K)
    H = np.zeros((1, 1, M, K), dtype=np.uint32)
    H[0, 0, np.arange(M), pi] = 1
    C = (100 * np.arange(3)[:, None] + np.arange(K)[None, :] + 1).astype(np.uint32).reshape(1, 1, 3, K)
    out = oracle.modgemm(H, C, None, [P30[0]])
    for j in range(3):
        assert out[0, 0, j].tolist() == [100 * j + int(pi[m]) + 1 for m in range(M)]


def test_zero_c_returns_zero_or_g():
    g = rng(5)
    q = P30[1]
    H = rand_u32(g, (1, 3, 4, 5))
    C = np.zeros((1, 3, 6, 5), dtype=np.uint32)
    G = rand_u32(g, (1, 3, 3, 4))
    out = oracle.modgemm(H, C, G, [q])
    assert (out[0, :, :3, :] == 0).all()                                  # "(0 | G)": left half zero
    assert np.array_equal(out[0, :, 3:, :], (G[0].astype(np.uint64) % q).astype(np.uint32))


# ---- against numpy's int64 matmul where nothing can wrap ---------------------------------------

def test_numpy_matmul_small_values():
    g = rng(6)
    T, NC, M, K, ncols, gcols = 2, 5, 17, 64, 6, 3
    H = rand_u32(g, (T, NC, M, K), 1 << 14)
    C = rand_u32(g, (T, NC, ncols, K), 1 << 14)
    G = rand_u32(g, (T, NC, gcols, M), 1 << 14)
    out = oracle.modgemm(H, C, G, P30, nthreads=3)
    for t in range(T):
        for c in range(NC):
            S = H[t, c].astype(np.int64) @ C[t, c].astype(np.int64).T      # M x ncols, < 2^34
            S[:, ncols - gcols:] += G[t, c].astype(np.int64).T
            assert np.array_equal(out[t, c], (S.T % P30[t]).astype(np.uint32))


def test_thread_count_invariance():
    g = rng(7)
    H = rand_u32(g, (2, 7, 5, 33))
    C = rand_u32(g, (2, 7, 4, 33))
    G = rand_u32(g, (2, 7, 2, 5))
    a = oracle.modgemm(H, C, G, P29, nthreads=1)
    assert np.array_equal(a, oracle.modgemm(H, C, G, P29, nthreads=4))


# ---- the paper's lazy-reduction method equals the definition --------------------

@pytest.mark.parametrize("defer", [1, 7, 32])
def test_lazy_equals_definition(defer):
    g = rng(8 + defer)
    T, NC, M, K, ncols, gcols = 2, 3, 8, 1280, 4, 2
    H = np.stack([rand_u32(g, (NC, M, K), q) for q in P29])
    C = np.stack([rand_u32(g, (NC, ncols, K), q) for q in P29])
    G = np.stack([rand_u32(g, (NC, gcols, M), q) for q in P29])
    H[:, 0, 0, :] = np.array(P29, dtype=np.uint32)[:, None] - 1   # worst case: every product (q-1)^2
    C[:, 0, 0, :] = np.array(P29, dtype=np.uint32)[:, None] - 1
    assert np.array_equal(oracle.modgemm_lazy(H, C, G, P29, defer), oracle.modgemm(H, C, G, P29))


def test_lazy_precondition():
    H = np.ones((1, 1, 1, 4), dtype=np.uint32)
    C = np.ones((1, 1, 1, 4), dtype=np.uint32)
    with pytest.raises(OverflowError):
        oracle.modgemm_lazy(H, C, None, [P30[0]])           # q >= 2^29
    with pytest.raises(OverflowError):
        oracle.modgemm_lazy(H, C, None, [P29[0]], defer=33)  # more than 32 deferred MACs
    H[0, 0, 0, 0] = P29[0]
    with pytest.raises(OverflowError):
        oracle.modgemm_lazy(H, C, None, [P29[0]])           # input >= q
    # 32 worst-case products + carry-in + G fit 64 bits; 2^64 / (2^29-1)^2 = 64.0..: the paper's 32 is safe
    assert 32 * (2**29 - 1) ** 2 + 2 * (2**29 - 1) < 2**64


# ---- linearity (eq. (1); RLWE additions / plaintext products PAPER.md:551-555) -----

def test_linearity_in_c_and_g():
    g = rng(9)
    q = P30[0]
    H = rand_u32(g, (1, 2, 6, 40), q)
    C1, C2 = rand_u32(g, (1, 2, 4, 40), q), rand_u32(g, (1, 2, 4, 40), q)
    G1, G2 = rand_u32(g, (1, 2, 2, 6), q), rand_u32(g, (1, 2, 2, 6), q)
    Cs = ((C1.astype(np.uint64) + C2) % q).astype(np.uint32)
    Gs = ((G1.astype(np.uint64) + G2) % q).astype(np.uint32)
    a = oracle.modgemm(H, C1, G1, [q]).astype(np.uint64)
    b = oracle.modgemm(H, C2, G2, [q]).astype(np.uint64)
    assert np.array_equal(oracle.modgemm(H, Cs, Gs, [q]), ((a + b) % q).astype(np.uint32))
    # scaling C by a constant scales H*C
    c = 123456789
    Cc = ((C1.astype(np.uint64) * c) % q).astype(np.uint32)
    a0 = oracle.modgemm(H, C1, None, [q]).astype(np.uint64)
    assert np.array_equal(oracle.modgemm(H, Cc, None, [q]), ((a0 * c) % q).astype(np.uint32))


# ---- meaning: point-wise products over NTT coefficients = negacyclic polynomial products -------

def _ntt_matrix(polys, q, psi):
    """polys[...][N] -> values[...][N] along the last axis."""
    arr = np.asarray(polys, dtype=object)
    out = np.empty(arr.shape, dtype=object)
    for idx in np.ndindex(arr.shape[:-1]):
        out[idx] = rlwe.ntt(list(arr[idx]), q, psi)
    return out


def test_pointwise_gemm_is_polynomial_matrix_product():
    """H, C, G are matrices of polynomials in Z_q[X]/(X^N+1).  The oracle on
    their NTTs, transformed back, must equal sum_i h_mi(X)*c_ij(X) + g (schoolbook, X^N = -1)."""
    g = rng(10)
    N, M, K, B = 8, 3, 4, 2
    q = rlwe.find_prime(N, 16, 1 << 20)
    psi = rlwe.primitive_2n_root(N, q)
    assert rlwe.intt(rlwe.ntt(list(range(N)), q, psi), q, psi) == list(range(N))
    h = g.integers(0, q, size=(M, K, N))
    c = g.integers(0, q, size=(K, 2 * B, N))
    gg = g.integers(0, q, size=(M, B, N))
    hN, cN, gN = _ntt_matrix(h, q, psi), _ntt_matrix(c, q, psi), _ntt_matrix(gg, q, psi)
    # tile-major operands: problem = NTT coefficient index
    H = np.array(hN.transpose(2, 0, 1).tolist(), dtype=np.uint32).reshape(1, N, M, K)
    C = np.array(cN.transpose(2, 1, 0).tolist(), dtype=np.uint32).reshape(1, N, 2 * B, K)
    G = np.array(gN.transpose(2, 1, 0).tolist(), dtype=np.uint32).reshape(1, N, B, M)
    out = oracle.modgemm(H, C, G, [q])                        # [1][N][2B][M]
    for m in range(M):
        for j in range(2 * B):
            want = [0] * N
            for i in range(K):
                prod = rlwe.negacyclic_mul(h[m, i], c[i, j], q)
                want = [(a + b) % q for a, b in zip(want, prod)]
            if j >= B:
                want = [(a + int(b)) % q for a, b in zip(want, gg[m, j - B])]
            got = rlwe.intt([int(out[0, cidx, j, m]) for cidx in range(N)], q, psi)
            assert got == want, (m, j)


# ---- end to end: Tiptoe-style ring packing, eq. (3) --------------------------

def test_ring_packing_round_trip():
    """M groups of N LWE ciphertexts (A, b) under secret s in {-1,0,1}^n with phases
    b + A s = m (mod p) are packed by H*C + (0|G) into M RLWE ciphertexts per client that decrypt
    to iota(m).  p is the LWE ciphertext modulus and the RLWE plaintext modulus."""
    g = rng(11)
    N, n, M, B, p = 16, 5, 2, 2, 16
    q = rlwe.find_prime(N, p, 1 << 29)                        # q = 1 mod 2N, q = 1 mod p, q < 2^29
    assert q % (2 * N) == 1 and q % p == 1
    delta = q // p
    assert delta * p + 1 == q
    psi = rlwe.primitive_2n_root(N, q)
    H = np.zeros((1, N, M, n), dtype=np.uint32)
    C = np.zeros((1, N, 2 * B, n), dtype=np.uint32)
    G = np.zeros((1, N, B, M), dtype=np.uint32)
    clients = []
    # the LWE "a" matrices are shared across clients here only through H's shape: one H, B clients
    A = g.integers(0, p, size=(M, N, n))                      # A[m] in Z_p^{N x n}
    for m in range(M):
        for i in range(n):
            H[0, :, m, i] = rlwe.ntt([int(x) for x in A[m, :, i]], q, psi)   # iota(A_i), lifted to Z_q
    for b_ in range(B):
        s_lwe = [int(x) for x in g.integers(-1, 2, size=n)]
        s_ring = rlwe.keygen(N, g)
        msgs = g.integers(0, p, size=(M, N))
        # LWE b-parts chosen so that b + A s = m mod p (eq. (2))
        bvec = [[(int(msgs[m, r]) - sum(int(A[m, r, i]) * s_lwe[i] for i in range(n))) % p for r in range(N)]
                for m in range(M)]
        for i in range(n):                                    # ct_Pack,i = Encrypt(s_i)
            a_i, b_i = rlwe.encrypt([s_lwe[i] % p] + [0] * (N - 1), s_ring, q, delta, g)
            C[0, :, b_, i] = rlwe.ntt(a_i, q, psi)            # a-parts: columns [0, B)
            C[0, :, B + b_, i] = rlwe.ntt(b_i, q, psi)        # b-parts: columns [B, 2B)
        for m in range(M):                                    # trivial encryption (0, Delta*iota(b))
            G[0, :, b_, m] = rlwe.ntt([delta * x % q for x in bvec[m]], q, psi)
        clients.append((s_ring, msgs))
    out = oracle.modgemm(H, C, G, [q])
    # noise: sum_i iota(A_i) * e_i, |.| <= n * N * (p-1) * 1  must stay below Delta/2
    assert n * N * (p - 1) < delta // 2
    for b_, (s_ring, msgs) in enumerate(clients):
        for m in range(M):
            a_res = rlwe.intt([int(out[0, c, b_, m]) for c in range(N)], q, psi)
            b_res = rlwe.intt([int(out[0, c, B + b_, m]) for c in range(N)], q, psi)
            assert rlwe.decrypt(a_res, b_res, s_ring, q, delta, p) == [int(x) for x in msgs[m]]


# ---- RNS: the same integers reduced per prime; CRT recovers the exact sum -----

def test_crt_recovers_exact_integer():
    g = rng(12)
    p0, p1 = P30
    NC, M, K, ncols = 2, 4, 64, 3
    Hi = g.integers(0, 1 << 24, size=(NC, M, K))
    Ci = g.integers(0, 1 << 24, size=(NC, ncols, K))
    Gi = g.integers(0, 1 << 24, size=(NC, 1, M))
    H = np.stack([(Hi % p).astype(np.uint32) for p in P30])
    C = np.stack([(Ci % p).astype(np.uint32) for p in P30])
    G = np.stack([(Gi % p).astype(np.uint32) for p in P30])
    out = oracle.modgemm(H, C, G, P30)
    inv = pow(p0, -1, p1)
    for c in range(NC):
        for j in range(ncols):
            for m in range(M):
                exact = sum(int(Hi[c, m, k]) * int(Ci[c, j, k]) for k in range(K))
                if j == ncols - 1:
                    exact += int(Gi[c, 0, m])
                assert exact < p0 * p1
                r0, r1 = int(out[0, c, j, m]), int(out[1, c, j, m])
                x = r0 + p0 * (((r1 - r0) * inv) % p1)
                assert x == exact


# ---- the seeded generator feeds residues below each modulus -------------------------------------

def test_generator_operands_are_residues():
    H = inputs.modgemm_operand(0, inputs.STREAM_MG_H, P30, 8, 12)
    assert H.shape == (2, 8, 12) and (H[0] < P30[0]).all() and (H[1] < P30[1]).all()
    part = inputs.modgemm_operand(0, inputs.STREAM_MG_H, P30, 8, 12, c0=3, nc=2)
    assert np.array_equal(part, H[:, 3:5])
    assert not np.array_equal(H, inputs.modgemm_operand(0, inputs.STREAM_MG_C, P30, 8, 12))
