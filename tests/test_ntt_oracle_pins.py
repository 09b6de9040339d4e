"""Pins for the CPU oracle of the lift + forward NTT that produces the ring-packing operands G and H
(oracle/vipir_ntt_oracle.c; PAPER.md:214 section 3.5.2, :667 Appendix C.1, :95-101 section 2.3).  No GPU.

Each test checks the oracle against something the paper or the mathematics fixes, never against its
own formula retyped and never against the CUDA path: powers of psi from Python's pow() (monomials
have closed-form transforms), the convolution theorem against a schoolbook product in
Z_q[X]/(X^N+1), the inverse transform in Python integers, linearity, the two lifts, the two output
layouts, and a toy RLWE ring-packing round trip of eq. (3) whose G and H come
from this routine and whose result must decrypt to the packed LWE plaintexts.
"""
import numpy as np
import pytest

import oracle
from oracle import rlwe

Q29 = [536608769, 533463041, 531628033]   # < 2^29, = 1 mod 2^18: also = 1 mod 2N for N = 4096


def rng(seed):
    return np.random.default_rng(seed)


def schoolbook_negacyclic(f, g, q):
    N = len(f)
    out = [0] * N
    for i in range(N):
        for j in range(N):
            s = int(f[i]) * int(g[j])
            if i + j >= N:
                out[i + j - N] = (out[i + j - N] - s) % q
            else:
                out[i + j] = (out[i + j] + s) % q
    return out


def test_smallest_psi_is_a_primitive_2n_root():
    for N, q in [(8, 17), (16, 97), (4096, Q29[0]), (4096, Q29[2])]:
        psi = oracle.smallest_psi(N, q)
        assert pow(psi, N, q) == q - 1 and pow(psi, 2 * N, q) == 1
        assert all(pow(x, N, q) != q - 1 for x in range(2, min(psi, 2000)))
    with pytest.raises(ValueError):
        oracle.smallest_psi(8, 19)     # 19 != 1 mod 16


def test_hand_example_n2():
    # N = 2, q = 5: psi^2 = -1 mod 5 -> psi = 2.  f = 1 + 3X: f(psi) = 7 = 2, f(psi^3) = 1 + 3*8 = 25 = 0
    assert oracle.smallest_psi(2, 5) == 2
    O = oracle.ntt_lift(np.array([[1, 3]], dtype=np.uint32), 2, [5], [2], [1], 2)
    assert O.shape == (1, 2, 1, 1) and [int(O[0, 0, 0, 0]), int(O[0, 1, 0, 0])] == [2, 0]


@pytest.mark.parametrize("N,q", [(8, 17), (64, 12289), (256, 7681)])
def test_monomials_have_closed_form_transforms(N, q):
    """NTT(scale * X^k)[c] = scale * psi^((2c+1) k): every root and every ordering mistake shows."""
    psi = oracle.smallest_psi(N, q)
    X = np.eye(N, dtype=np.uint32).reshape(1, N * N)          # polynomial m = X^m
    O = oracle.ntt_lift(X, N, [q], [psi], [3], 1)             # p = 2: words 0/1
    for k in range(N):
        want = [3 * pow(psi, (2 * c + 1) * k, q) % q for c in range(N)]
        assert [int(v) for v in O[0, :, 0, k]] == want, k


def test_monomials_at_the_papers_size():
    """N = 2^12, the three RNS primes of the benchmark, Delta-like scale."""
    N = 4096
    ks = [1, 1234, 4095]
    X = np.zeros((1, len(ks) * N), dtype=np.uint32)
    for i, k in enumerate(ks):
        X[0, i * N + k] = 1
    psi = [oracle.smallest_psi(N, q) for q in Q29]
    scale = [123456789 % q for q in Q29]
    O = oracle.ntt_lift(X, N, Q29, psi, scale, 18, nthreads=8)
    for t, q in enumerate(Q29):
        for i, k in enumerate(ks):
            for c in (0, 1, 2, 2047, 2048, 4095):
                assert int(O[t, c, 0, i]) == scale[t] * pow(psi[t], (2 * c + 1) * k, q) % q


def test_convolution_theorem_against_schoolbook():
    g = rng(1)
    N, q, pb = 32, 12289, 13                                   # 12289 = 1 mod 64; p = 8192 < q
    psi = oracle.smallest_psi(N, q)
    f = g.integers(0, 1 << pb, size=N, dtype=np.uint32)
    h = g.integers(0, 1 << pb, size=N, dtype=np.uint32)
    F = oracle.ntt_lift(np.stack([f, h]), N, [q], [psi], [1], pb)[0, :, :, 0]   # [N][2]
    prod = schoolbook_negacyclic(f, h, q)
    # point-wise product of the transforms, taken back with the inverse transform in Python integers
    Y = [int(F[c, 0]) * int(F[c, 1]) % q for c in range(N)]
    n_inv, psi_inv = pow(N, -1, q), pow(psi, -1, q)
    back = [n_inv * sum(Y[c] * pow(psi_inv, (2 * c + 1) * j, q) for c in range(N)) % q for j in range(N)]
    assert back == prod


def test_inverse_transform_in_python_integers():
    g = rng(2)
    N, q, pb = 64, 12289, 12
    psi = oracle.smallest_psi(N, q)
    x = g.integers(0, 1 << pb, size=N, dtype=np.uint32)
    Y = [int(v) for v in oracle.ntt_lift(x.reshape(1, N), N, [q], [psi], [1], pb)[0, :, 0, 0]]
    n_inv, psi_inv = pow(N, -1, q), pow(psi, -1, q)
    back = [n_inv * sum(Y[c] * pow(psi_inv, (2 * c + 1) * j, q) for c in range(N)) % q for j in range(N)]
    assert back == [int(v) for v in x]


def test_linearity_and_scale():
    g = rng(3)
    N, q, pb = 128, Q29[0], 18
    psi = oracle.smallest_psi(N, q)   # Q29[0] = 1 mod 2^18, so also = 1 mod 256
    a = g.integers(0, 1 << (pb - 1), size=N, dtype=np.uint32)
    b = g.integers(0, 1 << (pb - 1), size=N, dtype=np.uint32)
    Oa, Ob, Oab = (oracle.ntt_lift(v.reshape(1, N), N, [q], [psi], [7], pb)[0, :, 0, 0].astype(np.uint64)
                   for v in (a, b, a + b))
    assert np.array_equal((Oa + Ob) % q, Oab)
    O1 = oracle.ntt_lift(a.reshape(1, N), N, [q], [psi], [1], pb)[0, :, 0, 0].astype(np.uint64)
    assert np.array_equal(O1 * 7 % q, Oa)


def test_centered_lift_is_x_minus_p():
    g = rng(4)
    N, q, pb = 16, 97, 6
    p = 1 << pb
    psi = oracle.smallest_psi(N, q)
    x = g.integers(0, p, size=N, dtype=np.uint32)
    x[:4] = [0, p // 2 - 1, p // 2, p - 1]
    Oc = [int(v) for v in oracle.ntt_lift(x.reshape(1, N), N, [q], [psi], [1], pb, centered=True)[0, :, 0, 0]]
    lifted = [int(v) if v < p // 2 else int(v) - p for v in x]          # representative in [-p/2, p/2)
    want = [sum(lifted[j] * pow(psi, (2 * c + 1) * j, q) for j in range(N)) % q for c in range(N)]
    assert Oc == want
    Ou = [int(v) for v in oracle.ntt_lift(x.reshape(1, N), N, [q], [psi], [1], pb)[0, :, 0, 0]]
    want_u = [sum(int(x[j]) * pow(psi, (2 * c + 1) * j, q) for j in range(N)) % q for c in range(N)]
    assert Ou == want_u and Ou != Oc


def test_layouts_moduli_and_threads():
    g = rng(5)
    N, pb, n_a, M = 64, 10, 3, 5
    mods = [12289, 7681]                                       # both = 1 mod 128
    psi = [oracle.smallest_psi(N, q) for q in mods]
    X = g.integers(0, 1 << pb, size=(n_a, M * N), dtype=np.uint32)
    G = oracle.ntt_lift(X, N, mods, psi, [1, 2], pb, out_layout=oracle.LAYOUT_G)
    H = oracle.ntt_lift(X, N, mods, psi, [1, 2], pb, out_layout=oracle.LAYOUT_H, nthreads=4)
    assert G.shape == (2, N, n_a, M) and H.shape == (2, N, M, n_a)
    assert np.array_equal(G.transpose(0, 1, 3, 2), H)
    for t, q in enumerate(mods):                               # each prime on its own, each polynomial on its own
        a, m = 2, 3
        one = oracle.ntt_lift(X[a:a + 1, m * N:(m + 1) * N], N, [q], [psi[t]], [t + 1], pb)
        assert np.array_equal(one[0, :, 0, 0], G[t, :, a, m])
        assert (G[t] < q).all()


def test_argument_errors():
    X = np.zeros((1, 8), dtype=np.uint32)
    with pytest.raises(ValueError):
        oracle.ntt_lift(X, 8, [17], [2], [1], 3)               # 2^8 = 1 mod 17: not a primitive 16th root
    X[0, 3] = 8
    with pytest.raises(ValueError):
        oracle.ntt_lift(X, 8, [17], [oracle.smallest_psi(8, 17)], [1], 3)   # word >= p


# ---- end to end: the scan's LWE words -> G, H -> H*C + (0|G) -> RLWE decryption (eq. (3)) ----------

@pytest.mark.parametrize("centered", [False, True])
def test_ring_packing_round_trip_with_oracle_ntt(centered):
    """M groups of N LWE ciphertexts (A, b) mod p with b + A s = m (mod p) (eq. (2)).
    H = NTT(lift iota(A_i)) and G = NTT(Delta * lift iota(b)) come from the oracle under test; the
    packed result H*C + (0|G) must decrypt to iota(m)."""
    g = rng(11)
    N, n, M, B, pb = 16, 5, 2, 2, 4
    p = 1 << pb
    q = rlwe.find_prime(N, p, 1 << 29)
    delta = q // p
    assert delta * p + 1 == q
    psi = oracle.smallest_psi(N, q)
    A = g.integers(0, p, size=(n, M * N), dtype=np.uint32)     # hint layout: [column i][row]: A_i = column i
    H = oracle.ntt_lift(A, N, [q], [psi], [1], pb, centered=centered, out_layout=oracle.LAYOUT_H)   # [1][N][M][n]
    C = np.zeros((1, N, 2 * B, n), dtype=np.uint32)
    bwords = np.zeros((B, M * N), dtype=np.uint32)             # answer layout: [client][row]
    clients = []
    for b_ in range(B):
        s_lwe = [int(x) for x in g.integers(-1, 2, size=n)]
        s_ring = rlwe.keygen(N, g)
        msgs = g.integers(0, p, size=M * N)
        for r in range(M * N):
            bwords[b_, r] = (int(msgs[r]) - sum(int(A[i, r]) * s_lwe[i] for i in range(n))) % p
        for i in range(n):                                     # ct_Pack,i = Encrypt(s_i)
            a_i, b_i = rlwe.encrypt([s_lwe[i] % p] + [0] * (N - 1), s_ring, q, delta, g)
            C[0, :, b_, i] = rlwe.ntt(a_i, q, psi)
            C[0, :, B + b_, i] = rlwe.ntt(b_i, q, psi)
        clients.append((s_ring, msgs))
    G = oracle.ntt_lift(bwords, N, [q], [psi], [delta % q], pb, centered=centered, out_layout=oracle.LAYOUT_G)
    out = oracle.modgemm(H, C, G, [q])
    assert n * N * (p - 1) < delta // 2
    for b_, (s_ring, msgs) in enumerate(clients):
        for m in range(M):
            a_res = rlwe.intt([int(out[0, c, b_, m]) for c in range(N)], q, psi)
            b_res = rlwe.intt([int(out[0, c, B + b_, m]) for c in range(N)], q, psi)
            assert rlwe.decrypt(a_res, b_res, s_ring, q, delta, p) == [int(x) for x in msgs[m * N:(m + 1) * N]]
