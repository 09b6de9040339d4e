"""GPU parity of the lift + forward NTT (vipir_ntt_*, csrc/ntt_lift.cuh) against the CPU oracle, bit for
bit, through the C ABI; and the built chain end to end on the GPU with the paper's parameters:
scan (vipir_dbmul + fused 2^32 -> 2^18 switch) -> NTT (G, H) -> H*C + (0|G) (vipir_modgemm) -> a toy RLWE
client decrypts the packed ciphertexts to the LWE phases, which decode to the selected DB column."""
import numpy as np
import pytest

import oracle
from oracle import lwe, rlwe
from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built, run_dbmul

pytestmark = pytest.mark.gpu

Q29 = [536608769, 533463041, 531628033]   # < 2^29, = 1 mod 2^18
SMALL = {4: [97, 193], 8: [7681, 12289]}  # = 1 mod 2N


def run_ntt(X, log2n, moduli, psi, scale, p_bits, centered, layout):
    import torch
    ensure_built()
    N = 1 << log2n
    n_a, M = X.shape[0], X.shape[1] // N
    d_X = torch.from_numpy(np.ascontiguousarray(X).view(np.int32)).cuda()
    shape = (len(moduli), N, n_a, M) if layout == vipir.NTT_LAYOUT_G else (len(moduli), N, M, n_a)
    d_O = torch.full(shape, -1, dtype=torch.int32, device="cuda")
    with vipir.NttPlan(log2n, moduli, psi, scale, p_bits, centered) as plan:
        plan(d_X, n_a, M, layout, d_O)
        torch.cuda.synchronize()
        bad = plan.bad_input()
    return d_O.cpu().numpy().view(np.uint32), bad


@pytest.mark.parametrize("log2n,n_a,M", [(4, 3, 5), (4, 1, 700), (8, 2, 3), (8, 5, 70), (12, 1, 1), (12, 3, 11), (12, 9, 2)])
@pytest.mark.parametrize("layout", [vipir.NTT_LAYOUT_G, vipir.NTT_LAYOUT_H])
@pytest.mark.parametrize("centered", [False, True])
def test_ntt_matches_oracle(log2n, n_a, M, layout, centered):
    N = 1 << log2n
    moduli = Q29 if log2n == 12 else SMALL[log2n]
    p_bits = 18 if log2n == 12 else (6 if log2n == 4 else 12)
    psi = [oracle.smallest_psi(N, q) for q in moduli]
    scale = [(q // (1 << p_bits)) % q if t else 1 for t, q in enumerate(moduli)]
    g = np.random.default_rng(1000 * log2n + 10 * n_a + M)
    X = g.integers(0, 1 << p_bits, size=(n_a, M * N), dtype=np.uint32)
    X[0, :4] = [0, (1 << p_bits) - 1, 1 << (p_bits - 1), (1 << (p_bits - 1)) - 1]
    got, bad = run_ntt(X, log2n, moduli, psi, scale, p_bits, centered, layout)
    want = oracle.ntt_lift(X, N, moduli, psi, scale, p_bits, centered, layout, nthreads=16)
    assert not bad
    assert np.array_equal(got, want), f"{(got != want).sum()} of {got.size} words differ"


@pytest.mark.parametrize("which", ["below_2^29", "above_2^29", "mixed"])
def test_ntt_prime_ranges_adversarial(which):
    """Primes below 2^29 (the paper's) and just below 2^30 (the ABI's limit: the lazy butterflies keep
    values in [0, 4q) < 2^32) -- adversarial inputs (all words p - 1, scale q - 1) next to random ones, N = 2^12."""
    N, log2n, p_bits = 4096, 12, 18
    big = inputs.rns_primes(0, 2, 1 << 30, 8192)           # just below 2^30, = 1 mod 2N
    assert all(q > (1 << 29) for q in big)
    moduli = {"below_2^29": Q29, "above_2^29": big, "mixed": [Q29[0], big[0]]}[which]
    psi = [oracle.smallest_psi(N, q) for q in moduli]
    scale = [q - 1 for q in moduli]
    g = np.random.default_rng(7)
    X = g.integers(0, 1 << p_bits, size=(2, 3 * N), dtype=np.uint32)
    X[1, :N] = (1 << p_bits) - 1
    for centered in (False, True):
        got, bad = run_ntt(X, log2n, moduli, psi, scale, p_bits, centered, vipir.NTT_LAYOUT_G)
        want = oracle.ntt_lift(X, N, moduli, psi, scale, p_bits, centered, vipir.NTT_LAYOUT_G, nthreads=16)
        assert not bad and np.array_equal(got, want), f"{(got != want).sum()} of {got.size} words differ"


def test_ntt_monomials_and_bad_input_flag():
    N, log2n, p_bits = 4096, 12, 18
    psi = [oracle.smallest_psi(N, q) for q in Q29]
    X = np.zeros((1, 2 * N), dtype=np.uint32)
    X[0, 1] = 1            # polynomial 0 = X
    X[0, N + 4095] = 1     # polynomial 1 = X^4095
    got, bad = run_ntt(X, log2n, Q29, psi, [1, 1, 1], p_bits, False, vipir.NTT_LAYOUT_G)
    assert not bad
    for t, q in enumerate(Q29):
        for c in (0, 1, 2, 1000, 2048, 4095):
            assert int(got[t, c, 0, 0]) == pow(psi[t], 2 * c + 1, q)
            assert int(got[t, c, 0, 1]) == pow(psi[t], (2 * c + 1) * 4095, q)
    X[0, 7] = 1 << 18      # a word >= p: flagged
    _, bad = run_ntt(X, log2n, Q29, psi, [1, 1, 1], p_bits, False, vipir.NTT_LAYOUT_G)
    assert bad


def test_chain_scan_ntt_modgemm_decrypts():
    """The paper's parameters except the toy ring degree and LWE dimension: LWE p = 2^8, q = 2^32,
    Delta = 2^24; switch to 2^18 (:295, :698); RLWE plaintext modulus 2^18, three RNS
    primes < 2^29 with q_i = 1 mod 2^18 (:559, :578-607); N = 16, n = 6."""
    import torch
    ensure_built()
    g = np.random.default_rng(2026)
    N, log2n, n, M, B, p_bits = 16, 4, 6, 2, 2, 18
    rows, cols, p = M * N, 64, 1 << p_bits
    q = Q29[0] * Q29[1] * Q29[2]
    delta = q // p
    assert delta * p + 1 == q
    psi = [oracle.smallest_psi(N, qt) for qt in Q29]
    D = inputs.db_rows(7, rows, cols, 8)
    # ---- clients: one public A (same a-part for everybody), own secrets, own columns ----
    secrets, targets, b_rows, a_rows = [], [], [], None
    for b_ in range(B):
        s = lwe.keygen(n, g)
        i_star = int(g.integers(0, cols))
        Q, _ = lwe.simplepir_query(cols, i_star, s, np.random.default_rng(777))   # same stream: same a-part
        a_rows = Q[:n] if a_rows is None else a_rows
        assert np.array_equal(a_rows, Q[:n])
        b_rows.append(Q[n])
        secrets.append(s)
        targets.append(i_star)
    # ---- step 1 (GPU): scan + fused modulus switch: the hint (offline, n columns) and the answers (B) ----
    hint = run_dbmul(D, a_rows.reshape(1, n, cols), None, modswitch_bits=p_bits)[0]        # [n][rows] < 2^18
    ans = run_dbmul(D, np.stack(b_rows).reshape(1, B, cols), None, modswitch_bits=p_bits)[0]   # [B][rows]
    # ---- step 2 (GPU): lift + NTT into the GEMM operand layouts ----
    H, _ = run_ntt(hint, log2n, Q29, psi, [1, 1, 1], p_bits, False, vipir.NTT_LAYOUT_H)        # [T][N][M][n]
    G, _ = run_ntt(ans, log2n, Q29, psi, [delta % qt for qt in Q29], p_bits, False, vipir.NTT_LAYOUT_G)  # [T][N][B][M]
    # ---- the clients' packing keys: ct_Pack,i = Encrypt(s_i) under a ring secret (eq. (3)) ----
    T = len(Q29)
    C = np.zeros((T, N, 2 * B, n), dtype=np.uint32)
    ring_secrets = []
    for b_ in range(B):
        s_ring = rlwe.keygen(N, g)
        ring_secrets.append(s_ring)
        for i in range(n):
            a_i, b_i = rlwe.encrypt([int(secrets[b_][i]) % p] + [0] * (N - 1), s_ring, q, delta, g)
            for t, qt in enumerate(Q29):
                C[t, :, b_, i] = rlwe.ntt([x % qt for x in a_i], qt, psi[t])
                C[t, :, B + b_, i] = rlwe.ntt([x % qt for x in b_i], qt, psi[t])
    # ---- step 3 (GPU): H*C + (0|G) mod q_t ----
    d_O = torch.full((T, N, 2 * B, M), -1, dtype=torch.int32, device="cuda")
    with vipir.ModGemmPlan(T, N, M, n, 2 * B, B, Q29) as plan:
        plan.set_h(torch.from_numpy(H.view(np.int32)).cuda())
        plan(torch.from_numpy(C.view(np.int32)).cuda(), torch.from_numpy(G.view(np.int32)).cuda(), d_O)
        torch.cuda.synchronize()
    out = d_O.cpu().numpy().view(np.uint32)
    assert np.array_equal(out, oracle.modgemm(H, C, G, Q29))
    # ---- clients decrypt: CRT over the primes, inverse NTT, RLWE decryption -> LWE phases -> DB bytes ----
    def crt(res):
        x = 0
        for r, qt in zip(res, Q29):
            Mi = q // qt
            x = (x + r * Mi * pow(Mi, -1, qt)) % q
        return x
    delta_lwe = p >> lwe.P_BITS                                  # 2^10 after the switch
    for b_ in range(B):
        for m in range(M):
            parts = []
            for col in (b_, B + b_):
                coeffs_t = [rlwe.intt([int(out[t, c, col, m]) for c in range(N)], qt, psi[t]) for t, qt in enumerate(Q29)]
                parts.append([crt([coeffs_t[t][j] for t in range(T)]) for j in range(N)])
            phases = rlwe.decrypt(parts[0], parts[1], ring_secrets[b_], q, delta, p)   # LWE phases mod 2^18
            got = [((ph + (delta_lwe >> 1)) // delta_lwe) & 0xFF for ph in phases]
            assert got == [int(x) for x in D[m * N:(m + 1) * N, targets[b_]]], (b_, m)


@pytest.mark.parametrize("n_a,M,layout", [(32, 256, vipir.NTT_LAYOUT_G), (1280, 8, vipir.NTT_LAYOUT_H)])
def test_ntt_paper_shape_sampled_polynomials_and_coefficient_sums(n_a, M, layout):
    """The launch configuration bench.py times (N = 2^12, three primes, Delta scale; G for 32 clients x 256
    polynomials, H columns = 1280): sampled polynomials recomputed one by one by the oracle, plus an identity
    that covers every polynomial at any size: sum_c Y[c] = N * scale * lift(x_0) mod q, because
    sum_c psi^((2c+1) j) = 0 for 0 < j < N (psi^(2j) is a non-trivial N-th root of unity)."""
    N, log2n, p_bits = 4096, 12, 18
    psi = [oracle.smallest_psi(N, q) for q in Q29]
    q_all = Q29[0] * Q29[1] * Q29[2]
    scale = [(q_all >> p_bits) % q for q in Q29]
    X = (inputs.query(5, M * N, n_a) >> np.uint32(32 - p_bits))[0]       # [n_a][M*N] words < 2^18
    got, bad = run_ntt(X, log2n, Q29, psi, scale, p_bits, True, layout)
    assert not bad
    polys = got if layout == vipir.NTT_LAYOUT_G else got.transpose(0, 1, 3, 2)      # [T][N][n_a][M]
    g = np.random.default_rng(8)
    picks = {(0, 0), (n_a - 1, M - 1), (n_a - 1, 0), (0, M - 1)} | {(int(g.integers(n_a)), int(g.integers(M))) for _ in range(4)}
    for a, m in sorted(picks):
        want = oracle.ntt_lift(X[a:a + 1, m * N:(m + 1) * N], N, Q29, psi, scale, p_bits, True, oracle.LAYOUT_G, nthreads=16)
        assert np.array_equal(polys[:, :, a, m], want[:, :, 0, 0]), (a, m)
    x0 = X.reshape(n_a, M, N)[:, :, 0].astype(np.int64)
    lifted = np.where(x0 >= (1 << (p_bits - 1)), x0 - (1 << p_bits), x0)
    for t, q in enumerate(Q29):
        sums = polys[t].astype(np.uint64).sum(axis=0) % q                  # [n_a][M]
        want = np.array([[(N * scale[t] * int(v)) % q for v in row] for row in lifted], dtype=np.uint64)
        assert np.array_equal(sums, want), t
