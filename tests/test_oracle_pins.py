"""Pins for the CPU oracle (no GPU).  Each test checks oracle/ against something the paper
or the mathematics fixes -- never against the oracle's own formula retyped, and never
against the CUDA path.  A plausible mistake anywhere in the oracle (dropped term, wrong
sign or index, transposed operand, signed vs unsigned, wrong endianness, missed wrap) is
meant to fail at least one of these.
"""
import numpy as np
import pytest

import oracle
from oracle import lwe
from paper_2606_11536_b200 import inputs

Q32 = 1 << 32
PRIMES = [1073692673, 1073668097]


def rng(seed):
    return np.random.default_rng(seed)


# ---- brute force on tiny shapes (SURVEY.md 8(c) "Brute force") -----------------------------

@pytest.mark.parametrize("rows,cols,batch", [(1, 1, 1), (3, 5, 2), (8, 8, 4), (7, 3, 1), (2, 9, 3)])
@pytest.mark.parametrize("db_bits", [8, 16])
@pytest.mark.parametrize("moduli", [None, [97], PRIMES, [2, 1 << 29]])
def test_bruteforce_tiny(rows, cols, batch, db_bits, moduli):
    g = rng(rows * 1000 + cols * 10 + batch + db_bits)
    D = g.integers(0, 1 << db_bits, size=(rows, cols)).astype(np.uint8 if db_bits == 8 else np.uint16)
    T = 1 if moduli is None else len(moduli)
    Q = g.integers(0, Q32, size=(T, batch, cols), dtype=np.uint64).astype(np.uint32)
    # extreme words in the corners
    Q[0, 0, 0] = 0xFFFFFFFF
    D[0, 0] = (1 << db_bits) - 1
    want = oracle.dbmul_bruteforce(D, Q, moduli)
    assert np.array_equal(oracle.dbmul(D, Q, moduli), want)
    assert np.array_equal(oracle.dbmul_limbs(D, Q, moduli), want)


def test_hand_example(golden):
    h = golden["hand_example"]
    D = np.array(h["D"], dtype=np.uint8)
    Q = np.array(h["Q"], dtype=np.uint32)
    assert oracle.dbmul(D, Q)[0, 0].tolist() == h["answer"]
    assert oracle.dbmul_limbs(D, Q)[0, 0].tolist() == h["answer"]


# ---- closed forms ------------------------------------------------------------------------------

def test_all_ones_db_gives_query_sum():
    g = rng(1)
    cols, batch = 777, 3
    Q = g.integers(0, Q32, size=(1, batch, cols), dtype=np.uint64).astype(np.uint32)
    D = np.ones((5, cols), dtype=np.uint8)
    want = [sum(int(x) for x in Q[0, b]) % Q32 for b in range(batch)]
    A = oracle.dbmul(D, Q)
    for b in range(batch):
        assert (A[0, b] == want[b]).all()
    Qp = inputs.query(3, cols, batch, PRIMES)
    Ap = oracle.dbmul(D, Qp, PRIMES)
    for t, p in enumerate(PRIMES):
        for b in range(batch):
            assert (Ap[t, b] == sum(int(x) for x in Qp[t, b]) % p).all()


def test_all_max_wraps_and_int32_chunk_bound(golden):
    c = golden["all_max_wrap"]
    K = c["cols"]
    D = np.full((2, K), c["db_value"], dtype=np.uint8)
    Q = np.full((1, 1, K), c["query_word"], dtype=np.uint32)
    assert (oracle.dbmul(D, Q) == c["answer"]).all()
    b = golden["int32_chunk_bound"]
    # every limb accumulator reaches 255*255*k_chunk: exact at the contract and at the edge
    assert (oracle.dbmul_limbs(D, Q, k_chunk=b["k_chunk_contract"]) == c["answer"]).all()
    assert (oracle.dbmul_limbs(D, Q, k_chunk=b["k_max_exact"]) == c["answer"]).all()
    assert 255 * 255 * b["k_chunk_contract"] == b["acc_at_contract"] < b["int32_max"]
    with pytest.raises(OverflowError):
        oracle.dbmul_limbs(D, Q, k_chunk=b["k_max_exact"] + 1)


@pytest.mark.parametrize("p", PRIMES + [536608769])
def test_prime_all_ones_times_p_minus_1(p):
    K = 4099
    D = np.ones((3, K), dtype=np.uint8)
    Q = np.full((1, 2, K), p - 1, dtype=np.uint32)
    assert (oracle.dbmul(D, Q, [p]) == (-K) % p).all()
    assert (oracle.dbmul_limbs(D, Q, [p]) == (-K) % p).all()


# ---- structure: identity, permutation, unit vectors (PAPER.md:113 SimplePIR semantics) -----

def test_identity_db_returns_query():
    n = 64
    g = rng(2)
    Q = g.integers(0, Q32, size=(1, 3, n), dtype=np.uint64).astype(np.uint32)
    A = oracle.dbmul(np.eye(n, dtype=np.uint8), Q)
    assert np.array_equal(A, Q)  # answer[b][r] = Q[b][r]
    Ap = oracle.dbmul(np.eye(n, dtype=np.uint16), Q, [PRIMES[0]])
    assert np.array_equal(Ap[0], Q[0] % PRIMES[0])


def test_permutation_probe():
    rows, cols = 50, 70
    perm = rng(3).integers(0, cols, size=rows)
    D = np.zeros((rows, cols), dtype=np.uint8)
    D[np.arange(rows), perm] = 1
    Q = (np.arange(cols, dtype=np.uint32) + 1).reshape(1, 1, cols)
    assert np.array_equal(oracle.dbmul(D, Q)[0, 0], (perm + 1).astype(np.uint32))


@pytest.mark.parametrize("db_bits", [8, 16])
def test_unit_vector_query_returns_db_column(db_bits):
    rows, cols = 33, 41
    D = inputs.db_rows(5, rows, cols, db_bits)
    for j in (0, 17, cols - 1):
        Q = np.zeros((1, 2, cols), dtype=np.uint32)
        Q[0, 0, j] = 1
        c = 0x01020304
        Q[0, 1, j] = c
        A = oracle.dbmul(D, Q)
        assert np.array_equal(A[0, 0], D[:, j].astype(np.uint32))
        assert A[0, 1].tolist() == [(c * int(d)) % Q32 for d in D[:, j]]
        Ap = oracle.dbmul(D, np.concatenate([Q, Q]), PRIMES)
        for t, p in enumerate(PRIMES):
            assert Ap[t, 1].tolist() == [(c * int(d)) % p for d in D[:, j]]


# ---- linearity, eq. (1) PAPER.md:76 and phase linearity PAPER.md:516-524 ---------------------

@pytest.mark.parametrize("moduli", [None, PRIMES])
def test_linearity(moduli):
    rows, cols, batch = 19, 301, 2
    D = inputs.db_rows(7, rows, cols, 8)
    T = 1 if moduli is None else len(moduli)
    g = rng(4)
    Q1 = g.integers(0, Q32, size=(T, batch, cols), dtype=np.uint64)
    Q2 = g.integers(0, Q32, size=(T, batch, cols), dtype=np.uint64)
    c = 0x9E3779B1
    mods = [Q32] * T if moduli is None else moduli
    if moduli is not None:
        for t, p in enumerate(mods):
            Q1[t] %= p
            Q2[t] %= p
    Qs = np.stack([(Q1[t] + Q2[t]) % mods[t] for t in range(T)])
    Qc = np.stack([(Q1[t] * c) % mods[t] for t in range(T)])
    A1 = oracle.dbmul(D, Q1.astype(np.uint32), moduli).astype(np.uint64)
    A2 = oracle.dbmul(D, Q2.astype(np.uint32), moduli).astype(np.uint64)
    As = oracle.dbmul(D, Qs.astype(np.uint32), moduli).astype(np.uint64)
    Ac = oracle.dbmul(D, Qc.astype(np.uint32), moduli).astype(np.uint64)
    for t in range(T):
        assert np.array_equal(As[t], (A1[t] + A2[t]) % mods[t])
        assert np.array_equal(Ac[t].astype(object), (A1[t].astype(object) * c) % mods[t])


# ---- limb identity: the method equals the definition ---------------------

@pytest.mark.parametrize("db_bits,moduli,k_chunk", [
    (8, None, 32768), (8, None, 100), (16, None, 16384), (16, PRIMES, 16384), (8, PRIMES, 257), (16, [97, 1 << 29], 64),
])
def test_limb_method_equals_definition(db_bits, moduli, k_chunk):
    rows, cols, batch = 9, 1000, 3
    D = inputs.db_rows(11, rows, cols, db_bits)
    Q = inputs.query(11, cols, batch, moduli)
    if moduli is None:
        Q[0, 0, :7] = 0xFFFFFFFF
    assert np.array_equal(oracle.dbmul_limbs(D, Q, moduli, k_chunk=k_chunk), oracle.dbmul(D, Q, moduli))


# ---- reduces to a library routine where nothing can wrap ---------------------------------

def test_small_values_match_numpy_int64_matmul():
    rows, cols, batch = 40, 512, 5
    D = inputs.db_rows(13, rows, cols, 8)
    Qs = (inputs.query(13, cols, batch)[0] >> 18).astype(np.uint32)  # < 2^14 ; sums < 2^31: no wrap
    want = (D.astype(np.int64) @ Qs.T.astype(np.int64)).T  # [batch][rows]
    assert want.max() < Q32
    assert np.array_equal(oracle.dbmul(D, Qs.reshape(1, batch, cols))[0].astype(np.int64), want)
    Q = (inputs.query(13, cols, batch)[0] >> 12).astype(np.uint32)  # < 2^20 ; sums < 2^37 (exact in int64)
    want = (D.astype(np.int64) @ Q.T.astype(np.int64)).T
    assert np.array_equal(oracle.dbmul(D, Q.reshape(1, batch, cols))[0].astype(np.int64), want % Q32)
    p = PRIMES[1]
    assert np.array_equal(oracle.dbmul(D, Q.reshape(1, batch, cols), [p])[0].astype(np.int64), want % p)


def test_u16_is_little_endian_unsigned_lo_plus_256_hi():
    rows, cols = 12, 96
    D16 = inputs.db_rows(17, rows, cols, 16)
    raw = D16.view(np.uint8).reshape(rows, cols, 2)
    lo, hi = np.ascontiguousarray(raw[:, :, 0]), np.ascontiguousarray(raw[:, :, 1])
    Q = inputs.query(17, cols, 2)
    a = oracle.dbmul(D16, Q).astype(np.uint64)
    want = (oracle.dbmul(lo, Q).astype(np.uint64) + 256 * oracle.dbmul(hi, Q).astype(np.uint64)) % Q32
    assert np.array_equal(a, want)
    # unsigned: element 0xFFFF times 1 is 65535, not -1
    assert oracle.dbmul(np.array([[0xFFFF]], dtype=np.uint16), np.array([1], dtype=np.uint32))[0, 0, 0] == 65535
    assert oracle.dbmul(np.array([[0xFF]], dtype=np.uint8), np.array([1], dtype=np.uint32))[0, 0, 0] == 255


# ---- toy LWE round trip (SimplePIR PAPER.md:113-117) ---------------------

@pytest.mark.parametrize("cols,n", [(1024, 16), (300, 5)])
def test_toy_lwe_roundtrip_decrypts_selected_column(cols, n, golden):
    par = golden["lwe_parameters"]
    assert (lwe.DELTA, 1 << lwe.P_BITS, 1 << lwe.Q_BITS, lwe.SIGMA) == (par["delta"], par["p"], par["q"], par["sigma"])
    assert lwe.worst_case_noise_ok(cols)  # 255*19*cols < 2^23: decryption cannot fail
    rows = 48
    g = rng(cols + n)
    D = inputs.db_rows(19, rows, cols, 8)
    s = lwe.keygen(n, g)
    for i_star in (0, cols // 3, cols - 1):
        Q, e = lwe.simplepir_query(cols, i_star, s, g)
        assert np.abs(e).max() < 6 * lwe.SIGMA
        A = oracle.dbmul(D, Q.reshape(1, n + 1, cols))[0]  # [n+1][rows] = [hint | ans]
        assert np.array_equal(lwe.decrypt_answer(A, s), D[:, i_star])
        A2 = oracle.dbmul_limbs(D, Q.reshape(1, n + 1, cols))[0]
        assert np.array_equal(A2, A)


# ---- CRT consistency across RNS primes -------------------------------------

def test_crt_of_prime_answers_is_the_integer_sum():
    rows, cols, batch = 6, 2048, 2
    p0, p1 = PRIMES
    D = inputs.db_rows(23, rows, cols, 16)
    x = (inputs.query(23, cols, batch)[0] >> 2).astype(np.uint64)  # common integer x < 2^30
    Q = np.stack([(x % p0), (x % p1)]).astype(np.uint32)  # consistent residues
    A = oracle.dbmul(D, Q, PRIMES)
    inv = pow(p0, -1, p1)
    for b in range(batch):
        for r in range(rows):
            true = sum(int(D[r, k]) * int(x[b, k]) for k in range(cols))
            assert true < p0 * p1  # < 2^16 * 2^30 * 2^11 = 2^57
            a0, a1 = int(A[0, b, r]), int(A[1, b, r])
            crt = a0 + p0 * (((a1 - a0) * inv) % p1)
            assert crt == true
    assert (A[0] < p0).all() and (A[1] < p1).all()  # canonical range


def test_query_words_above_modulus_are_legal():
    # reading R5: defined on the integers, any u32 word is a legal input
    D = np.array([[3, 250]], dtype=np.uint8)
    Q = np.array([[[0xFFFFFFFF, 0xFFFFFFFE]]], dtype=np.uint32)
    p = 1073692673
    assert int(oracle.dbmul(D, Q, [p])[0, 0, 0]) == (3 * 0xFFFFFFFF + 250 * 0xFFFFFFFE) % p


def test_threads_do_not_change_the_answer():
    D = inputs.db_rows(29, 64, 256, 8)
    Q = inputs.query(29, 256, 3)
    assert np.array_equal(oracle.dbmul(D, Q, nthreads=4), oracle.dbmul(D, Q, nthreads=1))


def test_bad_arguments_are_rejected():
    D = np.zeros((2, 2), dtype=np.uint8)
    with pytest.raises(ValueError):
        oracle.dbmul(D, np.zeros((1, 1, 3), dtype=np.uint32))
    with pytest.raises(TypeError):
        oracle.dbmul(D.astype(np.int32), np.zeros(2, dtype=np.uint32))
    with pytest.raises(ValueError):
        oracle.dbmul(D, np.zeros((1, 1, 2), dtype=np.uint32), [1])  # modulus < 2


def test_rns_primes_are_as_recorded(golden):
    r = golden["rns_primes"]
    got = inputs.rns_primes(0, 4)
    assert got == r["seed0"] + r["next"]
    for p in got:
        assert p < (1 << 30) and p % 8192 == 1
        assert all(p % d for d in range(2, 40000))  # trial division: really prime (sqrt(2^30) = 32768)


# ---- NEXT-1: scalar-HE modulus switch 2^32 -> 2^18 --------------------

def test_modswitch_is_round_to_nearest_with_bounded_error():
    from fractions import Fraction
    xs = np.array([0, 1, 8191, 8192, 8193, 16383, 16384, 16385, 24576, 0x7FFFFFFF, 0x80000000,
                   0xFFFFDFFF, 0xFFFFE000, 0xFFFFFFFF, 123456789, 4000000000], dtype=np.uint32)
    ys = oracle.modswitch(xs, 18)
    for x, y in zip(xs.tolist(), ys.tolist()):
        exact = Fraction(x * (1 << 18), 1 << 32)
        want = int(exact + Fraction(1, 2)) % (1 << 18)  # floor(v + 1/2): nearest, ties up (R19)
        assert y == want, (x, y, want)
        assert 0 <= y < (1 << 18)
        err = (x - (y << 14) + (1 << 31)) % (1 << 32) - (1 << 31)  # centred difference mod 2^32
        assert abs(err) <= 1 << 13  # each rounding error within 2^31/p = 2^13
    rnd = np.random.default_rng(9).integers(0, 1 << 32, size=5000, dtype=np.uint64).astype(np.uint32)
    y = oracle.modswitch(rnd, 18).astype(np.int64)
    err = (rnd.astype(np.int64) - (y << 14) + (1 << 31)) % (1 << 32) - (1 << 31)
    assert np.abs(err).max() <= 1 << 13
    assert np.array_equal(oracle.modswitch(np.arange(0, 1 << 20, 1 << 14, dtype=np.uint32), 18),
                          np.arange(64, dtype=np.uint32))  # exact multiples of 2^14 map exactly
    assert np.array_equal(oracle.modswitch(rnd, 31), ((rnd.astype(np.uint64) + 1) >> 1).astype(np.uint32) & 0x7FFFFFFF)


def test_modswitched_answer_still_decrypts():
    # |E_round| <= (n+1) * 2^13 must stay below Delta/4 = 2^22: n = 15 is safe
    cols, rows, n = 512, 40, 15
    g = rng(77)
    D = inputs.db_rows(37, rows, cols, 8)
    s = lwe.keygen(n, g)
    Q, _ = lwe.simplepir_query(cols, 100, s, g)
    A = oracle.dbmul(D, Q.reshape(1, n + 1, cols))[0]
    A18 = oracle.modswitch(A, 18)
    assert A18.max() < (1 << 18)
    assert np.array_equal(lwe.decrypt_answer_switched(A18, s, 18), D[:, 100])


# ---- NEXT-3: signed database elements (centred plaintexts) -----------------------

@pytest.mark.parametrize("db_bits", [8, 16])
@pytest.mark.parametrize("moduli", [None, PRIMES, [97]])
def test_signed_db_bruteforce_and_relation_to_unsigned(db_bits, moduli):
    rows, cols, batch = 7, 37, 3
    Du = inputs.db_rows(91, rows, cols, db_bits)
    Ds = Du.view(np.int8 if db_bits == 8 else np.int16)
    Q = inputs.query(91, cols, batch, moduli)
    Q[0, 0, 0] = 0xFFFFFFFF
    mods = [Q32] if moduli is None else moduli
    got = oracle.dbmul_signed(Ds, Q, moduli)
    for t, q in enumerate(mods):
        for b in range(batch):
            for r in range(rows):
                s = sum(int(Ds[r, k]) * int(Q[t, b, k]) for k in range(cols))  # Python big ints
                assert int(got[t, b, r]) == s % q
    # SURVEY.md reading R1: signed and unsigned answers differ by 2^bits * sum of Q over the
    # elements whose top bit is set
    unsigned = oracle.dbmul(Du, Q, moduli)
    top = (Du >> (db_bits - 1)).astype(np.uint8)  # 0/1 mask as a DB of its own
    corr = oracle.dbmul(top, Q, moduli).astype(object)
    for t, q in enumerate(mods):
        assert np.array_equal((unsigned[t].astype(object) - (1 << db_bits) * corr[t]) % q, got[t].astype(object))


def test_signed_db_decrypts_to_the_same_bytes():
    # Delta * 2^8 = 2^32 = 0 mod q: a centred plaintext m and m + 256 decrypt to the same byte,
    # and the noise term sum_k D[r][k] e_k is about half as large (|D| <= 128 instead of 255)
    cols, rows, n = 1024, 30, 7
    g = rng(123)
    Du = inputs.db_rows(93, rows, cols, 8)
    s = lwe.keygen(n, g)
    Q, e = lwe.simplepir_query(cols, 500, s, g)
    A = oracle.dbmul_signed(Du.view(np.int8), Q.reshape(1, n + 1, cols))[0]
    assert np.array_equal(lwe.decrypt_answer(A, s), Du[:, 500])
    # worst case |sum_k D[r][k] e_k| <= max|D| * 19 * cols: 128 instead of 255
    assert 128 * 19 * cols < 255 * 19 * cols < (lwe.DELTA >> 1)
    # mean square over many independent error vectors: E[D^2] = 5461.5 (centred) against 21717.5
    # (unsigned), so the ratio is 1/4 up to sampling error (200 x 30 samples)
    E = lwe.sample_error((cols, 200), rng(124))
    ms_signed = float(np.mean((Du.view(np.int8).astype(np.int64) @ E).astype(np.float64) ** 2))
    ms_unsigned = float(np.mean((Du.astype(np.int64) @ E).astype(np.float64) ** 2))
    assert 0.2 < ms_signed / ms_unsigned < 0.3
    assert np.abs(Du.view(np.int8).astype(np.int64) @ e).max() < 128 * 19 * cols
