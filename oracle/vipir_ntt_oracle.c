/*
 * vipir_ntt_oracle.c -- CPU ORACLE for the lift + forward NTT that turns the scan's scalar-HE
 *                       output (and, offline, the hint) into the polynomial matrices G and H of
 *                       the ring-packing stage          (after NEXT-4).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with paper_2606_11536_b200/csrc (the CUDA path).
 *
 * What it computes.  PAPER.md:214 (section 3.5.2): "the D1 x n and D1 x B SimplePIR outputs
 * are first transformed into polynomials by treating each length-N vector along the D1
 * dimension as a polynomial in R_q, with integer elements interpreted as coefficients.  This
 * yields ceil(D1/N) x n and ceil(D1/N) x B polynomials, to which NTTs are applied
 * independently.  Let H and G denote these two polynomial matrices after the NTTs."
 * PAPER.md:667 (Appendix C.1): "the server lifts the coefficients of iota(A_i) and iota(b) from
 * Z_p to Z_q and transforms them into the NTT domain"; eq. (3) adds the b part as
 * the trivial encryption (0, Delta * iota(b)), so the b polynomials carry the factor Delta.
 * PAPER.md:95-101 (section 2.3): RNS turns a polynomial into a #RNS x N INT32 matrix, "NTT
 * applies a variant of the Fourier transform to each row", after which a product in
 * R_q = Z_q[X]/(X^N + 1) is an element-wise product.  PAPER.md:578-582 (Appendix A.4):
 * q_i = 1 mod 2N "is a sufficient condition for enabling NTT".
 *
 * Definition (the transform by its definition, O(N^2) per polynomial; the method -- PAPER.md:269,
 * a single-kernel O(N log N) NTT with Montgomery reduction -- reaches exactly this result).
 * Input X[a][m][j]: word j < N of polynomial (a, m), a < n_a (hint column / client), m < M
 * (M = ceil(D1/N)); i.e. X is the scan's answer layout [a][D1] with D1 = M*N.  For RNS prime
 * t < T with modulus q_t, primitive 2N-th root of unity psi_t (psi_t^N = -1 mod q_t) and
 * constant scale_t:
 *     x_j     = scale_t * lift_t(X[a][m][j])            mod q_t
 *     Y[c]    = sum_{j < N} x_j * psi_t^((2c+1) * j)    mod q_t,      c < N   (natural order:
 *               Y[c] is the polynomial evaluated at the c-th odd power of psi_t -- the roots of
 *               X^N + 1; reading R24)
 * lift_t (reading R23): X[a][m][j] is a residue mod p = 2^p_bits, stored as a u32 < p.
 *   centered == 0:  lift(x) = x                                   (representative in [0, p))
 *   centered == 1:  lift(x) = x          if x <  p/2
 *                           = x - p + q_t if x >= p/2              (representative in [-p/2, p/2))
 * Words >= p are rejected (-3).  p_bits <= 29 and p < q_t are required.
 * Output, canonical in [0, q_t), in the layout of the modular GEMMs' operands (PAPER.md:263:
 * the "layout transposition" between polynomial-major and tile-major):
 *   out_layout == 0 ("G"):  O[t][c][a][m]     (vipir_modgemm's d_G  [T][NC][gcols][M], a = client)
 *   out_layout == 1 ("H"):  O[t][c][m][a]     (vipir_modgemm's d_H  [T][NC][M][K],     a = k)
 *
 * Parity pins: tests/test_ntt_oracle_pins.py -- powers of psi from Python's pow() (closed forms
 * for the monomials), the convolution theorem against a schoolbook negacyclic product, the
 * inverse transform written with Python integers, linearity, both lifts against q - (p - x),
 * the layouts, and a toy RLWE ring-packing round trip (eq. (3)) in which G and H come from this
 * routine and the result must decrypt to the packed LWE plaintexts.  Nothing is "parity unpinned".
 */
#include <stddef.h>
#include <stdint.h>

static uint32_t mulmod(uint32_t a, uint32_t b, uint32_t q) { return (uint32_t)(((uint64_t)a * b) % q); }

static uint32_t powmod(uint32_t base, uint64_t e, uint32_t q) {
    uint32_t r = 1 % q;
    while (e) {
        if (e & 1) r = mulmod(r, base, q);
        base = mulmod(base, base, q);
        e >>= 1;
    }
    return r;
}

/* returns 0 on success; -1 bad argument; -2 psi is not a primitive 2N-th root of unity mod q_t
 * (psi^N != -1); -3 an input word is >= p */
int vipir_oracle_ntt_lift(uint32_t T, uint32_t n_a, uint32_t M, uint32_t N, const uint32_t *moduli,
                          const uint32_t *psi, const uint32_t *scale, uint32_t p_bits, int centered,
                          int out_layout, const uint32_t *X, uint32_t *O, int nthreads) {
    if (!moduli || !psi || !scale || !X || !O || T == 0 || n_a == 0 || M == 0 || N < 2 || (N & (N - 1)))
        return -1;
    if (p_bits < 1 || p_bits > 29 || (out_layout != 0 && out_layout != 1)) return -1;
    const uint32_t p = 1u << p_bits;
    for (uint32_t t = 0; t < T; ++t) {
        if (moduli[t] <= p || moduli[t] >= (1u << 30)) return -1;
        if (powmod(psi[t] % moduli[t], N, moduli[t]) != moduli[t] - 1) return -2;
    }
    const uint64_t n_words = (uint64_t)n_a * M * N;
    for (uint64_t i = 0; i < n_words; ++i)
        if (X[i] >= p) return -3;
    if (nthreads < 1) nthreads = 1;

    const int64_t n_poly = (int64_t)n_a * M;
    for (uint32_t t = 0; t < T; ++t) {
        const uint32_t q = moduli[t];
#pragma omp parallel for num_threads(nthreads) schedule(static)
        for (int64_t pi = 0; pi < n_poly; ++pi) {
            const uint32_t a = (uint32_t)(pi / M), m = (uint32_t)(pi % M);
            const uint32_t *x = X + (uint64_t)pi * N;
            for (uint32_t c = 0; c < N; ++c) {
                const uint32_t w = powmod(psi[t] % q, 2ull * c + 1, q); /* the c-th root of X^N + 1 */
                uint32_t acc = 0, wj = 1; /* wj = w^j */
                for (uint32_t j = 0; j < N; ++j) {
                    uint32_t v = x[j];
                    if (centered && v >= p / 2) v = v - p + q; /* x - p, taken mod q */
                    v = mulmod(v % q, scale[t] % q, q);
                    acc = (uint32_t)(((uint64_t)acc + mulmod(v, wj, q)) % q);
                    wj = mulmod(wj, w, q);
                }
                const uint64_t idx = out_layout == 0 ? (((uint64_t)t * N + c) * n_a + a) * M + m
                                                     : (((uint64_t)t * N + c) * M + m) * n_a + a;
                O[idx] = acc;
            }
        }
    }
    return 0;
}
