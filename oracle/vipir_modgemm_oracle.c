/*
 * vipir_modgemm_oracle.c -- CPU ORACLE for VIPIR's parallel INT32 modular GEMMs
 *                           Out = H * C + (0 | G)  mod q_t.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with paper_2606_11536_b200/csrc (the CUDA path).
 *
 * What it computes (section 3.5.2): "Let H and G denote these two polynomial
 * matrices after the NTTs.  The computation of H*C + (0 | G) follows, where C is an n x 2B
 * polynomial matrix corresponding to expanded special ciphertexts from B clients.  As RNS and
 * NTT transform a polynomial multiplication into point-wise multiplications over (#RNS * N)
 * coefficients, this reduces to (#RNS * N)-parallel ceil(D1/N) x 2B x n INT32 GEMMs with
 * additional modular reduction computations."  (Also PAPER.md:239 section 4, :261-265
 * section 4.2; the packing it implements is eq. (3), Appendix C.1.)
 *
 * One problem per (RNS prime t, NTT coefficient c), P = T*NC problems, each an
 * M x ncols x K product (M = ceil(D1/N), K = n, ncols = 2B) of 32-bit residues mod q_t, plus
 * the M x gcols matrix G added to the LAST gcols columns ("(0 | G)", gcols = B: the b-parts
 * of the B clients' ciphertexts, eq. (3)'s trivial encryption (0, Delta*iota(b)); DESIGN.md
 * reading R21).
 *
 * Layout ("tile-major (GEMM-friendly)": every problem's operands contiguous;
 * DESIGN.md reading R21).  All arrays uint32:
 *   H    [T][NC][M][K]        K contiguous
 *   C    [T][NC][ncols][K]    each column of C contiguous along K
 *   G    [T][NC][gcols][M]    (may be NULL when gcols == 0)
 *   Out  [T][NC][ncols][M]    canonical representative in [0, q_t)
 * Any u32 is a legal input word (also >= q_t): the sum is over the integers, then reduced.
 *
 * Two routines:
 *   vipir_oracle_modgemm       the plain definition: triple loop per problem, 128-bit
 *                              accumulator, one explicit "% q" per output word;
 *   vipir_oracle_modgemm_lazy  the paper's METHOD step by step (section 4.2):
 *                              "Using RNS primes smaller than 2^29 and 64-bit accumulators, we
 *                              defer reduction for up to 32 multiply-accumulates without
 *                              overflow".  Needs q_t < 2^29 and inputs < q_t (returns -3
 *                              otherwise); must equal the definition there.
 *
 * Parity pins: tests/test_modgemm_oracle_pins.py (brute force in Python big integers, closed
 * forms, identity, numpy int64 matmul, linearity, negacyclic polynomial products through a
 * naive NTT, a toy RLWE ring-packing round trip of eq. (3), CRT).  Nothing here is "parity
 * unpinned".
 */
#include <stddef.h>
#include <stdint.h>

typedef unsigned __int128 u128;

/*
 * The definition.  For t < T, c < NC, j < ncols, m < M:
 *   Out[t][c][j][m] = ( sum_{k<K} H[t][c][m][k] * C[t][c][j][k]
 *                       + (j >= ncols - gcols ? G[t][c][j - (ncols - gcols)][m] : 0) ) mod q_t
 * Returns 0, or -1 on a bad argument.  nthreads > 1 splits the problem loop with OpenMP.
 */
int vipir_oracle_modgemm(uint32_t T, uint64_t NC, uint64_t M, uint64_t K, uint64_t ncols, uint64_t gcols,
                         const uint32_t *moduli, const uint32_t *H, const uint32_t *C, const uint32_t *G,
                         uint32_t *Out, int nthreads) {
    if (!moduli || !H || !C || !Out || T == 0 || NC == 0 || M == 0 || K == 0 || ncols == 0) return -1;
    if (gcols > ncols || (gcols > 0 && !G)) return -1;
    for (uint32_t t = 0; t < T; ++t)
        if (moduli[t] < 2) return -1;
    const int64_t P = (int64_t)((uint64_t)T * NC);
    const uint64_t g0 = ncols - gcols;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 1 ? nthreads : 1)
#endif
    for (int64_t p = 0; p < P; ++p) {
        const uint64_t q = moduli[(uint64_t)p / NC];
        const uint32_t *Hp = H + (uint64_t)p * M * K;
        const uint32_t *Cp = C + (uint64_t)p * ncols * K;
        const uint32_t *Gp = gcols ? G + (uint64_t)p * gcols * M : NULL;
        uint32_t *Op = Out + (uint64_t)p * ncols * M;
        for (uint64_t j = 0; j < ncols; ++j) {
            for (uint64_t m = 0; m < M; ++m) {
                u128 acc = 0;
                for (uint64_t k = 0; k < K; ++k) acc += (u128)Hp[m * K + k] * Cp[j * K + k];
                if (j >= g0) acc += Gp[(j - g0) * M + m];
                Op[j * M + m] = (uint32_t)(acc % q);
            }
        }
    }
    return 0;
}

/*
 * The paper's method: 64-bit accumulator, a reduction every `defer` (<= 32)
 * multiply-accumulates.  With q < 2^29 and inputs < q every product is < 2^58, so 32 of them
 * plus a reduced carry-in (< 2^29) and G (< 2^29) stay below 2^63 + 2^30 < 2^64.
 * Returns 0; -1 bad argument; -3 if a modulus is >= 2^29, an input word is >= its modulus or
 * defer is not in [1, 32] (the method's precondition does not hold).
 */
int vipir_oracle_modgemm_lazy(uint32_t T, uint64_t NC, uint64_t M, uint64_t K, uint64_t ncols, uint64_t gcols,
                              const uint32_t *moduli, const uint32_t *H, const uint32_t *C, const uint32_t *G,
                              uint32_t *Out, uint32_t defer) {
    if (!moduli || !H || !C || !Out || T == 0 || NC == 0 || M == 0 || K == 0 || ncols == 0) return -1;
    if (gcols > ncols || (gcols > 0 && !G)) return -1;
    if (defer < 1 || defer > 32) return -3;
    for (uint32_t t = 0; t < T; ++t)
        if (moduli[t] < 2 || moduli[t] >= (1u << 29)) return moduli[t] < 2 ? -1 : -3;
    const uint64_t P = (uint64_t)T * NC;
    const uint64_t g0 = ncols - gcols;
    for (uint64_t p = 0; p < P; ++p) {
        const uint64_t q = moduli[p / NC];
        const uint32_t *Hp = H + p * M * K;
        const uint32_t *Cp = C + p * ncols * K;
        const uint32_t *Gp = gcols ? G + p * gcols * M : NULL;
        uint32_t *Op = Out + p * ncols * M;
        for (uint64_t i = 0; i < M * K; ++i)
            if (Hp[i] >= q) return -3;
        for (uint64_t i = 0; i < ncols * K; ++i)
            if (Cp[i] >= q) return -3;
        for (uint64_t i = 0; i < gcols * M; ++i)
            if (Gp[i] >= q) return -3;
        for (uint64_t j = 0; j < ncols; ++j) {
            for (uint64_t m = 0; m < M; ++m) {
                uint64_t acc = (j >= g0) ? Gp[(j - g0) * M + m] : 0; /* (0 | G) */
                uint32_t pending = 0;
                for (uint64_t k = 0; k < K; ++k) {
                    acc += (uint64_t)Hp[m * K + k] * Cp[j * K + k];
                    if (++pending == defer) { /* lazy reduction */
                        acc %= q;
                        pending = 0;
                    }
                }
                Op[j * M + m] = (uint32_t)(acc % q);
            }
        }
    }
    return 0;
}
